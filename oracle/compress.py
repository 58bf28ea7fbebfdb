"""Differential compression of the coupling matrix, Algorithm 2 of the paper (PAPER.md:151-175,
Sec. III.C) -- TEST INFRASTRUCTURE (oracle), plain numpy, shares nothing with the CUDA library.

The coupling matrix L is given by rows; row i is the set of positions j with L_ij = 1 (the
oscillators that influence i), here a sorted integer array instead of a bit vector.
In that representation the operations of Alg. 2 are:

    ROL(row, i): the bit at position j moves to position (j - i) mod N  ("circular shift ... left";
                 "implemented using the addition of bits' positions modulo N")
    XOR(a, b)  : symmetric difference of the two position sets
    COMPRESS   : V <- L_0;  for every i: d = XOR(ROL(L_i, i), V); C_i <- index of d in the
                 difference table D, d being appended to D if it is not there yet
    EXTRACT(i) : ROR(XOR(V, D[C_i]), i): positions (p + i) mod N for p in the symmetric difference

Reading R16: the listing is garbled (`return ROR(...)` printed above COMPRESS,
PAPER.md:157 vs :166); the text at PAPER.md:167 fixes the order of operations used here.

Pins (tests/test_oracle_compress.py): the paper's own example -- "a full mesh topology has a
common vector with all bits set and a difference table with a single entry having all bits unset"
(PAPER.md:171); EXTRACT(COMPRESS(L)) == L on random graphs; rings give one empty entry; the 3D
ball lattice of PAPER.md:313 gives (2P+1)^3 entries whose stored positions, at 4 bytes each, come to
the "approximately 16 megabytes" the paper quotes for P = 6.
"""
import numpy as np


def _rows(row_ptr, col_idx):
    return [np.asarray(col_idx[row_ptr[i]:row_ptr[i + 1]], dtype=np.int64) for i in range(len(row_ptr) - 1)]


def compress(row_ptr, col_idx):
    """COMPRESS of Alg. 2.  Returns (V, D, C): V sorted int64 positions of the common vector,
    D list of sorted int64 arrays (difference table), C int32[N] (row -> entry of D)."""
    rows = _rows(row_ptr, col_idx)
    n = len(rows)
    V = np.sort(rows[0] % n) if n else np.zeros(0, dtype=np.int64)      # ROL(L_0, 0) = L_0
    D, index, C = [], {}, np.zeros(n, dtype=np.int32)
    for i in range(n):
        shifted = (rows[i] - i) % n                                     # ROL(L_i, i)
        d = np.setxor1d(shifted, V)                                     # XOR with the common vector (sorted)
        key = d.tobytes()
        j = index.get(key)                                              # FIND(D_j == d)
        if j is None:
            j = len(D)
            index[key] = j
            D.append(d)
        C[i] = j
    return V, D, C


def extract(i, V, D, C, n):
    """EXTRACT of Alg. 2: row i of the coupling matrix as a sorted array of positions."""
    return np.sort((np.setxor1d(V, D[C[i]]) + i) % n)


def extract_all(V, D, C, n):
    """All rows as canonical CSR (row_ptr int64, col_idx int32)."""
    rows = [extract(i, V, D, C, n) for i in range(n)]
    row_ptr = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int64)
    col_idx = (np.concatenate(rows) if rows else np.zeros(0)).astype(np.int32)
    return row_ptr, col_idx


def stored_positions(V, D):
    """Positions held by the common vector and the difference table (the B*K of PAPER.md:173)."""
    return int(len(V) + sum(len(d) for d in D))
