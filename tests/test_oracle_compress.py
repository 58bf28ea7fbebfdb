"""Pins of the oracle's coupling-matrix compression (Alg. 2; oracle/compress.py).
Each compares with something the paper or the mathematics fixes, not with the oracle itself."""
import numpy as np
import pytest

from oracle import compress as cp
from oracle import oracle as ora


def _csr(rows):
    rp = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int64)
    ci = (np.concatenate(rows) if len(rows) else np.zeros(0)).astype(np.int32)
    return rp, ci


def test_full_mesh_is_the_papers_example():
    """"a full mesh topology has a common vector with all bits set and a difference
    table with a single entry having all bits unset"."""
    n = 37
    rp, ci = _csr([np.arange(n)] * n)
    V, D, C = cp.compress(rp, ci)
    assert np.array_equal(V, np.arange(n))
    assert len(D) == 1 and len(D[0]) == 0
    assert np.all(C == 0)


@pytest.mark.parametrize("n,P,inc", [(64, 5, False), (33, 16, True), (10, 1, False)])
def test_ring_is_shift_invariant(n, P, inc):
    """Every row of a ring is row 0 shifted by i, so the table holds one empty difference."""
    rp, ci = ora.topology_ring(n, P, inc)
    V, D, C = cp.compress(rp, ci)
    assert len(D) == 1 and len(D[0]) == 0 and len(V) == 2 * P + int(inc)
    rp2, ci2 = cp.extract_all(V, D, C, n)
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_round_trip_on_random_graphs(seed):
    """EXTRACT(COMPRESS(L)) = L for arbitrary rows (ragged, empty rows, self-loops)."""
    rng = np.random.default_rng(seed)
    n = 60
    rows = [np.sort(rng.choice(n, size=rng.integers(0, 9), replace=False)) for _ in range(n)]
    rp, ci = _csr(rows)
    V, D, C = cp.compress(rp, ci)
    for i in range(n):
        assert np.array_equal(cp.extract(i, V, D, C, n), rows[i])
    # brute force with explicit bit vectors: d = ROL(L_i, i) XOR V
    L = np.zeros((n, n), dtype=bool)
    for i, r in enumerate(rows):
        L[i, r] = True
    for i in range(n):
        d = np.roll(L[i], -i) ^ L[0]
        assert np.array_equal(np.flatnonzero(d), D[C[i]])


@pytest.mark.parametrize("n1,P", [(10, 2), (14, 3)])
def test_3d_ball_lattice_table_size(n1, P):
    """Index k N1^2 + j N1 + i: a wrap in z is a circular shift modulo N = N1^3 and
    is absorbed by ROL; wraps in x and y are not.  Sites fall into 2P + 1 classes per axis for x and
    for y (P distances to the low face, the interior, P distances to the high face), so the table
    has (2P + 1)^2 entries, whatever N1 -- "very few entries in the difference table" for regular
    networks, and the compressed size is dominated by the N row references
    (O(max(BK, N)))."""
    rp, ci = ora.topology_lattice((n1, n1, n1), P, True)
    V, D, C = cp.compress(rp, ci)
    assert len(V) == ora.lattice_degree(3, P, True)          # 33 / 123 links, the paper's count at P = 2
    assert len(D) == (2 * P + 1) ** 2
    assert sum(1 for d in D if len(d) == 0) == 1
    rp2, ci2 = cp.extract_all(V, D, C, n1 ** 3)
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
    # rows whose x and y are in the class of row 0 (x = y = 0) share its entry
    x = np.arange(n1 ** 3) % n1
    y = (np.arange(n1 ** 3) // n1) % n1
    assert np.all(C[(x == 0) & (y == 0)] == C[0])


def test_lattice_with_defects_adds_few_entries():
    """A lattice whose rows were edited at a few sites ("lattice with defects"): only the edited
    rows get new table entries; the round trip is exact."""
    n1, P = 12, 2
    n = n1 ** 3
    rp, ci = ora.topology_lattice((n1, n1, n1), P, False)
    rows = [ci[rp[i]:rp[i + 1]].astype(np.int64) for i in range(n)]
    base = len(cp.compress(rp, ci)[1])
    rng = np.random.default_rng(0)
    edited = rng.choice(n, 7, replace=False)
    for i in edited:
        r = rows[i]
        r = np.delete(r, rng.integers(0, len(r)))                    # a missing link
        r = np.union1d(r, [(i + n // 2 + 3) % n])                    # a long-range link
        rows[i] = r
    rp2, ci2 = _csr(rows)
    V, D, C = cp.compress(rp2, ci2)
    assert base <= len(D) <= base + len(edited)
    a, b = cp.extract_all(V, D, C, n)
    assert np.array_equal(a, rp2) and np.array_equal(b, ci2)


def test_round_trip_property_based():
    """Hypothesis: for any rows (any n <= 24, any subsets), EXTRACT(COMPRESS(L)) = L, rows that are
    circular shifts of row 0 share the empty entry, and the table never has more entries than rows."""
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=150, deadline=None)
    @given(st.integers(1, 24).flatmap(lambda n: st.tuples(st.just(n), st.lists(
        st.sets(st.integers(0, n - 1)), min_size=n, max_size=n))))
    def check(arg):
        n, sets = arg
        rows = [np.array(sorted(s), dtype=np.int64) for s in sets]
        rp, ci = _csr(rows)
        V, D, C = cp.compress(rp, ci)
        assert len(D) <= n and np.array_equal(V, rows[0])
        for i in range(n):
            assert np.array_equal(cp.extract(i, V, D, C, n), rows[i])
            if np.array_equal(np.sort((rows[0] + i) % n), rows[i]):
                assert len(D[C[i]]) == 0

    check()
