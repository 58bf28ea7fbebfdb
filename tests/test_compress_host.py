"""net_compress_csr (host-side COMPRESS of Alg. 2 in the library) against the oracle's
oracle/compress.py, bit for bit: same common vector, same difference table in the same order, same
row references.  No GPU needed (pure host call)."""
import numpy as np
import pytest

from oracle import compress as cp
from oracle import oracle as ora
from paper_2410_19075_b200 import binding as B


def _cases():
    rng = np.random.default_rng(4)
    out = []
    rp, ci = ora.topology_lattice((9, 8, 7), 2, False)
    out.append(("lattice 9x8x7 P=2", rp, ci))
    rp, ci = ora.topology_ring(50, 7, False)
    out.append(("ring", rp, ci))
    rp, ci = ora.topology_random_indegree(200, 6, 3)
    out.append(("random graph", rp, ci))
    n = 40
    rows = [np.sort(rng.choice(n, size=rng.integers(0, 6), replace=False)) for _ in range(n)]
    rp = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int64)
    out.append(("ragged with empty rows", rp, np.concatenate(rows).astype(np.int32)))
    n = 23
    out.append(("full mesh", (np.arange(n + 1) * n).astype(np.int64), np.tile(np.arange(n), n).astype(np.int32)))
    return out


@pytest.mark.parametrize("name,rp,ci", _cases(), ids=[c[0] for c in _cases()])
def test_library_compress_equals_oracle(name, rp, ci):
    V, D, C = cp.compress(rp, ci)
    cm = B.net_compress_csr(rp, ci)
    v, dptr, dpos, c = cm.arrays()
    assert np.array_equal(v, V)
    assert len(dptr) - 1 == len(D)
    for j, d in enumerate(D):
        assert np.array_equal(dpos[dptr[j]:dptr[j + 1]], d)
    assert np.array_equal(c, C)
    if name == "full mesh":
        assert len(D) == 1 and dptr[-1] == 0 and len(v) == 23


def test_compress_rejects_bad_input():
    rp = np.array([0, 2, 3], dtype=np.int64)
    with pytest.raises(B.OscnetError):
        B.net_compress_csr(rp, np.array([0, 5, 1], dtype=np.int32))      # index outside [0, n)
