"""Pins of the oracle's topology builders (no GPU)."""
import ctypes as C
import itertools
import os

import numpy as np
import pytest

from oracle import oracle as ora


def _rows(row_ptr, col_idx):
    return [col_idx[row_ptr[i]:row_ptr[i + 1]] for i in range(len(row_ptr) - 1)]


def test_ball_counts_printed_in_paper(golden_dir):
    for line in open(os.path.join(golden_dir, "lattice_link_counts.txt")):
        if line.startswith("#") or not line.strip():
            continue
        ndim, P, links = map(int, line.split())
        assert ora.lattice_degree(ndim, P, include_self=True) == links
        assert ora.lattice_degree(ndim, P, include_self=False) == links - 1


@pytest.mark.parametrize("ndim", [1, 2, 3])
@pytest.mark.parametrize("P", [1, 2, 3, 4, 5, 6])
def test_degree_by_enumeration(ndim, P):
    cnt = sum(1 for d in itertools.product(range(-P, P + 1), repeat=ndim)
              if sum(x * x for x in d) <= P * P)
    assert ora.lattice_degree(ndim, P, True) == cnt
    # the 32 / 256 neighbours the north-star configs quote
    if ndim == 3 and P == 2:
        assert cnt - 1 == 32
    if ndim == 3 and P == 4:
        assert cnt - 1 == 256


def test_ring_rows():
    n, P = 11, 3
    rp, ci = ora.topology_ring(n, P)
    for i, row in enumerate(_rows(rp, ci)):
        expect = sorted((i + d) % n for d in range(-P, P + 1) if d != 0)
        assert list(row) == expect
    rp, ci = ora.topology_ring(n, P, include_self=True)
    assert all(len(r) == 2 * P + 1 and i in r for i, r in enumerate(_rows(rp, ci)))
    with pytest.raises(ValueError):
        ora.topology_ring(6, 3)        # 2P >= n: a neighbour would be counted twice


def _dense_lattice(extent, P):
    """Brute force: dense 0/1 matrix from minimum-image squared distances."""
    ext = list(extent) + [1] * (3 - len(extent))
    nx, ny, nz = ext
    n = nx * ny * nz
    idx = np.arange(n)
    coords = np.stack([idx % nx, (idx // nx) % ny, idx // (nx * ny)], axis=1)
    L = np.zeros((n, n), dtype=np.int8)
    for i in range(n):
        d = np.abs(coords - coords[i])
        d = np.minimum(d, np.array(ext) - d)
        L[i] = ((d * d).sum(axis=1) <= P * P)
    np.fill_diagonal(L, 0)
    return L


@pytest.mark.parametrize("extent,P", [((7,), 2), ((5, 6), 2), ((4, 4), 1), ((5, 5, 5), 2),
                                      ((7, 5, 6), 2), ((9, 9, 9), 4)])
def test_lattice_against_dense_brute_force(extent, P):
    rp, ci = ora.topology_lattice(extent, P)
    L = _dense_lattice(extent, P)
    n = L.shape[0]
    deg = ora.lattice_degree(len(extent), P)
    for i, row in enumerate(_rows(rp, ci)):
        assert len(row) == deg
        assert list(row) == list(np.nonzero(L[i])[0])        # sorted, distinct, exact set
    assert (L == L.T).all()                                  # j in row i <=> i in row j


def test_lattice_index_map_x_fastest():
    # element (i,j,k) has number k*N1^2 + j*N1 + i.  With P=1 the
    # neighbours of site 0 on a 5x6x7 lattice are +-1 (x), +-5 (y), +-30 (z) mod extents.
    rp, ci = ora.topology_lattice((5, 6, 7), 1)
    assert sorted(ci[rp[0]:rp[1]]) == sorted([1, 4, 5, 25, 30, 180])


def test_lattice_row_ranges_match_full():
    rp, ci = ora.topology_lattice((6, 6, 6), 2)
    rp2, ci2 = ora.topology_lattice((6, 6, 6), 2, row_begin=50, row_count=20)
    assert (ci2 == ci[rp[50]:rp[70]]).all() and (rp2 == rp[50:71] - rp[50]).all()
    with pytest.raises(ValueError):
        ora.topology_lattice((4, 8, 8), 2)


def test_mix64_published_vector(golden_dir):
    f = ora.lib().ora_mix64
    f.restype, f.argtypes = C.c_uint64, [C.c_uint64]
    for line in open(os.path.join(golden_dir, "splitmix64_vectors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        a, b = (int(x, 16) for x in line.split())
        assert f(a) == b


def _py_random_rows(n, k, seed):
    """The rule of reading R8 in Python integers (independent of the C code)."""
    M, G = (1 << 64) - 1, 0x9E3779B97F4A7C15

    def mix(z):
        z ^= z >> 30
        z = (z * 0xBF58476D1CE4E5B9) & M
        z ^= z >> 27
        z = (z * 0x94D049BB133111EB) & M
        return z ^ (z >> 31)

    rows = []
    for i in range(n):
        hi, row, t = mix((seed + G * (i + 1)) & M), [], 0
        while len(row) < k:
            j = (mix((hi + G * (t + 1)) & M) * (n - 1)) >> 64
            j += j >= i
            if j not in row:
                row.append(j)
            t += 1
        rows.append(sorted(row))
    return rows


@pytest.mark.parametrize("n,k,seed", [(16, 5, 1), (9, 8, 7), (200, 100, 3), (1000, 3, 2 ** 63 + 5)])
def test_random_indegree_rule_and_properties(n, k, seed):
    rp, ci = ora.topology_random_indegree(n, k, seed)
    rows = _rows(rp, ci)
    assert [list(r) for r in rows] == _py_random_rows(n, k, seed)
    for i, r in enumerate(rows):
        assert len(r) == k and len(set(r)) == k and i not in r
        assert all(0 <= j < n for j in r) and list(r) == sorted(r)
    rp2, ci2 = ora.topology_random_indegree(n, k, seed, row_begin=3, row_count=4)
    assert (ci2 == ci[rp[3]:rp[7]]).all()


def test_random_indegree_sources_uniform():
    n, k = 2000, 50
    _, ci = ora.topology_random_indegree(n, k, 11)
    counts = np.bincount(ci, minlength=n)
    # out-degree of a uniform-source graph ~ Binomial(n*k, 1/n): mean k, var ~k
    assert abs(counts.mean() - k) < 1e-9
    assert 0.8 * k < counts.var() < 1.25 * k
    _, ci_b = ora.topology_random_indegree(n, k, 12)
    assert (ci != ci_b).mean() > 0.9                       # the seed matters
