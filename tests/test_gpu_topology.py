"""Topology builder on the device vs the oracle's: bit-exact (CSR index handling)."""
import numpy as np
import pytest

import harness as H
from oracle import oracle as ora
from paper_2410_19075_b200 import configs

pytestmark = pytest.mark.gpu


def _B():
    from paper_2410_19075_b200 import binding
    return binding


def _net(topo, n, model=0, params=None):
    B = _B()
    return B.Net(model, B.F64, n, topo, params or dict(K=1.0, alpha=0.1))


@pytest.mark.parametrize("n,P,self_", [(256, 64, False), (11, 5, False), (9, 0, False), (40, 3, True)])
def test_ring(n, P, self_):
    B = _B()
    net = _net(dict(kind=B.TOPO_RING, radius=P, include_self=self_), n)
    rp, ci = net.get_topology()
    rp0, ci0 = ora.topology_ring(n, P, self_)
    assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0)
    assert net.degree() == (len(ci0), 2 * P + int(self_))


@pytest.mark.parametrize("extent,P,self_", [((17,), 3, False), ((9, 12), 4, False), ((8, 8, 8), 2, False),
                                            ((10, 9, 11), 4, False), ((13, 13, 13), 6, True),
                                            ((6, 5, 4), 1, False)])
def test_lattice(extent, P, self_):
    B = _B()
    n = int(np.prod(extent))
    net = _net(dict(kind=B.TOPO_LATTICE, extent=extent, radius=P, include_self=self_), n)
    rp, ci = net.get_topology()
    rp0, ci0 = ora.topology_lattice(extent, P, self_)
    assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0)
    # a row range
    rp, ci = net.get_topology(n // 3, 7)
    rp0, ci0 = ora.topology_lattice(extent, P, self_, n // 3, 7)
    assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0)


@pytest.mark.parametrize("n,k,seed", [(16, 5, 1), (9, 8, 7), (5000, 100, 1), (3000, 0, 2), (2, 1, 2 ** 63 + 9)])
def test_random_indegree(n, k, seed):
    B = _B()
    net = _net(dict(kind=B.TOPO_RANDOM_INDEGREE, in_degree=k, seed=seed), n)
    rp, ci = net.get_topology()
    rp0, ci0 = ora.topology_random_indegree(n, k, seed)
    assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0)


def test_csr_given_roundtrip_and_validation():
    B = _B()
    rng = np.random.default_rng(5)
    n = 300
    deg = rng.integers(0, 9, n)
    rp = np.concatenate([[0], np.cumsum(deg)]).astype(np.int64)
    ci = np.concatenate([np.sort(rng.choice(n, d, replace=False)) for d in deg]).astype(np.int32)
    net = _net(dict(kind=B.TOPO_CSR, row_ptr=rp, col_idx=ci), n)
    rp1, ci1 = net.get_topology()
    assert np.array_equal(rp1, rp) and np.array_equal(ci1, ci)
    assert net.degree() == (len(ci), -1)
    rp2, ci2 = net.get_topology(10, 20)
    assert np.array_equal(ci2, ci[rp[10]:rp[30]])
    # dynamics on a given CSR (ragged rows incl. empty ones) against the oracle
    phi, om = rng.uniform(-3, 3, n), rng.normal(size=n)
    net.set_state(phi.reshape(1, -1))
    net.set_param_array(B.PARAM_OMEGA, om)
    ref = ora.OracleNet.ks(n, rp, ci, 1.0, 0.1, om).rhs(phi)
    assert H.rel_maxnorm(net.eval_rhs(), ref) <= 1e-12
    direct = B.Net(0, B.F64, n, dict(kind=B.TOPO_CSR, row_ptr=rp, col_idx=ci), dict(K=1.0, alpha=0.1),
                   method=B.METHOD_DIRECT)
    direct.set_state(phi.reshape(1, -1)); direct.set_param_array(B.PARAM_OMEGA, om)
    assert H.rel_maxnorm(direct.eval_rhs(), ref) <= 1e-12
    # device pointers
    import torch
    net_d = _net(dict(kind=B.TOPO_CSR, row_ptr=torch.from_numpy(rp).cuda(), col_idx=torch.from_numpy(ci).cuda()), n)
    assert np.array_equal(net_d.get_topology()[1], ci)
    bad = ci.copy(); bad[3] = n
    with pytest.raises(B.OscnetError) as e:
        _net(dict(kind=B.TOPO_CSR, row_ptr=rp, col_idx=bad), n)
    assert e.value.code == -3
    badp = rp.copy(); badp[5] = badp[6] + 1
    with pytest.raises(B.OscnetError) as e:
        _net(dict(kind=B.TOPO_CSR, row_ptr=badp, col_idx=ci), n)
    assert e.value.code == -3


def test_full_size_topologies_sampled_rows():
    """BASELINE sizes: rows sampled across the index range, bit-exact."""
    rng = np.random.default_rng(0)
    for cfg in ("3a", "4", "5", "2"):
        w = configs.get(cfg)
        net = _B().Net.from_workload(w)
        rows = np.unique(np.concatenate([[0, 1, w.n - 1, w.n // 2], rng.integers(0, w.n, 40)]))
        for r in rows:
            rp, ci = net.get_topology(int(r), 1)
            rp0, ci0 = H.oracle_topology(w, int(r), 1)
            assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0), (cfg, r)
        rp, ci = net.get_topology(w.n - 1000, 1000)
        rp0, ci0 = H.oracle_topology(w, w.n - 1000, 1000)
        assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0)
        net.close()
