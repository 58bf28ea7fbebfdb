"""NET_TOPO_COMPRESSED: the differentially compressed coupling matrix of Alg. 2 (
SURVEY.md 8(f).3) as a topology format.  The device EXTRACTs rows on the fly; the expanded rows must
equal the CSR the matrix was compressed from bit for bit, and RHS / trajectories must meet the north
star's tolerances against the oracle on that CSR."""
from dataclasses import replace

import numpy as np
import pytest

import harness as H
from oracle import oracle as ora
from paper_2410_19075_b200 import binding as B, configs

pytestmark = pytest.mark.gpu


def _lattice_with_defects(n1, P, n_def, seed):
    n = n1 ** 3
    rp, ci = ora.topology_lattice((n1, n1, n1), P, False)
    rows = [ci[rp[i]:rp[i + 1]].astype(np.int64) for i in range(n)]
    rng = np.random.default_rng(seed)
    for i in rng.choice(n, n_def, replace=False):
        r = np.delete(rows[i], rng.integers(0, len(rows[i])))
        rows[i] = np.union1d(r, [(i + n // 2 + 3) % n])
    rp2 = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int64)
    return rp2, np.concatenate(rows).astype(np.int32)


def _net(w, rp, ci, inp):
    cm = B.net_compress_csr(rp, ci)
    dtype = B.F32 if w.dtype == "f32" else B.F64
    net = B.Net(w.model, dtype, w.n, dict(kind=B.TOPO_COMPRESSED, compressed=cm), w.params)
    net.set_state(inp["y0"].astype(net.np_dtype))
    if inp["elem"] is not None:
        net.set_param_array(B.PARAM_OMEGA if w.model in (configs.KS, configs.KSI) else B.PARAM_IEXT,
                            inp["elem"].astype(net.np_dtype))
    return net, cm


def _oracle(w, rp, ci, inp):
    p = w.params
    if w.model == configs.KS:
        return ora.OracleNet.ks(w.n, rp, ci, p["K"], p["alpha"], inp["elem"])
    if w.model == configs.FHN:
        return ora.OracleNet.fhn(w.n, rp, ci, p["eps"], p["a"], p["sigma"], p["phi"])
    return ora.OracleNet.hh(w.n, rp, ci, inp["elem"], **p)


CASES = [("KS f64 lattice 12^3 P=2 with 9 defects", configs.get("3b", n1=12), 2, 9),
         ("KS f32 lattice 10^3 P=4 with 5 defects", configs.get("3a", n1=10), 4, 5),
         ("FHN f64 lattice 12^3 P=2 with 9 defects", replace(configs.get("5", n1=12), dtype="f64"), 2, 9),
         ("HH f64 lattice 8^3 P=2 with 4 defects", replace(configs.get("4", n=512), topo=configs.LATTICE), 2, 4)]


@pytest.mark.parametrize("name,w,P,ndef", CASES, ids=[c[0] for c in CASES])
def test_compressed_lattice_with_defects(name, w, P, ndef):
    n1 = round(w.n ** (1 / 3))
    rp, ci = _lattice_with_defects(n1, P, ndef, seed=3)
    inp = H.make_inputs(w, seed=2)
    net, cm = _net(w, rp, ci, inp)
    # (2P+1)^2 boundary classes + at most one entry per defect (tests/test_oracle_compress.py)
    assert (2 * P + 1) ** 2 <= cm.s.k <= (2 * P + 1) ** 2 + ndef
    grp, gci = net.get_topology()
    assert np.array_equal(grp, rp) and np.array_equal(gci, ci)
    a, b = net.get_topology(w.n // 3, 77)
    assert np.array_equal(b, ci[rp[w.n // 3]:rp[w.n // 3 + 77]])
    onet = _oracle(w, rp, ci, inp)
    assert H.rel_maxnorm(net.eval_rhs(), onet.rhs(inp["y0"]), H.rhs_floor(w)) <= H.TOL_RHS[w.dtype]
    net.integrate(100, w.dt)
    assert H.traj_err(w, net.get_state(), onet.rk4(inp["y0"], 100, w.dt)) <= H.TOL_TRAJ[w.dtype]
    th = onet.phase(onet.rk4(inp["y0"], 100, w.dt))
    if w.dtype == "f64":
        np.testing.assert_allclose(net.observable(B.OBS_LOCAL_ORDER), onet.local_order(th), atol=1e-8)
    net.close()


def test_compressed_ring_and_random_graph():
    # ring: one empty table entry, every row takes the shifted-common-pattern path
    w = configs.get("1", n=300)
    rp, ci = ora.topology_ring(w.n, w.radius)
    inp = H.make_inputs(w, seed=5)
    net, cm = _net(w, rp, ci, inp)
    assert cm.s.k == 1 and cm.s.d_ptr[1] == 0
    assert net.degree() == (w.n * 2 * w.radius, 2 * w.radius)
    onet = _oracle(w, rp, ci, inp)
    net.integrate(100, w.dt)
    assert H.traj_err(w, net.get_state(), onet.rk4(inp["y0"], 100, w.dt)) <= H.TOL_TRAJ["f64"]
    # random graph: nothing is shared, the table has about one entry per row; still exact
    w = configs.get("4", n=3000)
    rp, ci = ora.topology_random_indegree(w.n, w.in_degree, 7)
    inp = H.make_inputs(w, seed=5)
    net, cm = _net(w, rp, ci, inp)
    grp, gci = net.get_topology()
    assert np.array_equal(grp, rp) and np.array_equal(gci, ci)
    onet = _oracle(w, rp, ci, inp)
    assert H.rel_maxnorm(net.eval_rhs(), onet.rhs(inp["y0"]), 1.0) <= H.TOL_RHS["f64"]


def test_compressed_rejects_inconsistent_input():
    w = configs.get("1", n=64)
    rp, ci = ora.topology_ring(64, 5)
    cm = B.net_compress_csr(rp, ci)
    with pytest.raises(B.OscnetError):
        B.Net(w.model, B.F64, 65, dict(kind=B.TOPO_COMPRESSED, compressed=cm), w.params)   # n mismatch
    with pytest.raises(B.OscnetError):
        B.Net(w.model, B.F64, 64, dict(kind=B.TOPO_COMPRESSED, compressed=cm), w.params, method=B.METHOD_FAST)
