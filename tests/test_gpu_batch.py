"""Batches of independent rings (net_desc.batch > 1, "a large number
of network instances simultaneously"): the batch is one block-diagonal net, so the oracle of the
batch is the plain definition on the block-diagonal CSR; replica r must also equal the same ring
integrated alone (no leakage between replicas)."""
from dataclasses import replace

import numpy as np
import pytest

import harness as H
from paper_2410_19075_b200 import binding as B, configs

pytestmark = pytest.mark.gpu

CASES = [
    ("1", dict(n=256), 5),       # config 1 itself, five replicas
    ("1", dict(n=300), 3),       # ragged: 300 elements on 512 lanes (E = 2)
    ("2", dict(n=1024), 4),      # FHN ring, R = 358
    ("2", dict(n=2000), 2),      # E = 8, ragged tail
]


def _w(cfg, kw, batch):
    w = configs.get(cfg, **kw)
    return replace(w, batch=batch, name=w.name + " x %d" % batch)


@pytest.mark.parametrize("cfg,kw,batch", CASES)
@pytest.mark.parametrize("method", [B.METHOD_FAST, B.METHOD_DIRECT])
def test_batch_matches_block_diagonal_oracle(cfg, kw, batch, method):
    w = _w(cfg, kw, batch)
    inp = H.make_inputs(w, seed=3)
    onet = H.make_oracle(w, inp)
    net = H.make_gpu(w, inp, method=method)
    assert net.counters()[1] == method
    # topology: bit-exact block-diagonal CSR, element ids 0 .. batch*n - 1
    rp, ci = net.get_topology()
    rp0, ci0 = H.oracle_topology(w)
    assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0)
    e_rhs = H.rel_maxnorm(net.eval_rhs(), onet.rhs(inp["y0"]), H.rhs_floor(w))
    assert e_rhs <= H.TOL_RHS[w.dtype], e_rhs
    net.integrate(100, w.dt)
    e_tr = H.traj_err(w, net.get_state(), onet.rk4(inp["y0"], 100, w.dt))
    assert e_tr <= H.TOL_TRAJ[w.dtype], e_tr
    net.close()


def test_replica_equals_the_ring_integrated_alone():
    w = _w("1", dict(n=256), 4)
    inp = H.make_inputs(w, seed=5)
    net = H.make_gpu(w, inp, method=B.METHOD_FAST)
    net.integrate(50, w.dt)
    got = net.get_state().reshape(w.nvar, w.batch, w.n)
    net.close()
    w1 = configs.get("1", n=256)
    for r in (0, 3):
        sl = slice(r * w.n, (r + 1) * w.n)
        inp1 = dict(y0=inp["y0"][:, sl].copy(), elem=inp["elem"][sl].copy())
        # a batch runs 128 threads per ring, a single ring 256 (measured, ring_fast.cu: ring_plan): with
        # the same thread count the two are the same kernel and the same arithmetic -- bit-identical;
        # with the defaults only the order of the scan differs
        import os
        os.environ["OSCNET_RING_NT"] = "128"
        try:
            n1 = H.make_gpu(w1, inp1, method=B.METHOD_FAST)
            n1.integrate(50, w.dt)
            alone = n1.get_state()
            n1.close()
        finally:
            del os.environ["OSCNET_RING_NT"]
        assert np.array_equal(got[:, r, :], alone)
        n2 = H.make_gpu(w1, inp1, method=B.METHOD_FAST)
        n2.integrate(50, w.dt)
        assert np.abs(got[:, r, :] - n2.get_state()).max() <= 1e-12
        n2.close()


@pytest.mark.parametrize("cfg,kw,batch", [("5", dict(n1=10), 3), ("3b", dict(n1=9), 2), ("4", dict(n=700), 4),
                                          ("6", dict(n1=8), 2), ("3a", dict(n1=12), 2)])
def test_batches_of_lattices_and_graphs(cfg, kw, batch):
    """batch > 1 on every topology kind (batch is a property of net_create): the
    block-diagonal net on the per-link kernels; topology bit-exact, RHS and 100 steps within the
    north star's tolerances against the oracle on the block-diagonal CSR, replica = the net alone."""
    w = replace(configs.get(cfg, **kw), batch=batch)
    inp = H.make_inputs(w, seed=6)
    onet = H.make_oracle(w, inp)
    net = H.make_gpu(w, inp)
    assert net.counters()[1] == B.METHOD_DIRECT
    rp, ci = net.get_topology()
    rp0, ci0 = H.oracle_topology(w)
    assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0)
    a, b = net.get_topology(w.n - 3, 7)                    # a range that straddles two replicas
    a0, b0 = H.oracle_topology(w, w.n - 3, 7)
    assert np.array_equal(a, a0) and np.array_equal(b, b0)
    assert H.rel_maxnorm(net.eval_rhs(), onet.rhs(inp["y0"]), H.rhs_floor(w)) <= H.TOL_RHS[w.dtype]
    net.integrate(100, w.dt)
    got = net.get_state()
    assert H.traj_err(w, got, onet.rk4(inp["y0"], 100, w.dt)) <= H.TOL_TRAJ[w.dtype]
    w1 = replace(w, batch=1)
    r = batch - 1
    sl = slice(r * w.n, (r + 1) * w.n)
    inp1 = dict(y0=inp["y0"][:, sl].copy(), elem=None if inp["elem"] is None else inp["elem"][sl].copy())
    n1 = H.make_gpu(w1, inp1, method=B.METHOD_DIRECT)
    n1.integrate(100, w.dt)
    assert np.array_equal(got[:, sl], n1.get_state())      # same kernel, same arithmetic: bit-identical
    rep = net.observable(B.OBS_REPLICA_ORDER).reshape(batch, 2)
    assert abs(rep[r, 0] - n1.observable(B.OBS_GLOBAL_ORDER)[0]) < 1e-12


def test_batch_refusals():
    w = replace(configs.get("5", n1=16), batch=2)
    with pytest.raises(B.OscnetError) as ei:               # the tiled lattice kernels take one lattice
        B.Net.from_workload(w, method=B.METHOD_FAST)
    assert ei.value.code == -5
    w = replace(configs.get("1"), batch=0)
    with pytest.raises(B.OscnetError) as ei:
        B.Net.from_workload(w)
    assert ei.value.code == -1


def test_replica_order_parameter_matches_oracle_per_ring():
    """NET_OBS_REPLICA_ORDER: {R_r, Psi_r} of every replica = the oracle's global order parameter of
    that ring's phases alone; the ensemble value (NET_OBS_GLOBAL_ORDER) = the oracle's over all."""
    from oracle import oracle as ora
    for cfg, kw, batch in (("1", dict(n=256), 6), ("2", dict(n=1024), 3)):
        w = _w(cfg, kw, batch)
        inp = H.make_inputs(w, seed=9)
        onet = H.make_oracle(w, inp)
        net = H.make_gpu(w, inp)
        net.integrate(20, w.dt)
        y = net.get_state().astype(np.float64)
        theta = net.observable(B.OBS_PHASE)
        got = net.observable(B.OBS_REPLICA_ORDER).reshape(batch, 2)
        ens = net.observable(B.OBS_GLOBAL_ORDER)
        net.close()
        th_ref = y[0] if w.model == configs.KS else np.arctan2(y[1], y[0])
        np.testing.assert_allclose(theta, th_ref, atol=1e-13)
        ring = ora.OracleNet.ks(w.n, *ora.topology_ring(w.n, w.radius), 1.0, 0.0, np.zeros(w.n))
        for r in range(batch):
            R, Psi = ring.global_order(th_ref[r * w.n:(r + 1) * w.n])
            assert abs(got[r, 0] - R) < 1e-13
            assert abs(np.angle(np.exp(1j * (got[r, 1] - Psi)))) < 1e-11
        R, Psi = onet.global_order(th_ref)
        assert abs(ens[0] - R) < 1e-13
