"""Kuramoto-Sakaguchi with inertia (eq. (3) in full): the persistent
ring kernel (FAST) for rings, the field-split lattice kernels (FAST) for 3D balls of radius 2 / 4, the
per-link DIRECT form elsewhere; parity with the pinned oracle (tests/test_oracle_dynamics.py::test_ksi_*)
on every topology kind, both dtypes."""
from dataclasses import replace

import numpy as np
import pytest

import harness as H
from paper_2410_19075_b200 import binding as B, configs

pytestmark = pytest.mark.gpu

P6 = dict(K=0.32, alpha=0.45, m=1.0, eps=0.05, omega0=0.0)


def _cases():
    base = configs.get("6", n1=12)                                   # 3D ball of radius 2, 1728 elements
    ring = replace(base, topo=configs.RING, n=1000, extent=(), radius=37, name="KSI ring N=1000 P=37",
                   params=dict(P6, K=1.0, m=0.7, eps=0.2, omega0=0.3))
    lat2 = replace(base, n=23 * 17, extent=(23, 17), radius=3, name="KSI 2D 23x17 radius 3")
    rnd = replace(base, topo=configs.RANDOM_INDEGREE, n=3000, extent=(), radius=0, in_degree=20,
                  name="KSI random graph N=3000 k=20", params=dict(P6, K=0.8))
    out = []
    for w in (base, ring, lat2, rnd):
        out.append(w)
        out.append(replace(w, dtype="f32", name=w.name.replace("f64", "f32") + " (f32)"))
    return out


@pytest.mark.parametrize("w", _cases(), ids=lambda w: w.name)
def test_ksi_direct_matches_oracle(w):
    inp = H.make_inputs(w, seed=4)
    onet = H.make_oracle(w, inp)
    net = H.make_gpu(w, inp)
    launches, method = net.counters()
    # rings: the persistent prefix-sum kernel; 3D balls: the field-split lattice kernels; graphs:
    # warp-per-row gathers (all FAST); 2D lattices: the per-link DIRECT form
    fast = w.topo != configs.LATTICE or len(w.extent) == 3
    assert method == (B.METHOD_FAST if fast else B.METHOD_DIRECT)
    rp, ci = net.get_topology()
    rp0, ci0 = H.oracle_topology(w)
    assert np.array_equal(rp, rp0) and np.array_equal(ci, ci0)
    e_rhs = H.rel_maxnorm(net.eval_rhs(), onet.rhs(inp["y0"]))
    assert e_rhs <= H.TOL_RHS[w.dtype], e_rhs
    net.integrate(100, w.dt)
    got = net.get_state().astype(np.float64)
    ref = onet.rk4(inp["y0"], 100, w.dt)
    assert np.abs(got - ref).max() <= H.TOL_TRAJ[w.dtype], np.abs(got - ref).max()
    # observables see the phase variable
    R, Psi = onet.global_order(ref[0])
    assert abs(net.observable(B.OBS_GLOBAL_ORDER)[0] - R) < (1e-9 if w.dtype == "f64" else 1e-4)
    net.close()


@pytest.mark.parametrize("method", [B.METHOD_FAST, B.METHOD_DIRECT])
@pytest.mark.parametrize("batch", [1, 3])
def test_ksi_ring_fast_and_direct_and_batches(method, batch):
    ring = [w for w in _cases() if w.topo == configs.RING and w.dtype == "f64"][0]
    w = replace(ring, n=700, batch=batch, name=ring.name + " x %d" % batch)
    inp = H.make_inputs(w, seed=6)
    onet = H.make_oracle(w, inp)
    net = H.make_gpu(w, inp, method=method)
    assert net.counters()[1] == method
    assert H.rel_maxnorm(net.eval_rhs(), onet.rhs(inp["y0"])) <= H.TOL_RHS["f64"]
    net.integrate(100, w.dt)
    assert np.abs(net.get_state() - onet.rk4(inp["y0"], 100, w.dt)).max() <= H.TOL_TRAJ["f64"]
    net.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n1,radius", [(12, 2), (20, 4), (36, 2), (16, 6)])
def test_ksi_lattice_fast_and_direct(n1, radius, dtype):
    """The paper's performance model (Fig. 6c) on the field-split lattice kernels: RHS instance of the
    KS kernel + one pointwise update of (phi, psi); FAST against the oracle and against DIRECT."""
    w = replace(configs.get("6", n1=n1), radius=radius, dtype=dtype,
                name="KSI 3D %d^3 radius %d %s" % (n1, radius, dtype))
    inp = H.make_inputs(w, seed=5)
    onet = H.make_oracle(w, inp)
    fast = H.make_gpu(w, inp, method=B.METHOD_FAST)
    assert fast.kernel_family() == 6
    direct = H.make_gpu(w, inp, method=B.METHOD_DIRECT)
    ref = onet.rhs(inp["y0"])
    assert H.rel_maxnorm(fast.eval_rhs(), ref) <= H.TOL_RHS[dtype]
    assert H.rel_maxnorm(fast.eval_rhs(), direct.eval_rhs()) <= 2 * H.TOL_RHS[dtype]
    fast.integrate(37, w.dt)
    fast.integrate(63, w.dt)
    got = fast.get_state().astype(np.float64)
    assert H.traj_err(w, got, onet.rk4(inp["y0"], 100, w.dt)) <= H.TOL_TRAJ[dtype]
    # RHS after steps: the exchange field of the current state is the one the last stage left
    assert H.rel_maxnorm(fast.eval_rhs(), onet.rhs(got)) <= 10 * H.TOL_RHS[dtype]
    fast.close(); direct.close()


def test_ksi_fast_is_refused_on_2d_lattices_and_mass_must_be_positive():
    w = replace(configs.get("6", n1=12), n=23 * 17, extent=(23, 17), radius=3)
    with pytest.raises(B.OscnetError) as ei:
        B.Net.from_workload(w, method=B.METHOD_FAST)
    assert ei.value.code == -5
    w = configs.get("6", n1=12)
    bad = replace(w, params=dict(P6, m=0.0))
    with pytest.raises(B.OscnetError) as ei:
        B.Net.from_workload(bad)
    assert ei.value.code == -1

