"""Second-workload models of SURVEY.md 8(f).4 on the GPU against the pinned oracle
(tests/test_oracle_eq12.py): FitzHugh-Nagumo exactly as eq. (2) with delay tau = delay_steps * dt,
noise and applied current (NET_MODEL_FHN2, reading R17), Hodgkin-Huxley with the synaptic gating
ODE of eq. (1) (NET_MODEL_HHS, reading R18); rings, 2D discs, 3D balls, graphs."""
import numpy as np
import pytest

import harness as H
from oracle import oracle as ora
from paper_2410_19075_b200 import binding as B, configs

pytestmark = pytest.mark.gpu

P2 = dict(eps=0.05, a=0.5, sigma=0.3, I_app=0.1)


def _topo(kind, n):
    if kind == "ring":
        return dict(kind=B.TOPO_RING, radius=11), ora.topology_ring(n, 11)
    if kind == "disc":                       # 2D periodic lattice, disc of radius 3
        return dict(kind=B.TOPO_LATTICE, extent=(24, 20), radius=3), ora.topology_lattice((24, 20), 3)
    if kind == "ball":
        return dict(kind=B.TOPO_LATTICE, extent=(10, 8, 6), radius=2), ora.topology_lattice((10, 8, 6), 2)
    return dict(kind=B.TOPO_RANDOM_INDEGREE, in_degree=9, seed=4), ora.topology_random_indegree(n, 9, 4)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kind,m,D", [("ring", 0, 0.0), ("ring", 1, 0.0), ("ring", 7, 0.05), ("disc", 5, 0.0),
                                      ("ball", 3, 0.02), ("graph", 12, 0.0), ("graph", 2, 0.1)])
def test_fhn2_delay_noise_matches_oracle(kind, m, D, dtype):
    n = 480
    topo, (rp, ci) = _topo(kind, n)
    rng = np.random.default_rng(8)
    npdt = np.float32 if dtype == "f32" else np.float64
    y0 = rng.uniform(-1.5, 1.5, size=(2, n)).astype(npdt).astype(np.float64)
    onet = ora.OracleNet.fhn2(n, rp, ci, **P2)
    net = B.Net(B.MODEL_FHN2, B.F32 if dtype == "f32" else B.F64, n, topo, dict(P2, D=D, seed=21), delay_steps=m)
    net.set_state(y0.astype(npdt))
    grp, gci = net.get_topology()
    assert np.array_equal(grp, rp) and np.array_equal(gci, ci)
    assert H.rel_maxnorm(net.eval_rhs(), onet.rhs(y0)) <= H.TOL_RHS[dtype]
    dt = 0.01
    net.integrate(60, dt)                                  # two calls: the history carries over
    net.integrate(40, dt)
    ref, _ = onet.fhn2_rk4(y0, 100, dt, m=m, D=D, seed=21)
    assert np.abs(net.get_state().astype(np.float64) - ref).max() <= H.TOL_TRAJ[dtype]
    # a new state resets the history to the constant initial function
    net.set_state(y0.astype(npdt))
    net.integrate(25, dt)
    ref2, _ = onet.fhn2_rk4(y0, 25, dt, m=m, D=D, seed=21)
    assert np.abs(net.get_state().astype(np.float64) - ref2).max() <= H.TOL_TRAJ[dtype]
    net.close()


def test_fhn2_statistics_and_refusals():
    n = 400
    topo, (rp, ci) = _topo("ring", n)
    y0 = np.random.default_rng(9).uniform(-1.5, 1.5, size=(2, n))
    net = B.Net(B.MODEL_FHN2, B.F64, n, topo, dict(P2, D=0.0), delay_steps=4)
    net.set_state(y0)
    got = net.integrate_observed(200, 0.01, 10)
    assert got["n_samples"] == 11 and 0.0 <= got["R_mean"] <= 1.0
    with pytest.raises(B.OscnetError):                      # adaptive steps cannot carry the fixed-step history
        net.integrate_adaptive(5.0, 1e-6, 1e-9, 0.01)
    with pytest.raises(B.OscnetError):                      # a delay on a model that has none
        B.Net(B.MODEL_FHN, B.F64, n, topo, dict(eps=0.05, a=0.5, sigma=0.1, phi=1.0), delay_steps=3)
    nodelay = B.Net(B.MODEL_FHN2, B.F64, n, topo, dict(P2))
    nodelay.set_state(y0)
    info = nodelay.integrate_adaptive(1.0, 1e-6, 1e-9, 0.01)          # no delay, no noise: allowed
    ref, rinfo = ora.OracleNet.fhn2(n, rp, ci, **P2).dp5(y0, 0.0, 1.0, 1e-6, 1e-9, 0.01)
    assert info["accepted"] == rinfo["accepted"] and np.abs(nodelay.get_state() - ref).max() <= 1e-9


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kind", ["graph", "ring", "ball"])
def test_hhs_gating_ode_matches_oracle(kind, dtype):
    n = 480
    topo, (rp, ci) = _topo(kind, n)
    rng = np.random.default_rng(10)
    npdt = np.float32 if dtype == "f32" else np.float64
    V = (-70 + 20 * rng.random(n)).astype(npdt).astype(np.float64)
    Iext = (9 + 2 * rng.random(n)).astype(npdt).astype(np.float64)
    onet = ora.OracleNet.hhs(n, rp, ci, Iext, a_s=2.0, b_s=0.5)
    net = B.Net(B.MODEL_HHS, B.F32 if dtype == "f32" else B.F64, n, topo, dict(configs._HH, a_s=2.0, b_s=0.5))
    y0 = np.zeros((5, n))
    y0[0] = V
    net.set_state(y0.astype(npdt))
    net.set_param_array(B.PARAM_IEXT, Iext.astype(npdt))
    net.hh_steady_gates()
    y0 = net.get_state().astype(np.float64)
    m, h, g = ora.hh_steady_gates(V)
    S = 1 / (1 + np.exp(-V / 2.0))
    np.testing.assert_allclose(y0[1:], np.stack([m, h, g, 2 * S / (2 * S + 0.5)]), rtol=0, atol=1e-14 if dtype == "f64" else 1e-6)
    y1 = y0.copy()
    y1[1:] = np.clip(y1[1:] * rng.uniform(0.5, 1.5, size=(4, n)), 0, 1).astype(npdt)
    net.set_state(y1.astype(npdt))
    # graphs: warp-per-row gathers of the gate (FAST); rings and lattices: the per-link form
    assert net.counters()[1] == (B.METHOD_FAST if kind == "graph" else B.METHOD_DIRECT)
    assert H.rel_maxnorm(net.eval_rhs(), onet.rhs(y1)) <= H.TOL_RHS[dtype]
    net.integrate(100, 0.01)
    got, ref = net.get_state().astype(np.float64), onet.rk4(y1, 100, 0.01)
    # fp32: V is ~70 mV, one fp32 rounding of it is already 8e-6 -- the 1e-4 is taken relative to the
    # size of each variable (the north star states its fp32 tolerance for O(1) phases)
    scale = np.abs(ref).max(axis=1, keepdims=True).clip(1.0) if dtype == "f32" else 1.0
    assert (np.abs(got - ref) / scale).max() <= H.TOL_TRAJ[dtype]
    th = onet.phase(onet.rk4(y1, 100, 0.01))
    assert np.abs(net.observable(B.OBS_PHASE) - th).max() <= (1e-9 if dtype == "f64" else 1e-3)
    net.close()
