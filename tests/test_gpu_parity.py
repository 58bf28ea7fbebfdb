"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are the north star's (tests/harness.py)."""
from dataclasses import replace

import numpy as np
import pytest

import harness as H
from paper_2410_19075_b200 import configs

pytestmark = pytest.mark.gpu

DIRECT, FAST_OR_AUTO = 1, 0


def B():
    from paper_2410_19075_b200 import binding
    return binding


def small_workloads():
    w3 = configs.get("3a", n1=20)
    return [
        configs.get("1"),
        configs.get("2", n=2048),
        w3,
        configs.get("3b", n1=20),
        replace(configs.get("3b", n1=12), extent=(24, 12, 10), n=24 * 12 * 10, name="KS 3D 24x12x10 f64"),
        replace(configs.get("3a", n1=9), name="KS 3D 9^3 f32 (ragged, not a multiple of 4)"),
        configs.get("4", n=20000),
        configs.get("5", n1=32),
        replace(configs.get("5", n1=12), extent=(36, 20, 12), n=36 * 20 * 12, name="FHN 3D 36x20x12 f32"),
        replace(configs.get("5", n1=7), name="FHN 3D 7^3 f32 (ragged)"),
    ]


SMALL = small_workloads()
IDS = [w.name for w in SMALL]


@pytest.mark.parametrize("method", [DIRECT, FAST_OR_AUTO], ids=["direct", "auto"])
@pytest.mark.parametrize("w", SMALL, ids=IDS)
def test_rhs_parity(w, method):
    inp = H.make_inputs(w, seed=1)
    ref = H.make_oracle(w, inp).rhs(inp["y0"])
    net = H.make_gpu(w, inp, method)
    got = net.eval_rhs()
    assert np.isfinite(got).all()
    assert H.rel_maxnorm(got, ref, H.rhs_floor(w)) <= H.TOL_RHS[w.dtype]
    if w.model == configs.HH:       # gates off their steady state: pure relative norm
        y1 = H.perturb_gates(w, inp["y0"])
        net.set_state(y1)
        assert H.rel_maxnorm(net.eval_rhs(), H.make_oracle(w, inp).rhs(y1)) <= H.TOL_RHS[w.dtype]


@pytest.mark.parametrize("method", [DIRECT, FAST_OR_AUTO], ids=["direct", "auto"])
@pytest.mark.parametrize("w", SMALL, ids=IDS)
def test_trajectory_100_steps(w, method):
    inp = H.make_inputs(w, seed=2)
    ref = H.make_oracle(w, inp).rk4(inp["y0"], 100, w.dt)
    net = H.make_gpu(w, inp, method)
    net.integrate(100, w.dt)
    got = net.get_state()
    t, step = net.time()
    assert step == 100 and abs(t - 100 * w.dt) < 1e-12
    assert H.traj_err(w, got, ref) <= H.TOL_TRAJ[w.dtype]


def test_integrate_is_split_invariant():
    # 100 steps = 37 + 63 steps = graph replays + single steps; identical bits
    w = configs.get("5", n1=16)
    inp = H.make_inputs(w, 3)
    a, b = H.make_gpu(w, inp), H.make_gpu(w, inp)
    a.integrate(100, w.dt)
    b.integrate(37, w.dt)
    b.integrate(63, w.dt)
    assert np.array_equal(a.get_state(), b.get_state())


@pytest.mark.parametrize("w", [configs.get("1"), configs.get("2", n=512),
                               configs.with_steps(configs.get("3b", n1=12), 100, 10),
                               configs.with_steps(configs.get("3a", n1=12), 100, 10),
                               configs.with_steps(configs.get("4", n=2000), 1000, 100),
                               configs.with_steps(configs.get("5", n1=16), 200, 10)],
                         ids=lambda w: w.name)
def test_long_run_statistics(w):
    """Order-parameter statistics over the second half of the run (reading R9), 1e-3."""
    inp = H.make_inputs(w, seed=1)
    ref = H.make_oracle(w, inp).run_statistics(inp["y0"], w.n_steps, w.dt, w.obs_every)
    net = H.make_gpu(w, inp)
    got = net.integrate_observed(w.n_steps, w.dt, w.obs_every)
    assert got["n_samples"] == ref["n_samples"]
    for k in ("R_mean", "R_std", "Rloc_mean", "vel_mean", "vel_std"):
        scale = max(1.0, abs(ref[k]))
        assert abs(got[k] - ref[k]) <= H.TOL_STATS * scale, (k, got[k], ref[k])
    vel = net.observable(B().OBS_MEAN_PHASE_VELOCITY)
    assert np.abs(vel - ref["vel"]).max() <= (1e-6 if w.dtype == "f64" else 5e-2)


@pytest.mark.parametrize("w", [configs.get("1"), configs.get("2", n=300), configs.get("3b", n1=10),
                               configs.get("4", n=500), configs.get("5", n1=10), configs.get("3a", n1=12),
                               configs.get("3b", n1=24), replace(configs.get("5", n1=20), dtype="f64"),
                               configs.get("2", n=5000), configs.get("6", n1=12),
                               replace(configs.get("1", n=300), batch=3)],
                         ids=lambda w: w.name)
def test_observables_of_a_state(w):
    inp = H.make_inputs(w, seed=4)
    onet = H.make_oracle(w, inp)
    net = H.make_gpu(w, inp)
    th = onet.phase(inp["y0"])
    np.testing.assert_allclose(net.observable(B().OBS_PHASE), th, atol=1e-12)
    R, Psi = onet.global_order(th)
    g = net.observable(B().OBS_GLOBAL_ORDER)
    assert abs(g[0] - R) < 1e-12 and abs(g[1] - Psi) < 1e-9
    # fp32 lattices: the ball sum of the unit phasors runs in the arithmetic type of the net
    np.testing.assert_allclose(net.observable(B().OBS_LOCAL_ORDER), onet.local_order(th),
                               atol=1e-12 if w.dtype == "f64" else 2e-6)


def test_hh_steady_gates_match_oracle():
    from oracle import oracle as ora
    w = configs.get("4", n=4096)
    inp = H.make_inputs(w, 5)
    y = inp["y0"].copy()
    y[1:] = 0.0
    net = H.make_gpu(w, dict(y0=y, elem=inp["elem"]))
    net.hh_steady_gates()
    got = net.get_state()
    m, h, g = ora.hh_steady_gates(y[0])
    np.testing.assert_allclose(got[1:], np.stack([m, h, g]), rtol=0, atol=1e-14)
    # the removable singularities (V = -40, -55 exactly) on the GPU too
    y2 = y.copy(); y2[0, :4] = [-40.0, -55.0, -40.0 + 1e-11, -55.0 - 1e-11]
    net.set_state(y2)
    ref = H.make_oracle(w, inp).rhs(y2)
    assert H.rel_maxnorm(net.eval_rhs(), ref, 1.0) <= 1e-12


def test_fast_rewrite_error_against_direct_on_gpu():
    """Error of the rewrites, measured on the GPU itself (north star item 3): FAST vs DIRECT in
    an incoherent (random) and a coherent (nearly in-phase) state."""
    for w in (configs.get("3a", n1=24), configs.get("3b", n1=24), configs.get("5", n1=32),
              configs.get("2", n=4096), configs.get("1")):
        for coherent in (False, True):
            inp = H.make_inputs(w, 7)
            if coherent:
                inp["y0"] = inp["y0"] * 1e-2 + 0.3
            fa, di = H.make_gpu(w, inp, FAST_OR_AUTO), H.make_gpu(w, inp, DIRECT)
            err = H.rel_maxnorm(fa.eval_rhs(), di.eval_rhs())
            assert err <= 2 * H.TOL_RHS[w.dtype], (w.name, coherent, err)
