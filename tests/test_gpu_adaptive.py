"""Dormand-Prince 5(4) with on-device step control (net_integrate_adaptive; SURVEY.md 8(f).2,
PAPER.md:99, reading R15) against the pinned oracle (tests/test_oracle_dp5.py): the same
accepted / rejected step counts, the same time reached and the state to 1e-9 (fp64) at t_end, on
every kernel family (ring prefix sums, field-split lattice, pair lattice, blocked CSR, DIRECT)."""
from dataclasses import replace

import numpy as np
import pytest

import harness as H
from paper_2410_19075_b200 import binding as B, configs

pytestmark = pytest.mark.gpu

CASES = [
    ("cfg 1 ring", configs.get("1"), 25.0, 1e-6, 1e-9, 0.05, 0),
    ("cfg 2 ring N=4096", configs.get("2", n=4096), 4.0, 1e-6, 1e-8, 0.01, 0),
    ("cfg 3b lattice 20^3", configs.get("3b", n1=20), 5.0, 1e-6, 1e-9, 0.05, 0),
    ("cfg 4 graph N=20000", configs.get("4", n=20000), 6.0, 1e-5, 1e-7, 0.01, 0),
    ("cfg 4 graph N=40000 blocked", replace(configs.get("4", n=40000), in_degree=20), 3.0, 1e-5, 1e-7, 0.01, 0),
    ("cfg 5 lattice 32^3 (f64 state)", replace(configs.get("5", n1=32), dtype="f64"), 1.0, 1e-6, 1e-8, 0.01, 0),
    ("cfg 6 KSI lattice 12^3", configs.get("6", n1=12), 5.0, 1e-7, 1e-10, 0.05, 0),
    ("cfg 3b direct", configs.get("3b", n1=12), 3.0, 1e-6, 1e-9, 0.05, 1),
]


@pytest.mark.parametrize("name,w,t_end,rtol,atol,h0,method", CASES, ids=[c[0] for c in CASES])
def test_dp5_matches_oracle(name, w, t_end, rtol, atol, h0, method):
    inp = H.make_inputs(w, seed=2)
    ref, rinfo = H.make_oracle(w, inp).dp5(inp["y0"], 0.0, t_end, rtol, atol, h0)
    net = H.make_gpu(w, inp, method)
    info = net.integrate_adaptive(t_end, rtol, atol, h0)
    assert (info["accepted"], info["rejected"]) == (rinfo["accepted"], rinfo["rejected"]), (info, rinfo)
    assert info["t"] == t_end and net.time()[0] == t_end and net.time()[1] == info["accepted"]
    assert abs(info["h_next"] - rinfo["h_next"]) <= 1e-9 * rinfo["h_next"]
    assert H.traj_err(w, net.get_state(), ref) <= H.TOL_TRAJ["f64"]
    assert rinfo["accepted"] >= 5
    net.close()


def test_dp5_continues_and_mixes_with_rk4():
    """Two adaptive calls in a row and a fixed-step call in between keep time and state consistent;
    the exchange fields of the lattice kernels are rebuilt after the adaptive call."""
    w = configs.get("3b", n1=16)
    inp = H.make_inputs(w, seed=3)
    onet = H.make_oracle(w, inp)
    net = H.make_gpu(w, inp)
    i1 = net.integrate_adaptive(1.0, 1e-6, 1e-9, 0.05)
    y1, r1 = onet.dp5(inp["y0"], 0.0, 1.0, 1e-6, 1e-9, 0.05)
    net.integrate(10, w.dt)
    y2 = onet.rk4(y1, 10, w.dt)
    t2 = net.time()[0]
    i3 = net.integrate_adaptive(t2 + 1.0, 1e-6, 1e-9, i1["h_next"])
    y3, r3 = onet.dp5(y2, t2, t2 + 1.0, 1e-6, 1e-9, r1["h_next"])
    assert (i3["accepted"], i3["rejected"]) == (r3["accepted"], r3["rejected"])
    assert H.traj_err(w, net.get_state(), y3) <= H.TOL_TRAJ["f64"]


def test_dp5_f32_and_errors():
    w = configs.get("5", n1=24)                # fp32 state: the controller still runs in double
    inp = H.make_inputs(w, seed=4)
    ref, rinfo = H.make_oracle(w, inp).dp5(inp["y0"], 0.0, 0.5, 1e-4, 1e-6, 0.01)
    net = H.make_gpu(w, inp)
    info = net.integrate_adaptive(0.5, 1e-4, 1e-6, 0.01)
    assert abs(info["accepted"] - rinfo["accepted"]) <= 1 and info["t"] == 0.5
    assert H.traj_err(w, net.get_state(), ref) <= 1e-3
    with pytest.raises(B.OscnetError):
        net.integrate_adaptive(0.2, 1e-4, 1e-6, 0.01)          # t_end behind the net's time
    with pytest.raises(B.OscnetError):
        net.integrate_adaptive(1.0, 1e-4, 1e-6, -1.0)
    with pytest.raises(B.OscnetError) as ei:
        net.integrate_adaptive(50.0, 1e-10, 1e-12, 1e-6, max_attempts=5)
    assert "max_attempts" in str(ei.value)


@pytest.mark.parametrize("name,w,method", [("cfg 1 ring", configs.get("1"), 0), ("cfg 3b lattice 16^3", configs.get("3b", n1=16), 0),
                                           ("cfg 4 graph N=5000", configs.get("4", n=5000), 0),
                                           ("cfg 5 lattice 24^3 f32", configs.get("5", n1=24), 0)],
                         ids=["ring", "lattice", "graph", "lattice_f32"])
def test_dp5_dense_output_matches_oracle(name, w, method):
    """Dense output (CONTD5 interpolant evaluated on the device after each accepted step) at output
    times that fall inside steps, several in one step, and on the end point; the step sequence is the
    one of the run without outputs."""
    inp = H.make_inputs(w, seed=3)
    T = 2.0 if w.dtype == "f64" else 0.4
    t_out = np.array([0.013, 0.0131, 0.25, 0.5, 0.77, 0.9999, 1.0]) * T
    rtol, atol = (1e-6, 1e-9) if w.dtype == "f64" else (1e-4, 1e-6)
    ref, rinfo = H.make_oracle(w, inp).dp5_dense(inp["y0"], 0.0, t_out, rtol, atol, 0.01)
    net = H.make_gpu(w, inp, method)
    out, info = net.integrate_adaptive_dense(t_out, rtol, atol, 0.01)
    if w.dtype == "f64":
        assert (info["accepted"], info["rejected"]) == (rinfo["accepted"], rinfo["rejected"])
        for q in range(len(t_out)):
            assert H.traj_err(w, out[q], ref[q]) <= H.TOL_TRAJ["f64"], q
        # theta = 1: y + (y5 - y), the state itself up to one rounding
        np.testing.assert_allclose(out[-1], net.get_state(), rtol=1e-14, atol=1e-13)
    else:
        assert abs(info["accepted"] - rinfo["accepted"]) <= 1
        assert np.abs(out.astype(np.float64) - ref).max() <= 1e-3
    assert net.time()[0] == t_out[-1]
    with pytest.raises(B.OscnetError):
        net.integrate_adaptive_dense(np.array([t_out[-1] + 1.0, t_out[-1] + 0.5]), rtol, atol, 0.01)   # not ascending
    with pytest.raises(B.OscnetError):
        net.integrate_adaptive_dense(np.array([t_out[-1]]), rtol, atol, 0.01)                           # not after the net's time
    net.close()
