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
