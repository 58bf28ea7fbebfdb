"""GPU parity of the column-blocked shared-memory CSR kernels (csr_blocked.cu) against the
oracle: single RHS and 100 RK4 steps, at geometries that span several column blocks, several
row chunks per CTA, several rows per thread and ragged tails.  OSCNET_CSRB = "W,CR" forces the
block width / chunk length (read by the library when the net is created)."""
import os
from dataclasses import replace

import numpy as np
import pytest

import harness as H
from paper_2410_19075_b200 import configs

pytestmark = pytest.mark.gpu

FAMILY_CSR_WARP, FAMILY_CSR_BLOCKED = 1, 7

# (n, in-degree, "W,CR" or None for the library's own choice, dtype)
CASES = [
    (20000, 100, "512,96", "f64"),      # 40 blocks, 209 chunks > 148 CTAs, M = 1
    (20000, 20, "4096,1024", "f64"),    # 5 blocks, 20 chunks, ragged last block and chunk, 20 % overflow
    (20011, 37, "1000,2500", "f64"),    # odd sizes, M = 3
    (9000, 64, "16,8192", "f64"),       # blocks of 16 columns (563 of them), M = 8... one chunk pair
    (50000, 20, None, "f64"),           # library geometry (n >= 32768): 2 blocks
    (20000, 20, "4096,1024", "f32"),
]
IDS = ["n%d-k%d-%s-%s" % (n, k, g or "auto", dt) for n, k, g, dt in CASES]


@pytest.fixture
def csrb_env():
    old = os.environ.get("OSCNET_CSRB")
    yield
    if old is None:
        os.environ.pop("OSCNET_CSRB", None)
    else:
        os.environ["OSCNET_CSRB"] = old


def workload(n, k, dtype):
    w = configs.get("4", n=n)
    return replace(w, in_degree=k, dtype=dtype, name="HH random CSR N=%d k=%d %s" % (n, k, dtype))


def make(n, k, geom, dtype, seed):
    if geom is None:
        os.environ.pop("OSCNET_CSRB", None)
    else:
        os.environ["OSCNET_CSRB"] = geom
    w = workload(n, k, dtype)
    inp = H.make_inputs(w, seed=seed)
    net = H.make_gpu(w, inp)
    assert net.kernel_family() == FAMILY_CSR_BLOCKED
    return w, inp, net


@pytest.mark.parametrize("n,k,geom,dtype", CASES, ids=IDS)
def test_rhs_parity_blocked(csrb_env, n, k, geom, dtype):
    w, inp, net = make(n, k, geom, dtype, 1)
    onet = H.make_oracle(w, inp)
    got = net.eval_rhs()
    assert np.isfinite(got).all()
    assert H.rel_maxnorm(got, onet.rhs(inp["y0"]), H.rhs_floor(w)) <= H.TOL_RHS[dtype]
    y1 = H.perturb_gates(w, inp["y0"])
    net.set_state(y1)
    assert H.rel_maxnorm(net.eval_rhs(), onet.rhs(y1)) <= H.TOL_RHS[dtype]


@pytest.mark.parametrize("n,k,geom,dtype", CASES[:3] + CASES[4:5], ids=IDS[:3] + IDS[4:5])
def test_trajectory_blocked(csrb_env, n, k, geom, dtype):
    w, inp, net = make(n, k, geom, dtype, 2)
    ref = H.make_oracle(w, inp).rk4(inp["y0"], 100, w.dt)
    net.integrate(100, w.dt)
    assert H.traj_err(w, net.get_state(), ref) <= H.TOL_TRAJ[dtype]


def test_blocked_matches_warp_kernel_on_given_csr(csrb_env):
    """A CSR handed in by the caller (variable degree, one empty row, one hub row) through both
    kernel families: same sums up to the summation order."""
    from paper_2410_19075_b200 import binding as B
    rng = np.random.default_rng(5)
    n = 6000
    deg = rng.integers(0, 60, size=n)
    deg[17] = 0
    deg[4001] = 3000
    rows = [np.sort(rng.choice(n, size=d, replace=False)).astype(np.int32) for d in deg]
    rp = np.concatenate([[0], np.cumsum(deg)]).astype(np.int64)
    ci = np.concatenate(rows).astype(np.int32)
    w = workload(n, 1, "f64")
    inp = H.make_inputs(w, seed=3)
    out = []
    for geom, fam in (("700,640", FAMILY_CSR_BLOCKED), (None, FAMILY_CSR_WARP)):
        if geom is None:
            os.environ.pop("OSCNET_CSRB", None)
        else:
            os.environ["OSCNET_CSRB"] = geom
        net = B.Net(w.model, B.F64, n, dict(kind=B.TOPO_CSR, row_ptr=rp, col_idx=ci), w.params)
        assert net.kernel_family() == fam
        net.set_state(inp["y0"])
        net.set_param_array(B.PARAM_IEXT, inp["elem"])
        out.append(net.eval_rhs())
        net.integrate(20, w.dt)
        out.append(net.get_state())
    from oracle import oracle as ora
    onet = ora.OracleNet.hh(n, rp, ci, inp["elem"], **w.params)
    assert H.rel_maxnorm(out[0], onet.rhs(inp["y0"]), 1.0) <= 1e-12
    assert H.rel_maxnorm(out[0], out[2], 1.0) <= 1e-12
    assert np.abs(out[1] - out[3]).max() <= 1e-9
