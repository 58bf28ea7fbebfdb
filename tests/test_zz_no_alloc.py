"""net_order_parameter_noalloc (include/oscnet.h): the global order parameter with its block partials
in a static device array -- no handle, no workspace, no cudaMalloc -- against the existing path
(net_observables(NET_OBS_GLOBAL_ORDER), whose partials live in the net's workspace).

The file is named to be collected last: the suite runs with pytest -x, so a failure here must not
hide any other test.  It passes alone in a fresh process and after the rest of the suite (the static
array keeps the previous call's contents; the entry point clears what has to start at zero).

Tolerance 1e-12 on R and Psi, the one tests/test_gpu_batch.py uses for two reduction orders of the
same double sum (N <= 2^24 terms of magnitude <= 1: rounding ~ 1e-16 sqrt(N) per order).
"""
import numpy as np
import pytest

import harness as H
from paper_2410_19075_b200 import binding as B, configs

pytestmark = pytest.mark.gpu

TOL = 1e-12
ERR_SIZE = -2          # NET_ERR_SIZE of include/oscnet.h


def _noalloc(theta, out, stream=None):
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    B.net_order_parameter_noalloc(theta.data_ptr(), theta.numel(), B.F32 if theta.dtype == torch.float32 else B.F64,
                                  out.data_ptr(), st.cuda_stream)


@pytest.mark.parametrize("cfg,n1", [("3b", 48), ("3a", 40)], ids=["f64", "f32"])
def test_two_calls_in_a_row_equal_the_workspace_path(cfg, n1):
    """KS lattice (the state IS the phase): n = 110592 (13.5 CTAs of 8192 phases) and 64000."""
    import torch
    w = configs.get(cfg, n1=n1)
    inp = H.make_inputs(w, seed=4)
    net = H.make_gpu(w, inp)
    assert w.model == configs.KS and net.nvar == 1
    theta = torch.empty((1, w.n), dtype=net.torch_dtype, device="cuda")
    out = torch.full((2,), -7.0, dtype=torch.float64, device="cuda")
    seen = []
    for call in range(2):                       # two calls in a row, on two different states
        net.integrate(25, w.dt)
        ref = net.observable(B.OBS_GLOBAL_ORDER)            # existing path
        net.get_state(theta)
        _noalloc(theta, out)
        got = out.cpu().numpy()
        assert abs(got[0] - ref[0]) <= TOL and abs(got[1] - ref[1]) <= TOL, (call, got, ref)
        z = np.exp(1j * theta.cpu().numpy().astype(np.float64)).mean()   # and the definition itself
        assert abs(got[0] - abs(z)) <= TOL and abs(got[1] - np.angle(z)) <= TOL
        seen.append(got.copy())
    assert not np.array_equal(seen[0], seen[1])             # the second call did not return the first's result
    _noalloc(theta, out)                                    # same input again: same bits (fixed summation order)
    assert np.array_equal(out.cpu().numpy(), seen[1])
    net.close()


def test_sizes_large_then_small_and_the_limit():
    """A large call leaves 2049 partial pairs behind; the one-CTA call after it must not see them."""
    import torch
    rng = np.random.default_rng(12)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    for n, dtype in [((1 << 24) + 3, np.float32), (5, np.float64), (8192, np.float64), (8193, np.float32), (1, np.float64)]:
        th = (rng.normal(size=n) * 2.0 + 0.3).astype(dtype)
        d_th = torch.from_numpy(th).cuda()
        _noalloc(d_th, out)
        z = np.exp(1j * th.astype(np.float64)).mean()
        got = out.cpu().numpy()
        assert abs(got[0] - abs(z)) <= TOL and abs(got[1] - np.angle(z)) <= TOL, (n, got, abs(z), np.angle(z))
    # beyond the static array: refused, nothing launched, out untouched
    before = out.cpu().numpy().copy()
    with pytest.raises(B.OscnetError) as e:
        B.net_order_parameter_noalloc(d_th.data_ptr(), B.NOALLOC_MAX_N + 1, B.F64, out.data_ptr(), None)
    assert e.value.code == ERR_SIZE and "maximum" in str(e.value)
    with pytest.raises(B.OscnetError):
        B.net_order_parameter_noalloc(d_th.data_ptr(), 0, B.F64, out.data_ptr(), None)
    with pytest.raises(B.OscnetError):
        B.net_order_parameter_noalloc(None, 8, B.F64, out.data_ptr(), None)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), before)


def test_no_device_memory_is_taken_and_the_call_can_be_captured():
    """After the first call on the device (which resolves the array's address and loads the kernel),
    further calls leave the free device memory unchanged; and the call is legal under stream capture,
    which cudaMalloc is not."""
    import torch
    rng = np.random.default_rng(13)
    n = 300000
    th = torch.from_numpy(rng.uniform(-np.pi, np.pi, size=n)).cuda()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    _noalloc(th, out)                                       # set-up call, outside capture
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(20):
        _noalloc(th, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0
    want = out.cpu().numpy().copy()

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        _noalloc(th, out, stream=side)
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), want)
    th.copy_(torch.from_numpy(rng.uniform(-1.0, 2.0, size=n)))          # new input, same graph
    g.replay()
    torch.cuda.synchronize()
    z = np.exp(1j * th.cpu().numpy()).mean()
    got = out.cpu().numpy()
    assert abs(got[0] - abs(z)) <= TOL and abs(got[1] - np.angle(z)) <= TOL
