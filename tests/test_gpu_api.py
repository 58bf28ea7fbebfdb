"""Edge cases and error behaviour of the C ABI on a GPU."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _B():
    from paper_2410_19075_b200 import binding
    return binding


def test_state_roundtrip_unaligned_n_and_device_pointers():
    import torch
    B = _B()
    n = 1001                                     # not a multiple of the internal stride
    net = B.Net(B.MODEL_HH, B.F32, n, dict(kind=B.TOPO_RING, radius=2), dict(
        gNa=120.0, gK=36.0, gL=0.3, ENa=50.0, EK=-77.0, EL=-54.4, C=1.0, g_syn=0.1, E_syn=0.0,
        theta_syn=0.0, k_syn=2.0))
    y = np.random.default_rng(0).normal(size=(4, n)).astype(np.float32)
    net.set_state(y)
    assert np.array_equal(net.get_state(), y)
    yd = torch.from_numpy(y * 2).cuda()
    net.set_state(yd)
    out = torch.empty_like(yd)
    net.get_state(out)
    torch.cuda.synchronize()
    assert torch.equal(out, yd)
    pinned = torch.empty((4, n), dtype=torch.float32).pin_memory()
    net.get_state(pinned)
    assert np.array_equal(pinned.numpy(), y * 2)


def test_degenerate_networks():
    B = _B()
    # one element, no neighbours: pure local dynamics; KS: phi(t) = phi0 + omega t
    net = B.Net(B.MODEL_KS, B.F64, 1, dict(kind=B.TOPO_RING, radius=0), dict(K=1.0, alpha=0.3, omega0=0.5))
    net.set_state(np.array([[0.25]]))
    net.integrate(100, 0.01)
    assert abs(net.get_state()[0, 0] - 0.75) < 1e-13
    # zero steps is a no-op; in-degree 0 graph
    net.integrate(0, 0.01)
    assert net.time() == (1.0, 100) or abs(net.time()[0] - 1.0) < 1e-12
    g = B.Net(B.MODEL_FHN, B.F64, 50, dict(kind=B.TOPO_RANDOM_INDEGREE, in_degree=0, seed=1),
              dict(eps=0.05, a=0.5, sigma=0.1, phi=0.2))
    y = np.stack([np.full(50, -0.5), np.full(50, -0.5 + 0.125 / 3)])
    g.set_state(y)
    assert np.abs(g.eval_rhs()).max() < 1e-14          # the FHN fixed point


def test_errors_are_reported_not_thrown():
    B = _B()
    with pytest.raises(B.OscnetError) as e:
        B.Net(B.MODEL_KS, B.F64, 10, dict(kind=B.TOPO_RING, radius=5), dict(K=1.0, alpha=0.0))
    assert e.value.code == -1
    with pytest.raises(B.OscnetError):
        B.Net(B.MODEL_KS, B.F64, 64, dict(kind=B.TOPO_LATTICE, extent=(4, 4, 4), radius=2), dict(K=1.0, alpha=0.0))
    net = B.Net(B.MODEL_KS, B.F64, 10, dict(kind=B.TOPO_RING, radius=2), dict(K=1.0, alpha=0.0))
    with pytest.raises(B.OscnetError):
        net.set_param_array(B.PARAM_IEXT, np.zeros(10))
    with pytest.raises(B.OscnetError):
        net.hh_steady_gates()
    with pytest.raises(B.OscnetError):
        net.integrate_observed(10, 0.1, 3)
    with pytest.raises(B.OscnetError):
        net.observable(B.OBS_STATS)
    # workspace too small / misaligned
    import torch
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.OscnetError) as e:
        B.net_create(net.desc, net.params, ws.data_ptr(), 1024, 0)
    assert e.value.code == -2
    launches, method = net.counters()
    assert launches >= 1 and method in (B.METHOD_DIRECT, B.METHOD_FAST)


@pytest.mark.gpu
def test_latency_probe_is_a_ring_diagnostic_and_leaves_the_state_alone():
    """net_probe_latency: four positive latencies for a ring net on the FAST path (the grid barrier
    is 0 for a single-CTA ring), state and results untouched; refused for other nets."""
    import numpy as np
    import harness as H
    from paper_2410_19075_b200 import binding as B, configs
    for cfg, kw, multi in (("1", {}, False), ("2", dict(n=8192), True)):
        w = configs.get(cfg, **kw)
        inp = H.make_inputs(w, seed=2)
        net = H.make_gpu(w, inp)
        before = net.get_state()
        L = net.probe_latency()
        assert (L["grid_barrier_us"] > 0) == multi
        assert 0 < L["l2_round_trip_us"] < 5 and 0 < L["block_scan_us"] < 5 and 0 < L["fp64_sincos_us"] < 5
        assert np.array_equal(net.get_state(), before)
        net.integrate(10, w.dt)
        ref = H.make_gpu(w, inp)
        ref.integrate(10, w.dt)
        assert np.array_equal(net.get_state(), ref.get_state())
        net.close(); ref.close()
    lat = H.make_gpu(configs.get("5", n1=16), H.make_inputs(configs.get("5", n1=16)))
    with pytest.raises(B.OscnetError) as ei:
        lat.probe_latency()
    assert ei.value.code == -5
    lat.close()


def test_probe_peaks_and_launch_config_leave_the_state_alone():
    """net_probe_peaks: positive, physically plausible numbers; the state,
    the time and the results of the net are untouched.  net_get_launch_config names the kernel family."""
    import harness as H
    from paper_2410_19075_b200 import configs
    w = configs.get("3b", n1=24)
    inp = H.make_inputs(w, seed=3)
    a, b = H.make_gpu(w, inp), H.make_gpu(w, inp)
    a.integrate(5, w.dt)
    b.integrate(5, w.dt)
    pk = a.probe_peaks()
    assert 5e3 < pk["ffma_ginstr_s"] < 6e4 and 2e3 < pk["dfma_ginstr_s"] < 3e4
    assert 0.3 < pk["dfma_ginstr_s"] / pk["ffma_ginstr_s"] < 0.7          # FP64 at half the FP32 rate
    assert 0.3 < pk["fadd2_ginstr_s"] / pk["ffma_ginstr_s"] < 0.7         # packed adds: half the instruction rate
    assert 500 < pk["mufu_ginstr_s"] < 1e4 and pk["l2_gather_gops"] > 10 and pk["smem_gbs"] > 1e3
    assert 500 < pk["sm_mhz"] < 3000
    assert a.time() == b.time()
    a.integrate(5, w.dt)
    b.integrate(5, w.dt)
    assert np.array_equal(a.get_state(), b.get_state())
    lc = a.launch_config()
    assert lc["family"] == a.kernel_family() == 6 and lc["tile_x"] > 0 and lc["threads"] % 32 == 0
