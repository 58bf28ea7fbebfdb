"""Pins of the oracle's second-workload models: FitzHugh-Nagumo exactly as
eq. (2) (x-only coupling, delay tau, noise D n(t), I_app, reading R17) and the
Hodgkin-Huxley element with the synaptic gating ODE of eq. (1) (reading R18).
Each check compares with a dense formula written out here, a closed form or a statistical law."""
import math

import numpy as np
import pytest

from oracle import oracle as ora


def _dense(rp, ci, n):
    L = np.zeros((n, n))
    for i in range(n):
        L[i, ci[rp[i]:rp[i + 1]]] = 1.0
    return L


# ------------------------------------------------------------------ eq. (2) without delay / noise
def _f2_dense(L, x, y, xd, eps, a, sigma, Iapp):
    om = L.sum(1)
    s = np.where(om > 0, sigma / np.maximum(om, 1), 0.0)
    cx = L @ xd - om * x
    return np.stack([(x - x ** 3 / 3 - y + s * cx + Iapp) / eps, x + a])


@pytest.mark.parametrize("topo", ["ring", "rand"])
def test_fhn2_rhs_is_eq2_with_an_explicit_matrix(topo):
    n = 14
    rp, ci = ora.topology_ring(n, 3) if topo == "ring" else ora.topology_random_indegree(n, 4, 5)
    net = ora.OracleNet.fhn2(n, rp, ci, 0.05, 0.5, 0.3, I_app=0.2)
    rng = np.random.default_rng(1)
    y = rng.uniform(-2, 2, size=(2, n))
    ref = _f2_dense(_dense(rp, ci, n), y[0], y[1], y[0], 0.05, 0.5, 0.3, 0.2)
    np.testing.assert_allclose(net.rhs(y), ref, rtol=1e-13, atol=1e-13)
    # no delay, no noise: the special integrator is plain RK4
    a, _ = net.fhn2_rk4(y, 30, 0.01, m=0)
    np.testing.assert_allclose(a, net.rk4(y, 30, 0.01), rtol=0, atol=1e-14)


def test_fhn2_delay_first_interval_is_an_ode_with_constant_history():
    """Method of steps: for 0 <= t <= tau the delayed values are the constant initial function, so
    the system is an ordinary ODE with a known forcing; a dense RK4 with a 5x finer step written
    here is the reference."""
    n, P, eps, a, sigma = 12, 2, 0.1, 0.5, 0.4
    rp, ci = ora.topology_ring(n, P)
    L = _dense(rp, ci, n)
    net = ora.OracleNet.fhn2(n, rp, ci, eps, a, sigma)
    rng = np.random.default_rng(2)
    y0 = rng.uniform(-1.5, 1.5, size=(2, n))
    m, dt = 200, 0.001                     # tau = 0.2
    got, _ = net.fhn2_rk4(y0, m, dt, m=m)  # integrate exactly to t = tau
    f = lambda z: _f2_dense(L, z[0], z[1], y0[0], eps, a, sigma, 0.0)
    z, h = y0.copy(), dt / 5
    for _ in range(5 * m):
        k1 = f(z); k2 = f(z + h / 2 * k1); k3 = f(z + h / 2 * k2); k4 = f(z + h * k3)
        z = z + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    assert np.abs(got - z).max() < 5e-9       # RK4 truncation at dt = 0.001 (4.9e-7 at dt = 0.005: fourth order)


def test_fhn2_delay_is_fourth_order_beyond_the_first_interval():
    """Past t = tau the delayed values come from the stored history and its Hermite midpoint; the
    scheme must keep RK4's order: halving dt (and doubling m) divides the error by ~16."""
    n = 10
    rp, ci = ora.topology_ring(n, 2)
    net = ora.OracleNet.fhn2(n, rp, ci, 0.2, 0.5, 0.5)
    th = np.linspace(0, 2 * np.pi, n, endpoint=False)
    y0 = np.stack([1.5 * np.cos(th), 1.5 * np.sin(th)])
    tau, T = 0.25, 1.5

    def run(k):                              # dt = tau / (5 k)
        m = 5 * k
        dt = tau / m
        return net.fhn2_rk4(y0, int(round(T / dt)), dt, m=m)[0]

    ref = run(32)
    e1, e2 = np.abs(run(1) - ref).max(), np.abs(run(2) - ref).max()
    assert 11 <= e1 / e2 <= 22, e1 / e2
    # and the delay matters: the undelayed run differs at order one
    assert np.abs(net.fhn2_rk4(y0, 300, 0.005, m=0)[0] - ref).max() > 1e-3


def test_fhn2_delay_continues_across_calls():
    n = 9
    rp, ci = ora.topology_ring(n, 2)
    net = ora.OracleNet.fhn2(n, rp, ci, 0.1, 0.5, 0.3)
    y0 = np.random.default_rng(3).uniform(-1, 1, size=(2, n))
    a, _ = net.fhn2_rk4(y0, 50, 0.01, m=7, D=0.1, seed=5)
    b, hist = net.fhn2_rk4(y0, 20, 0.01, m=7, D=0.1, seed=5)
    b, hist = net.fhn2_rk4(b, 30, 0.01, m=7, D=0.1, seed=5, hist=hist)
    assert np.array_equal(a, b)


# ------------------------------------------------------------------ noise
def test_gauss_stream_is_standard_normal_and_uncorrelated():
    xs = np.array([[ora.gauss(9, i, n) for n in range(200)] for i in range(200)])
    N = xs.size
    assert abs(xs.mean()) < 4 / math.sqrt(N)
    assert abs(xs.var() - 1) < 4 * math.sqrt(2 / N)
    assert abs((xs ** 4).mean() - 3) < 0.25                     # Gaussian kurtosis
    assert abs(np.mean(xs[:, 1:] * xs[:, :-1])) < 4 / math.sqrt(N)   # successive steps
    assert abs(np.mean(xs[1:] * xs[:-1])) < 4 / math.sqrt(N)         # neighbouring elements
    assert ora.gauss(9, 3, 4) != ora.gauss(10, 3, 4) and ora.gauss(9, 3, 4) == ora.gauss(9, 3, 4)
    # hand value of the rule: u1, u2 from the published splitmix64 finaliser (reading R8)
    M = (1 << 64) - 1
    def mix(z):
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9 & M
        z = (z ^ (z >> 27)) * 0x94D049BB133111EB & M
        return z ^ (z >> 31)
    G = 0x9E3779B97F4A7C15
    hi = mix((9 + G * 4) & M)
    a, b = mix((hi + G * 9) & M), mix((hi + G * 10) & M)
    u1, u2 = ((a >> 11) + 1) / 2 ** 53, (b >> 11) / 2 ** 53
    assert abs(ora.gauss(9, 3, 4) - math.sqrt(-2 * math.log(u1)) * math.cos(2 * math.pi * u2)) < 1e-14


def test_noise_enters_y_only_with_amplitude_D_sqrt_dt():
    n = 6
    rp, ci = ora.topology_ring(n, 1)
    net = ora.OracleNet.fhn2(n, rp, ci, 0.1, 0.5, 0.2)
    y0 = np.random.default_rng(4).uniform(-1, 1, size=(2, n))
    dt, D = 0.01, 0.3
    a, _ = net.fhn2_rk4(y0, 1, dt, D=0.0)
    b, _ = net.fhn2_rk4(y0, 1, dt, D=D, seed=11)
    assert np.array_equal(a[0], b[0])
    xi = np.array([ora.gauss(11, i, 0) for i in range(n)])
    np.testing.assert_allclose(b[1] - a[1], D * math.sqrt(dt) * xi, rtol=0, atol=1e-15)


# ------------------------------------------------------------------ HH with gating ODE
def test_hhs_rhs_dense_and_gating_fixed_point():
    n = 12
    rp, ci = ora.topology_random_indegree(n, 4, 3)
    L = _dense(rp, ci, n)
    rng = np.random.default_rng(6)
    Iext = 9 + 2 * rng.random(n)
    a_s, b_s = 2.0, 0.5
    net = ora.OracleNet.hhs(n, rp, ci, Iext, a_s=a_s, b_s=b_s)
    hh = ora.OracleNet.hh(n, rp, ci, Iext)
    V = rng.uniform(-80, 30, n)
    y = np.vstack([V, rng.random((3, n)), rng.random((1, n))])
    f = net.rhs(y)
    # the channel part equals the pinned HH right-hand side with the synapse switched off ...
    f0 = ora.OracleNet.hh(n, rp, ci, Iext, g_syn=0.0).rhs(y[:4])
    p = ora.HH_DEFAULT
    Isyn = p["g_syn"] / 4 * (p["E_syn"] - V) * (L @ y[4])
    np.testing.assert_allclose(f[0], f0[0] + Isyn / p["C"], rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(f[1:4], f0[1:4], rtol=0, atol=0)
    S = 1 / (1 + np.exp(-(V - p["theta_syn"]) / p["k_syn"]))
    np.testing.assert_allclose(f[4], a_s * S * (1 - y[4]) - b_s * y[4], rtol=1e-14, atol=1e-15)
    # ... and s at a_s S/(a_s S + b_s) is a fixed point of the gating equation
    y[4] = a_s * S / (a_s * S + b_s)
    assert np.abs(net.rhs(y)[4]).max() < 1e-15
    assert hh.nvar == 4 and net.nvar == 5


def test_hhs_gate_relaxes_with_its_time_constant():
    """One element, voltage clamped by a huge capacitance: s(t) relaxes exponentially to
    s_inf = a S/(a S + b) with rate a S + b (closed form of a linear ODE)."""
    rp = np.array([0, 0], dtype=np.int64)
    net = ora.OracleNet.hhs(1, rp, np.zeros(0, dtype=np.int32), np.zeros(1), a_s=2.0, b_s=0.5, C=1e12)
    V = 10.0
    m, h, g = ora.hh_steady_gates(np.array([V]))
    y0 = np.array([[V], m, h, g, [0.0]])
    S = 1 / (1 + math.exp(-(V - 0.0) / 2.0))
    rate, sinf = 2.0 * S + 0.5, 2.0 * S / (2.0 * S + 0.5)
    y = net.rk4(y0, 400, 0.005)
    assert abs(y[4, 0] - sinf * (1 - math.exp(-rate * 2.0))) < 1e-9
