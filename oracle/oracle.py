"""ctypes front end of the CPU oracle (TEST INFRASTRUCTURE, see oscnet_oracle.c).

All arithmetic of the method lives in ``oscnet_oracle.c``; this file only
marshals numpy arrays and restates the observable *statistics* procedure
(reading R9) as a plain Python loop over samples.
"""
import ctypes as C
import math
import os

import numpy as np

from .build import build

MODEL_KS, MODEL_FHN, MODEL_HH, MODEL_KSI, MODEL_FHN2, MODEL_HHS = 0, 1, 2, 3, 4, 5
NVAR = {MODEL_KS: 1, MODEL_FHN: 2, MODEL_HH: 4, MODEL_KSI: 2, MODEL_FHN2: 2, MODEL_HHS: 5}

_lib = None


class _OraNet(C.Structure):
    _fields_ = [("model", C.c_int32), ("pad_", C.c_int32), ("n", C.c_int64),
                ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p),
                ("elem_param", C.c_void_p), ("p", C.c_double * 16)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.ora_lattice_degree.restype = C.c_int64
        _lib.ora_lattice_degree.argtypes = [C.c_int32, C.c_int32, C.c_int32]
        _lib.ora_gauss.restype = C.c_double
        _lib.ora_gauss.argtypes = [C.c_uint64, C.c_int64, C.c_int64]
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def omp_threads() -> int:
    """Threads the OpenMP loops will use (OMP_NUM_THREADS or all cores)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


# ----------------------------------------------------------------- topology
def lattice_degree(ndim, P, include_self=False):
    return int(lib().ora_lattice_degree(ndim, P, int(include_self)))


def topology_ring(n, P, include_self=False, row_begin=0, row_count=None):
    row_count = n if row_count is None else row_count
    deg = 2 * P + (1 if include_self else 0)
    row_ptr = np.zeros(row_count + 1, dtype=np.int64)
    col_idx = np.zeros(max(1, row_count * deg), dtype=np.int32)
    rc = lib().ora_topology_ring(C.c_int64(n), C.c_int32(P), C.c_int32(int(include_self)),
                                 C.c_int64(row_begin), C.c_int64(row_count), _p(row_ptr),
                                 _p(col_idx))
    if rc != 0:
        raise ValueError("ora_topology_ring: invalid arguments")
    return row_ptr, col_idx[:row_count * deg]


def topology_lattice(extent, P, include_self=False, row_begin=0, row_count=None):
    ndim = len(extent)
    ext = np.array(list(extent) + [1] * (3 - ndim), dtype=np.int64)
    n = int(np.prod(ext))
    row_count = n if row_count is None else row_count
    deg = lattice_degree(ndim, P, include_self)
    row_ptr = np.zeros(row_count + 1, dtype=np.int64)
    col_idx = np.zeros(max(1, row_count * deg), dtype=np.int32)
    rc = lib().ora_topology_lattice(C.c_int32(ndim), _p(ext), C.c_int32(P),
                                    C.c_int32(int(include_self)), C.c_int64(row_begin),
                                    C.c_int64(row_count), _p(row_ptr), _p(col_idx))
    if rc != 0:
        raise ValueError("ora_topology_lattice: invalid arguments")
    return row_ptr, col_idx[:row_count * deg]


def topology_random_indegree(n, k, seed, row_begin=0, row_count=None):
    row_count = n if row_count is None else row_count
    row_ptr = np.zeros(row_count + 1, dtype=np.int64)
    col_idx = np.zeros(max(1, row_count * k), dtype=np.int32)
    rc = lib().ora_topology_random_indegree(C.c_int64(n), C.c_int32(k), C.c_uint64(seed),
                                            C.c_int64(row_begin), C.c_int64(row_count),
                                            _p(row_ptr), _p(col_idx))
    if rc != 0:
        raise ValueError("ora_topology_random_indegree: invalid arguments")
    return row_ptr, col_idx[:row_count * k]


# ------------------------------------------------------------------ network
def fhn_rotation(phi):
    """(b_uu, b_uv, b_vu, b_vv) = (cos phi, sin phi, -sin phi, cos phi)."""
    return (math.cos(phi), math.sin(phi), -math.sin(phi), math.cos(phi))


HH_DEFAULT = dict(gNa=120.0, gK=36.0, gL=0.3, ENa=50.0, EK=-77.0, EL=-54.4, C=1.0,
                  g_syn=0.1, E_syn=0.0, theta_syn=0.0, k_syn=2.0)
HH_PHASE_MAP = (-20.0, 0.55, 100.0)  # (V_c, n_c, V_s), reading R9


class OracleNet:
    """A network = model + parameters + canonical CSR topology (full rows)."""

    def __init__(self, model, n, row_ptr, col_idx, params, elem_param=None):
        self.model, self.n = model, int(n)
        self.row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
        self.col_idx = np.ascontiguousarray(col_idx, dtype=np.int32)
        assert self.row_ptr.shape[0] == self.n + 1
        if elem_param is None:
            elem_param = np.zeros(self.n)
        self.elem_param = np.ascontiguousarray(np.broadcast_to(
            np.asarray(elem_param, dtype=np.float64), (self.n,)))
        self.params = [float(x) for x in params]
        self._s = _OraNet()
        self._s.model, self._s.n = model, self.n
        self._s.row_ptr, self._s.col_idx = _p(self.row_ptr).value, _p(self.col_idx).value
        self._s.elem_param = _p(self.elem_param).value
        for q, v in enumerate(self.params):
            self._s.p[q] = v

    # constructors in the notation of the configs
    @classmethod
    def ks(cls, n, row_ptr, col_idx, K, alpha, omega):
        return cls(MODEL_KS, n, row_ptr, col_idx, [K, alpha], omega)

    @classmethod
    def ksi(cls, n, row_ptr, col_idx, K, alpha, m, eps, omega=0.0):
        """Kuramoto-Sakaguchi with inertia, eq. (3) PAPER.md:79 in full; state [phi | phi']
        (GPU: NET_MODEL_KSI).  Its phase variable is phi, so the observables
        treat it as a phase model like KS (reading R9)."""
        return cls(MODEL_KSI, n, row_ptr, col_idx, [K, alpha, m, eps], omega)

    @classmethod
    def fhn(cls, n, row_ptr, col_idx, eps, a, sigma, phi):
        return cls(MODEL_FHN, n, row_ptr, col_idx, [eps, a, sigma, *fhn_rotation(phi)])

    @classmethod
    def hh(cls, n, row_ptr, col_idx, I_ext, **kw):
        p = dict(HH_DEFAULT)
        p.update(kw)
        return cls(MODEL_HH, n, row_ptr, col_idx,
                   [p[k] for k in ("gNa", "gK", "gL", "ENa", "EK", "EL", "C", "g_syn",
                                   "E_syn", "theta_syn", "k_syn")], I_ext)

    @classmethod
    def fhn2(cls, n, row_ptr, col_idx, eps, a, sigma, I_app=0.0):
        """FitzHugh-Nagumo exactly as eq. (2) PAPER.md:70-75 (x-only coupling, I_app); the delay and
        the noise belong to the integrator (fhn2_rk4).  SURVEY.md 8(f).4, reading R17."""
        return cls(MODEL_FHN2, n, row_ptr, col_idx, [eps, a, sigma, I_app])

    @classmethod
    def hhs(cls, n, row_ptr, col_idx, I_ext, a_s=2.0, b_s=0.5, **kw):
        """Hodgkin-Huxley with the synaptic gating ODE of eq. (1) (reading R18); state [V|m|h|n|s]."""
        p = dict(HH_DEFAULT)
        p.update(kw)
        return cls(MODEL_HHS, n, row_ptr, col_idx,
                   [p[k] for k in ("gNa", "gK", "gL", "ENa", "EK", "EL", "C", "g_syn",
                                   "E_syn", "theta_syn", "k_syn")] + [a_s, b_s], I_ext)

    def fhn2_rk4(self, y, n_steps, dt, m=0, D=0.0, seed=0, hist=None):
        """RK4 steps of eq. (2) with delay tau = m dt and noise amplitude D (ora_fhn2_rk4).
        hist: None to start from the constant initial function, or the dict a previous call returned
        to continue.  Returns (state, hist)."""
        y = np.array(y, dtype=np.float64).reshape(2 * self.n)
        if hist is None:
            hist = dict(step=0, x=np.zeros((m + 2) * self.n), d=np.zeros((m + 2) * self.n))
        rc = lib().ora_fhn2_rk4(C.byref(self._s), _p(y), C.c_int64(n_steps), C.c_double(dt),
                                C.c_int64(m), C.c_double(D), C.c_uint64(seed),
                                C.c_int64(hist["step"]), _p(hist["x"]), _p(hist["d"]))
        assert rc == 0
        hist = dict(hist, step=hist["step"] + n_steps)
        return y.reshape(2, self.n), hist

    @property
    def nvar(self):
        return NVAR[self.model]

    def rhs(self, y):
        y = np.ascontiguousarray(y, dtype=np.float64).reshape(self.nvar * self.n)
        f = np.empty_like(y)
        rc = lib().ora_rhs(C.byref(self._s), _p(y), _p(f))
        assert rc == 0
        return f.reshape(self.nvar, self.n)

    def rk4(self, y, n_steps, dt, fast=False):
        """Returns the state after n_steps classical RK4 steps (y is not modified).
        fast=True: the accelerated restatement of the neighbour sum (ora_rk4_fast), for the long
        statistics runs of tests/golden/make_stats_cache.py only."""
        y = np.array(y, dtype=np.float64).reshape(self.nvar * self.n)
        if fast:
            rc = lib().ora_rk4_fast(C.byref(self._s), _p(y), C.c_int64(n_steps), C.c_double(dt),
                                    C.c_int64(self.ring_P))
        else:
            rc = lib().ora_rk4(C.byref(self._s), _p(y), C.c_int64(n_steps), C.c_double(dt))
        assert rc == 0
        return y.reshape(self.nvar, self.n)

    ring_P = 0      # > 0: the rows are the ring windows of that radius (lets ora_rhs_fast use prefix sums)

    def rhs_fast(self, y):
        """ora_rhs_fast: factorised sine / precomputed S(V) / prefix sums (last
        paragraph).  Only for the long statistics runs, after it was shown equal to rhs()."""
        y = np.ascontiguousarray(y, dtype=np.float64).reshape(self.nvar * self.n)
        f = np.empty_like(y)
        rc = lib().ora_rhs_fast(C.byref(self._s), _p(y), _p(f), C.c_int64(self.ring_P))
        assert rc == 0
        return f.reshape(self.nvar, self.n)

    # ------------------------------------------------------------ Dormand-Prince 5(4)
    def dp5_step(self, y, h):
        """One uncontrolled DOPRI5 step: (5th-order solution, embedded error vector)."""
        y = np.ascontiguousarray(y, dtype=np.float64).reshape(self.nvar * self.n)
        y5, e = np.empty_like(y), np.empty_like(y)
        rc = lib().ora_dp5_step(C.byref(self._s), _p(y), C.c_double(h), _p(y5), _p(e))
        assert rc == 0
        return y5.reshape(self.nvar, self.n), e.reshape(self.nvar, self.n)

    def dp5(self, y, t0, t_end, rtol, atol, h0, max_attempts=1000000, log=False):
        """Adaptive DOPRI5 from t0 to t_end (reading R15).  Returns (state, info):
        info = dict(accepted, rejected, h_last, h_next, t[, h_log: attempted step sizes, negative
        when rejected])."""
        y = np.array(y, dtype=np.float64).reshape(self.nvar * self.n)
        out = np.zeros(5)
        cap = 1 << 16
        hl = np.zeros(cap if log else 1)
        rc = lib().ora_dp5(C.byref(self._s), _p(y), C.c_double(t0), C.c_double(t_end),
                           C.c_double(rtol), C.c_double(atol), C.c_double(h0),
                           C.c_int64(max_attempts), _p(out), _p(hl) if log else None,
                           C.c_int64(cap if log else 0))
        assert rc in (0, 1)
        info = dict(accepted=int(out[0]), rejected=int(out[1]), h_last=out[2], h_next=out[3],
                    t=out[4], exhausted=bool(rc))
        if log:
            info["h_log"] = hl[:min(cap, info["accepted"] + info["rejected"])].copy()
        return y.reshape(self.nvar, self.n), info

    def dp5_dense(self, y, t0, t_out, rtol, atol, h0, max_attempts=1000000):
        """Adaptive DOPRI5 with dense output (ora_dp5_dense): the states at the ascending times t_out
        (the last one is also the end of the integration).  Returns (out[n_out][nvar][n], info)."""
        y = np.array(y, dtype=np.float64).reshape(self.nvar * self.n)
        t_out = np.ascontiguousarray(t_out, dtype=np.float64)
        out = np.empty((len(t_out), self.nvar * self.n))
        st = np.zeros(5)
        rc = lib().ora_dp5_dense(C.byref(self._s), _p(y), C.c_double(t0), C.c_int64(len(t_out)), _p(t_out),
                                 _p(out), C.c_double(rtol), C.c_double(atol), C.c_double(h0),
                                 C.c_int64(max_attempts), _p(st))
        assert rc in (0, 1)
        info = dict(accepted=int(st[0]), rejected=int(st[1]), h_last=st[2], h_next=st[3], t=st[4])
        return out.reshape(len(t_out), self.nvar, self.n), info

    # ------------------------------------------------------------ observables
    def phase(self, y, phase_map=HH_PHASE_MAP):
        y = np.ascontiguousarray(y, dtype=np.float64).reshape(self.nvar * self.n)
        pm = np.array(phase_map, dtype=np.float64)
        th = np.empty(self.n)
        lib().ora_phase(C.c_int32(self.model), C.c_int64(self.n), _p(y), _p(pm), _p(th))
        return th

    def global_order(self, theta):
        theta = np.ascontiguousarray(theta, dtype=np.float64)
        R, Psi = C.c_double(), C.c_double()
        lib().ora_global_order(C.c_int64(self.n), _p(theta), C.byref(R), C.byref(Psi))
        return R.value, Psi.value

    def local_order(self, theta):
        theta = np.ascontiguousarray(theta, dtype=np.float64)
        out = np.empty(self.n)
        lib().ora_local_order(C.c_int64(self.n), _p(self.row_ptr), _p(self.col_idx),
                              _p(theta), _p(out))
        return out

    def run_statistics(self, y0, n_steps, dt, obs_every, phase_map=HH_PHASE_MAP, fast=False):
        """Long-run statistics, reading R9.

        Samples are taken after steps obs_every, 2*obs_every, ..., n_steps.  The
        window is the samples with step >= n_steps/2; t_a / t_b are its first /
        last sample times.  Returns a dict with mean and (population) std of the
        global R over the window, the mean over i of the local R_i at the last
        sample, and mean and std over i of the mean phase velocity on
        [t_a, t_b]: KS and KS with inertia (phase models: the state variable phi is the unwrapped
        phase, reading R9) (phi(t_b)-phi(t_a))/(t_b-t_a); FHN/HH the sum of the
        increments of theta between consecutive samples, each wrapped to
        (-pi, pi], divided by (t_b-t_a).
        """
        assert n_steps % obs_every == 0
        y = np.array(y0, dtype=np.float64).reshape(self.nvar, self.n)
        Rs, wind, theta_prev, y_a, s_a = [], np.zeros(self.n), None, None, None
        theta = None
        for s in range(obs_every, n_steps + 1, obs_every):
            y = self.rk4(y, obs_every, dt, fast=fast)
            if 2 * s < n_steps:
                continue
            theta = self.phase(y, phase_map)
            Rs.append(self.global_order(theta)[0])
            if theta_prev is None:
                y_a, s_a = y.copy(), s
            else:
                d = theta - theta_prev
                wind += d - 2.0 * np.pi * np.round(d / (2.0 * np.pi))
            theta_prev = theta
        T = (n_steps - s_a) * dt
        if self.model in (MODEL_KS, MODEL_KSI):
            vel = (y[0] - y_a[0]) / T if T > 0 else np.zeros(self.n)
        else:
            vel = wind / T if T > 0 else np.zeros(self.n)
        Rs = np.array(Rs)
        return dict(R_mean=float(Rs.mean()), R_std=float(Rs.std()),
                    Rloc_mean=float(self.local_order(theta).mean()),
                    vel_mean=float(vel.mean()), vel_std=float(vel.std()),
                    n_samples=int(Rs.size), vel=vel, y=y)


def gauss(seed, i, n):
    """Standard normal deviate (i, n) of the counter-based stream `seed` (ora_gauss)."""
    return float(lib().ora_gauss(C.c_uint64(seed), C.c_int64(i), C.c_int64(n)))


def hh_steady_gates(V):
    V = np.ascontiguousarray(V, dtype=np.float64)
    m, h, g = np.empty_like(V), np.empty_like(V), np.empty_like(V)
    lib().ora_hh_steady_gates(C.c_int64(V.size), _p(V), _p(m), _p(h), _p(g))
    return m, h, g
