"""Thin ctypes binding of liboscnet.so (include/oscnet.h).

Argument marshalling only: every step of the hot path runs in the CUDA library.
PyTorch supplies device memory (the workspace), streams and pinned host memory.
The module-level ``net_*`` functions mirror the C ABI one to one; ``Net`` is a
small convenience wrapper that owns the workspace tensor.  There is no CPU
fallback: a missing library or a missing GPU raises.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liboscnet.so")

NET_OK = 0
MODEL_KS, MODEL_FHN, MODEL_HH, MODEL_KSI, MODEL_FHN2, MODEL_HHS = 0, 1, 2, 3, 4, 5
TOPO_RING, TOPO_LATTICE, TOPO_CSR, TOPO_RANDOM_INDEGREE, TOPO_COMPRESSED = 0, 1, 2, 3, 4
F32, F64 = 0, 1
METHOD_AUTO, METHOD_DIRECT, METHOD_FAST = 0, 1, 2
PARAM_OMEGA, PARAM_IEXT = 0, 1
OBS_PHASE, OBS_GLOBAL_ORDER, OBS_LOCAL_ORDER, OBS_MEAN_PHASE_VELOCITY, OBS_STATS, OBS_REPLICA_ORDER = 0, 1, 2, 3, 4, 5
NVAR = {MODEL_KS: 1, MODEL_FHN: 2, MODEL_HH: 4, MODEL_KSI: 2, MODEL_FHN2: 2, MODEL_HHS: 5}

ABI_SYMBOLS = [
    "net_workspace_bytes", "net_create", "net_destroy", "net_set_state", "net_get_state",
    "net_set_param_array", "net_hh_steady_gates", "net_integrate", "net_integrate_observed",
    "net_eval_rhs", "net_observables", "net_get_topology", "net_get_degree", "net_get_time",
    "net_set_time", "net_get_counters", "net_get_kernel_family", "net_synchronize", "net_last_error", "net_version",
    "net_probe_latency", "net_probe_peaks", "net_get_launch_config",
    "net_adaptive_workspace_bytes", "net_integrate_adaptive",
    "net_compress_csr", "net_compressed_free", "net_integrate_adaptive_dense",
    "net_order_parameter_noalloc",
]


class KSParams(C.Structure):
    _fields_ = [("K", C.c_double), ("alpha", C.c_double), ("omega0", C.c_double)]


class KSIParams(C.Structure):
    _fields_ = [("K", C.c_double), ("alpha", C.c_double), ("m", C.c_double), ("eps", C.c_double),
                ("omega0", C.c_double)]


class FHNParams(C.Structure):
    _fields_ = [("eps", C.c_double), ("a", C.c_double), ("sigma", C.c_double), ("phi", C.c_double)]


class HHParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("gNa", "gK", "gL", "ENa", "EK", "EL", "C", "g_syn", "E_syn", "theta_syn", "k_syn",
                 "I_ext0", "V_c", "n_c", "V_s")]


class FHN2Params(C.Structure):
    _fields_ = [("eps", C.c_double), ("a", C.c_double), ("sigma", C.c_double), ("I_app", C.c_double),
                ("D", C.c_double), ("seed", C.c_uint64)]


class HHSParams(C.Structure):
    _fields_ = [("hh", HHParams), ("a_s", C.c_double), ("b_s", C.c_double)]


HH_PHASE_MAP = dict(V_c=-20.0, n_c=0.55, V_s=100.0)


class Topology(C.Structure):
    _fields_ = [("kind", C.c_int32), ("ndim", C.c_int32), ("extent", C.c_int64 * 3),
                ("radius", C.c_int32), ("include_self", C.c_int32), ("row_ptr", C.c_void_p),
                ("col_idx", C.c_void_p), ("nnz", C.c_int64), ("ptrs_are_device", C.c_int32),
                ("in_degree", C.c_int32), ("seed", C.c_uint64), ("compressed", C.c_void_p)]


class Compressed(C.Structure):
    """net_compressed: V, D, C of Alg. 2 (host arrays)."""
    _fields_ = [("n", C.c_int64), ("v_len", C.c_int64), ("v_pos", C.POINTER(C.c_int32)),
                ("k", C.c_int64), ("d_ptr", C.POINTER(C.c_int64)), ("d_pos", C.POINTER(C.c_int32)),
                ("c", C.POINTER(C.c_int32))]


class Desc(C.Structure):
    _fields_ = [("model", C.c_int32), ("dtype", C.c_int32), ("n", C.c_int64), ("batch", C.c_int32),
                ("method", C.c_int32), ("topo", Topology), ("delay_steps", C.c_int32),
                ("reserved_", C.c_int32)]


class OscnetError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("oscnet error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    """Loads liboscnet.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise OSError("liboscnet.so is missing: run `python -m paper_2410_19075_b200.build` "
                          "(the product path has no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.net_last_error.restype = C.c_char_p
        L.net_last_error.argtypes = [C.c_void_p]
        L.net_version.restype = C.c_char_p
        L.net_workspace_bytes.argtypes = [C.POINTER(Desc), C.POINTER(C.c_size_t)]
        L.net_create.argtypes = [C.POINTER(Desc), C.c_void_p, C.c_size_t, C.c_void_p, C.c_size_t,
                                 C.c_void_p, C.POINTER(C.c_void_p)]
        L.net_destroy.argtypes = [C.c_void_p]
        L.net_set_state.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
        L.net_get_state.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
        L.net_set_param_array.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32]
        L.net_hh_steady_gates.argtypes = [C.c_void_p]
        L.net_integrate.argtypes = [C.c_void_p, C.c_int64, C.c_double]
        L.net_integrate_observed.argtypes = [C.c_void_p, C.c_int64, C.c_double, C.c_int64]
        L.net_eval_rhs.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
        L.net_observables.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32]
        L.net_get_topology.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p,
                                       C.c_int32]
        L.net_get_degree.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32)]
        L.net_get_time.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.net_set_time.argtypes = [C.c_void_p, C.c_double, C.c_int64]
        L.net_get_counters.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32)]
        L.net_synchronize.argtypes = [C.c_void_p]
        L.net_probe_latency.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.net_probe_peaks.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.net_get_launch_config.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.net_adaptive_workspace_bytes.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        L.net_integrate_adaptive.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double,
                                             C.c_int64, C.c_void_p, C.c_size_t, C.POINTER(C.c_double)]
        L.net_integrate_adaptive_dense.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                                   C.c_double, C.c_int64, C.c_void_p, C.c_size_t, C.POINTER(C.c_double)]
        L.net_compress_csr.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.POINTER(C.POINTER(Compressed))]
        L.net_compressed_free.argtypes = [C.POINTER(Compressed)]
        L.net_order_parameter_noalloc.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p]
        for name in ABI_SYMBOLS:
            if name not in ("net_last_error", "net_version"):
                getattr(L, name).restype = C.c_int32
        _lib = L
    return _lib


def _check(rc, handle=None):
    if rc != NET_OK:
        msg = lib().net_last_error(handle)
        raise OscnetError(rc, msg.decode() if msg else "")


# ---------------------------------------------------------------- C-ABI mirrors
def net_version():
    return lib().net_version().decode()


def net_workspace_bytes(desc):
    out = C.c_size_t()
    _check(lib().net_workspace_bytes(C.byref(desc), C.byref(out)))
    return out.value


def net_create(desc, params, workspace_ptr, workspace_bytes, stream_ptr):
    h = C.c_void_p()
    _check(lib().net_create(C.byref(desc), C.byref(params), C.sizeof(params), workspace_ptr,
                            workspace_bytes, stream_ptr, C.byref(h)))
    return h


def net_destroy(h):
    _check(lib().net_destroy(h))


def net_set_state(h, ptr, is_device):
    _check(lib().net_set_state(h, ptr, int(is_device)), h)


def net_get_state(h, ptr, is_device):
    _check(lib().net_get_state(h, ptr, int(is_device)), h)


def net_set_param_array(h, which, ptr, is_device):
    _check(lib().net_set_param_array(h, which, ptr, int(is_device)), h)


def net_hh_steady_gates(h):
    _check(lib().net_hh_steady_gates(h), h)


def net_integrate(h, n_steps, dt):
    _check(lib().net_integrate(h, n_steps, dt), h)


def net_integrate_observed(h, n_steps, dt, obs_every):
    _check(lib().net_integrate_observed(h, n_steps, dt, obs_every), h)


class CompressedMatrix:
    """Owner of a net_compressed returned by net_compress_csr (freed with the object)."""

    def __init__(self, ptr):
        self.ptr = ptr

    @property
    def s(self):
        return self.ptr.contents

    def arrays(self):
        """(V, d_ptr, d_pos, C) as numpy copies."""
        s = self.s
        dptr = np.ctypeslib.as_array(s.d_ptr, shape=(s.k + 1,)).copy()
        return (np.ctypeslib.as_array(s.v_pos, shape=(max(s.v_len, 1),))[:s.v_len].copy(), dptr,
                np.ctypeslib.as_array(s.d_pos, shape=(max(int(dptr[-1]), 1),))[:int(dptr[-1])].copy(),
                np.ctypeslib.as_array(s.c, shape=(s.n,)).copy())

    def __del__(self):
        try:
            if self.ptr:
                lib().net_compressed_free(self.ptr)
                self.ptr = None
        except Exception:
            pass


def net_compress_csr(row_ptr, col_idx):
    """COMPRESS of Alg. 2 on host CSR arrays (int64 row_ptr, int32 col_idx)."""
    rp = np.ascontiguousarray(row_ptr, dtype=np.int64)
    ci = np.ascontiguousarray(col_idx, dtype=np.int32)
    out = C.POINTER(Compressed)()
    _check(lib().net_compress_csr(len(rp) - 1, rp.ctypes.data, ci.ctypes.data, C.byref(out)))
    return CompressedMatrix(out)


def net_adaptive_workspace_bytes(h):
    out = C.c_size_t()
    _check(lib().net_adaptive_workspace_bytes(h, C.byref(out)), h)
    return out.value


def net_integrate_adaptive(h, t_end, rtol, atol, h0, max_attempts, work_ptr, work_bytes):
    out = (C.c_double * 5)()
    rc = lib().net_integrate_adaptive(h, t_end, rtol, atol, h0, max_attempts, work_ptr, work_bytes, out)
    info = dict(accepted=int(out[0]), rejected=int(out[1]), h_last=out[2], h_next=out[3], t=out[4])
    _check(rc, h)
    return info


def net_eval_rhs(h, ptr, is_device):
    _check(lib().net_eval_rhs(h, ptr, int(is_device)), h)


def net_observables(h, what, ptr, is_device):
    _check(lib().net_observables(h, what, ptr, int(is_device)), h)


def net_get_topology(h, row_begin, row_count, row_ptr_ptr, col_idx_ptr, is_device):
    _check(lib().net_get_topology(h, row_begin, row_count, row_ptr_ptr, col_idx_ptr,
                                  int(is_device)), h)


def net_get_degree(h):
    nnz, deg = C.c_int64(), C.c_int32()
    _check(lib().net_get_degree(h, C.byref(nnz), C.byref(deg)), h)
    return nnz.value, deg.value


def net_get_time(h):
    t, s = C.c_double(), C.c_int64()
    _check(lib().net_get_time(h, C.byref(t), C.byref(s)), h)
    return t.value, s.value


def net_set_time(h, t, step):
    _check(lib().net_set_time(h, t, step), h)


def net_get_counters(h):
    k, m = C.c_int64(), C.c_int32()
    _check(lib().net_get_counters(h, C.byref(k), C.byref(m)), h)
    return k.value, m.value


def net_get_kernel_family(h):
    f = C.c_int32()
    _check(lib().net_get_kernel_family(h, C.byref(f)), h)
    return f.value


def net_probe_latency(h):
    out = (C.c_double * 4)()
    _check(lib().net_probe_latency(h, out), h)
    return dict(grid_barrier_us=out[0], l2_round_trip_us=out[1], block_scan_us=out[2], fp64_sincos_us=out[3])


def net_get_launch_config(h):
    out = (C.c_int32 * 8)()
    _check(lib().net_get_launch_config(h, out), h)
    return dict(family=out[0], tile_x=out[1], tile_y=out[2], lz=out[3], depth=out[4], grid=out[5],
                threads=out[6], smem_bytes=out[7])


def net_probe_peaks(h):
    out = (C.c_double * 8)()
    _check(lib().net_probe_peaks(h, out), h)
    return dict(ffma_ginstr_s=out[0], fadd2_ginstr_s=out[1], dfma_ginstr_s=out[2], mufu_ginstr_s=out[3],
                smem_gbs=out[4], l2_gather_gops=out[5], gather_array_bytes=out[6], sm_mhz=out[7])


def net_synchronize(h):
    _check(lib().net_synchronize(h), h)


NOALLOC_MAX_N = 1 << 27


def net_order_parameter_noalloc(d_theta_ptr, n, dtype, d_out2_ptr, stream_ptr=None):
    """{R, Psi} of n device phases into a device double[2]; allocates nothing (static device scratch,
    n <= NOALLOC_MAX_N; calls that overlap on the GPU race).  Pointers are device addresses (ints)."""
    _check(lib().net_order_parameter_noalloc(d_theta_ptr, n, dtype, d_out2_ptr, stream_ptr))


# ------------------------------------------------------------------ convenience
def make_params(model, p):
    if model == MODEL_KS:
        return KSParams(p["K"], p["alpha"], p.get("omega0", 0.0))
    if model == MODEL_KSI:
        return KSIParams(p["K"], p["alpha"], p["m"], p["eps"], p.get("omega0", 0.0))
    if model == MODEL_FHN:
        return FHNParams(p["eps"], p["a"], p["sigma"], p["phi"])
    if model == MODEL_FHN2:
        return FHN2Params(p["eps"], p["a"], p["sigma"], p.get("I_app", 0.0), p.get("D", 0.0), int(p.get("seed", 0)))
    q = dict(HH_PHASE_MAP, I_ext0=0.0)
    q.update(p)
    hh = HHParams(*[q[k] for k, _ in HHParams._fields_])
    if model == MODEL_HHS:
        return HHSParams(hh, p.get("a_s", 2.0), p.get("b_s", 0.5))
    return hh


def _np_dtype(dtype):
    return np.float32 if dtype == F32 else np.float64


class Net:
    """Owns a workspace tensor and a handle; methods mirror the C ABI."""

    def __init__(self, model, dtype, n, topo, params, method=METHOD_AUTO, device="cuda:0",
                 stream=None, batch=1, delay_steps=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("oscnet needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.device = torch.device(device)
        # self.n: elements of all replicas together (arrays are [nvar][batch][n] = [nvar][self.n])
        self.model, self.dtype, self.n, self.batch = model, dtype, int(n) * int(batch), int(batch)
        self.nvar = NVAR[model]
        self.np_dtype = _np_dtype(dtype)
        self.torch_dtype = torch.float32 if dtype == F32 else torch.float64
        d = Desc()
        d.model, d.dtype, d.n, d.batch, d.method = model, dtype, int(n), int(batch), method
        d.delay_steps = int(delay_steps)
        t = d.topo
        t.kind = topo["kind"]
        ext = list(topo.get("extent", ())) + [1, 1, 1]
        t.ndim = len(topo.get("extent", ())) or 1
        for q in range(3):
            t.extent[q] = ext[q]
        t.radius = topo.get("radius", 0)
        t.include_self = int(topo.get("include_self", False))
        t.in_degree = topo.get("in_degree", 0)
        t.seed = topo.get("seed", 0)
        self._keep = []
        if t.kind == TOPO_CSR:
            rp, ci = topo["row_ptr"], topo["col_idx"]
            if isinstance(rp, np.ndarray):
                rp = np.ascontiguousarray(rp, dtype=np.int64)
                ci = np.ascontiguousarray(ci, dtype=np.int32)
                t.row_ptr, t.col_idx = rp.ctypes.data, ci.ctypes.data
                t.nnz, t.ptrs_are_device = int(rp[-1]), 0
            else:
                t.row_ptr, t.col_idx = rp.data_ptr(), ci.data_ptr()
                t.nnz, t.ptrs_are_device = int(ci.numel()), 1
            self._keep += [rp, ci]
        if t.kind == TOPO_COMPRESSED:
            cm = topo["compressed"]
            t.compressed = C.cast(cm.ptr, C.c_void_p)
            self._keep.append(cm)
        self.desc = d
        self.params = make_params(model, params)
        with torch.cuda.device(self.device):
            # a stream of its own: the legacy default stream cannot be captured into a CUDA graph
            self.stream = stream or torch.cuda.Stream(device=self.device)
            self.stream.wait_stream(torch.cuda.current_stream())
            self.workspace_bytes = net_workspace_bytes(d)
            self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8,
                                         device=self.device)
            self.workspace.record_stream(self.stream)
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            self.h = net_create(d, self.params, base, self.workspace_bytes,
                                self.stream.cuda_stream)

    @classmethod
    def from_workload(cls, w, method=METHOD_AUTO, device="cuda:0", stream=None):
        from . import configs
        dtype = F32 if w.dtype == "f32" else F64
        if w.topo == configs.RING:
            topo = dict(kind=TOPO_RING, radius=w.radius)
        elif w.topo == configs.LATTICE:
            topo = dict(kind=TOPO_LATTICE, extent=w.extent, radius=w.radius)
        else:
            topo = dict(kind=TOPO_RANDOM_INDEGREE, in_degree=w.in_degree, seed=w.topo_seed)
        return cls(w.model, dtype, w.n, topo, w.params, method=method, device=device,
                   stream=stream, batch=getattr(w, "batch", 1),
                   delay_steps=w.extra.get("delay_steps", 0))

    def close(self):
        if getattr(self, "h", None):
            net_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # state --------------------------------------------------------------------
    def _ptr(self, x):
        """(pointer, is_device) of a numpy array or torch tensor (must be contiguous)."""
        if isinstance(x, np.ndarray):
            assert x.flags["C_CONTIGUOUS"]
            return x.ctypes.data, False
        assert x.is_contiguous()
        if x.is_cuda:       # order the net's stream after the producer of the tensor
            self.stream.wait_stream(self.torch.cuda.current_stream())
            x.record_stream(self.stream)
        return x.data_ptr(), x.is_cuda

    def _publish(self, x):
        """Makes torch's current stream wait for a device-side result written on the net's stream."""
        if not isinstance(x, np.ndarray) and x.is_cuda:
            self.torch.cuda.current_stream().wait_stream(self.stream)

    def set_state(self, y):
        if isinstance(y, np.ndarray):
            y = np.ascontiguousarray(y, dtype=self.np_dtype).reshape(self.nvar, self.n)
        else:
            assert y.dtype == self.torch_dtype and y.numel() == self.nvar * self.n
        net_set_state(self.h, *self._ptr(y))

    def get_state(self, out=None):
        if out is None:
            out = np.empty((self.nvar, self.n), dtype=self.np_dtype)
        net_get_state(self.h, *self._ptr(out))
        self._publish(out)
        return out

    def set_param_array(self, which, x):
        if isinstance(x, np.ndarray):
            x = np.ascontiguousarray(x, dtype=self.np_dtype)
        net_set_param_array(self.h, which, *self._ptr(x))

    def hh_steady_gates(self):
        net_hh_steady_gates(self.h)

    # dynamics -----------------------------------------------------------------
    def integrate(self, n_steps, dt):
        net_integrate(self.h, int(n_steps), float(dt))

    def integrate_adaptive(self, t_end, rtol, atol, h0, max_attempts=1000000):
        """Dormand-Prince 5(4) from the net's time to t_end; returns the step statistics."""
        torch = self.torch
        need = net_adaptive_workspace_bytes(self.h)
        if getattr(self, "_adaptive_work", None) is None or self._adaptive_work.numel() < need + 256:
            with torch.cuda.device(self.device):
                self._adaptive_work = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
                self._adaptive_work.record_stream(self.stream)
            self.stream.wait_stream(torch.cuda.current_stream())
        base = (self._adaptive_work.data_ptr() + 255) // 256 * 256
        return net_integrate_adaptive(self.h, float(t_end), float(rtol), float(atol), float(h0),
                                      int(max_attempts), base, need)

    def integrate_adaptive_dense(self, t_out, rtol, atol, h0, max_attempts=1000000):
        """Dormand-Prince 5(4) to t_out[-1] with dense output at the ascending times t_out; returns
        (states [n_out][nvar][n] as a numpy array, step statistics)."""
        torch = self.torch
        t_out = np.ascontiguousarray(t_out, dtype=np.float64)
        need = net_adaptive_workspace_bytes(self.h) + (8 * len(t_out) + 255) // 256 * 256
        with torch.cuda.device(self.device):
            work = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
            out = torch.empty((len(t_out), self.nvar, self.n), dtype=self.torch_dtype, device=self.device)
        work.record_stream(self.stream)
        out.record_stream(self.stream)
        self.stream.wait_stream(torch.cuda.current_stream())
        base = (work.data_ptr() + 255) // 256 * 256
        st = (C.c_double * 5)()
        rc = lib().net_integrate_adaptive_dense(self.h, len(t_out), t_out.ctypes.data, out.data_ptr(), float(rtol),
                                                float(atol), float(h0), int(max_attempts), base, need, st)
        _check(rc, self.h)
        torch.cuda.current_stream().wait_stream(self.stream)
        info = dict(accepted=int(st[0]), rejected=int(st[1]), h_last=st[2], h_next=st[3], t=st[4])
        return out.cpu().numpy(), info

    def integrate_observed(self, n_steps, dt, obs_every):
        net_integrate_observed(self.h, int(n_steps), float(dt), int(obs_every))
        st = np.empty(8)
        net_observables(self.h, OBS_STATS, st.ctypes.data, False)
        return dict(R_mean=st[0], R_std=st[1], Rloc_mean=st[2], vel_mean=st[3], vel_std=st[4],
                    n_samples=int(st[5]), t_a=st[6], t_b=st[7])

    def eval_rhs(self, out=None):
        if out is None:
            out = np.empty((self.nvar, self.n), dtype=self.np_dtype)
        net_eval_rhs(self.h, *self._ptr(out))
        self._publish(out)
        return out

    def observable(self, what):
        size = (2 if what == OBS_GLOBAL_ORDER else 8 if what == OBS_STATS else
                2 * self.batch if what == OBS_REPLICA_ORDER else self.n)
        out = np.empty(size)
        net_observables(self.h, what, out.ctypes.data, False)
        return out

    def get_topology(self, row_begin=0, row_count=None):
        row_count = self.n - row_begin if row_count is None else row_count
        nnz, deg = net_get_degree(self.h)
        rp = np.empty(row_count + 1, dtype=np.int64)
        if deg >= 0:
            cnt = row_count * deg
        else:       # general CSR: at most nnz entries
            cnt = nnz
        ci = np.empty(max(cnt, 1), dtype=np.int32)
        net_get_topology(self.h, row_begin, row_count, rp.ctypes.data, ci.ctypes.data, False)
        return rp, ci[:rp[-1]]

    def degree(self):
        return net_get_degree(self.h)

    def time(self):
        return net_get_time(self.h)

    def counters(self):
        return net_get_counters(self.h)

    def kernel_family(self):
        return net_get_kernel_family(self.h)

    def probe_latency(self):
        return net_probe_latency(self.h)

    def launch_config(self):
        return net_get_launch_config(self.h)

    def probe_peaks(self):
        return net_probe_peaks(self.h)

    def synchronize(self):
        net_synchronize(self.h)
