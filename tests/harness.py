"""Shared helpers of the parity tests: build the same workload on the oracle and on the GPU."""
import numpy as np

from oracle import oracle as ora
from paper_2410_19075_b200 import configs, inputs

TOL_RHS = {"f64": 1e-12, "f32": 1e-5}      # max-norm relative, per variable (reading R11)
TOL_TRAJ = {"f64": 1e-9, "f32": 1e-4}      # absolute after 100 steps (fp32 phases mod 2 pi, reading R6)
TOL_STATS = 1e-3


def ntot(w):
    """Elements of all replicas of the workload together."""
    return w.n * getattr(w, "batch", 1)


def make_inputs(w, seed=1):
    """Seeded inputs in float64, already rounded to the dtype of the net (reading R13).
    A batch gets independent draws for every replica: arrays are [nvar][batch * n]."""
    dt = np.float32 if w.dtype == "f32" else np.float64
    n_all = ntot(w)
    rnd = lambda a: np.ascontiguousarray(a.astype(dt).astype(np.float64))
    elem = None
    if w.model == configs.KS:
        y0 = inputs.ks_phases(n_all, seed).reshape(1, -1)
        if w.extra.get("omega") == "lorentzian":
            elem = inputs.lorentzian_omega(n_all, seed, w.extra["gamma"], w.extra["omega_max"])
        else:
            elem = np.full(n_all, w.params["omega0"])
    elif w.model == configs.KSI:
        # phases as for KS; initial frequencies psi = 0.1 (2u - 1) from the FHN stream of the seed
        y0 = np.stack([inputs.ks_phases(n_all, seed), 0.05 * inputs.fhn_circle(n_all, seed)[0]])
        elem = np.full(n_all, w.params["omega0"])
    elif w.model == configs.FHN:
        y0 = inputs.fhn_circle(n_all, seed)
    else:
        V = rnd(inputs.hh_voltage(n_all, seed))
        m, h, g = ora.hh_steady_gates(V)           # tests may call the oracle
        y0 = np.stack([V, m, h, g])
        elem = inputs.hh_current(n_all, seed)
    return dict(y0=rnd(y0), elem=None if elem is None else rnd(elem))


def _single_topology(w, row_begin=0, row_count=None):
    if w.topo == configs.RING:
        return ora.topology_ring(w.n, w.radius, False, row_begin, row_count)
    if w.topo == configs.LATTICE:
        return ora.topology_lattice(w.extent, w.radius, False, row_begin, row_count)
    return ora.topology_random_indegree(w.n, w.in_degree, w.topo_seed, row_begin, row_count)


def oracle_topology(w, row_begin=0, row_count=None):
    if getattr(w, "batch", 1) > 1:
        # the batch as one block-diagonal net: replica r owns elements r*n .. (r+1)*n - 1
        rp1, ci1 = _single_topology(w)
        B = w.batch
        ci = np.concatenate([ci1.astype(np.int64) + r * w.n for r in range(B)]).astype(np.int32)
        rp = np.concatenate([[0], np.cumsum(np.tile(np.diff(rp1), B))]).astype(np.int64)
        row_count = ntot(w) - row_begin if row_count is None else row_count
        lo, hi = rp[row_begin], rp[row_begin + row_count]
        return rp[row_begin:row_begin + row_count + 1] - lo, ci[lo:hi]
    return _single_topology(w, row_begin, row_count)


def make_oracle(w, inp, rows=None):
    """OracleNet of the workload.  rows = sorted element ids: only those rows get their
    neighbour lists (the others are left empty), for sampled checks at full size."""
    if rows is None:
        rp, ci = oracle_topology(w)
    else:
        lens = np.zeros(ntot(w) + 1, dtype=np.int64)
        parts = []
        for r in rows:
            _, c = oracle_topology(w, int(r), 1)
            parts.append(c)
            lens[r + 1] = len(c)
        rp = np.cumsum(lens)
        ci = np.concatenate(parts) if parts else np.zeros(0, dtype=np.int32)
    p = w.params
    if w.model == configs.KS:
        return ora.OracleNet.ks(ntot(w), rp, ci, p["K"], p["alpha"], inp["elem"])
    if w.model == configs.KSI:
        return ora.OracleNet.ksi(ntot(w), rp, ci, p["K"], p["alpha"], p["m"], p["eps"], inp["elem"])
    if w.model == configs.FHN:
        return ora.OracleNet.fhn(ntot(w), rp, ci, p["eps"], p["a"], p["sigma"], p["phi"])
    return ora.OracleNet.hh(ntot(w), rp, ci, inp["elem"], **p)


def make_gpu(w, inp, method=0):
    from paper_2410_19075_b200 import binding as B
    net = B.Net.from_workload(w, method=method)
    net.set_state(inp["y0"].astype(net.np_dtype))
    if inp["elem"] is not None:
        which = B.PARAM_OMEGA if w.model in (configs.KS, configs.KSI) else B.PARAM_IEXT
        net.set_param_array(which, inp["elem"].astype(net.np_dtype))
    return net


def rel_maxnorm(got, ref, floor=0.0):
    """max_v ||got_v - ref_v||_inf / max(||ref_v||_inf, floor)  (reading R11).

    floor > 0 is for states at which a variable's RHS vanishes identically (HH gates at their
    steady state: f = alpha (1-x) - beta x = 0 up to the rounding of its O(1) terms)."""
    got, ref = np.asarray(got, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    worst = 0.0
    for v in range(ref.shape[0]):
        den = max(np.abs(ref[v]).max(), floor)
        worst = max(worst, np.abs(got[v] - ref[v]).max() / (den if den > 0 else 1.0))
    return worst


def rhs_floor(w):
    """Denominator floor of the RHS parity norm: 1 (per ms) for HH, whose north-star initial
    state has the gates exactly at steady state; 0 (pure relative norm) otherwise."""
    return 1.0 if w.model == configs.HH else 0.0


def perturb_gates(w, y0, seed=11):
    """HH only: moves the gates off their steady state so every component of f is O(0.1)."""
    if w.model != configs.HH:
        return y0
    y = y0.copy()
    r = np.random.default_rng(seed).uniform(0.5, 1.5, size=(3, w.n))
    y[1:] = np.clip(y[1:] * r, 0.0, 1.0)
    dt = np.float32 if w.dtype == "f32" else np.float64
    return np.ascontiguousarray(y.astype(dt).astype(np.float64))


def traj_err(w, got, ref):
    """Max-norm state error.  fp64: plain absolute difference (the north star's 1e-9 absolute; a
    2 pi slip of a phase is an error).  fp32 phase models: the phase rows are compared modulo 2 pi
    (reading R6: unwrapped fp32 phases of fast elements lose absolute precision, their position on
    the circle does not)."""
    d = np.asarray(got, dtype=np.float64) - ref
    if w.dtype == "f32" and w.model in (configs.KS, configs.KSI):
        d[0] = d[0] - 2 * np.pi * np.round(d[0] / (2 * np.pi))
    return np.abs(d).max()
