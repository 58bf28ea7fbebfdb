#!/usr/bin/env python
"""bench.py -- oscillator-steps/s of the fused RK4 hot path on B200, against its roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]
                    [--no-per-config] [--no-cpu-baseline] [--no-rewrite-error] [--next-rows]

One bench "step" = one net_integrate call of BENCH_RK4[cfg] RK4 steps over the whole network
(the output interval `obs_every` of the workload for the large nets; the whole 1000-step run
for the 256-oscillator ring, whose single call is one persistent kernel).  `value` = N x RK4 steps / s with the
state resident in HBM; `e2e` = the same through the C ABI with HOST buffers (net_set_state from
pinned memory + net_integrate + net_get_state to pinned memory inside the timed region).
The headline workload is config 5 (the metric is quoted per config;
config 5 is the largest one and has a clean HBM roofline); `per_config` carries the same
measurement for every other north-star config (and the same facts as a compact table in
`roofline.per_config`); `next_rows` measures the SURVEY.md 8(f) rows (Dormand-Prince 5(4), the
compressed coupling matrix, eq. (2) with delay and noise).  N > 1 GPUs = independent replicas (weak
scaling, no collective on the data path).  `--impl reference` times the CPU oracle, as it
stands, on a bounded sample of the same workload.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "oscillator-steps/s"
HEADLINE = "5"
# 1b: config 1 as a batch of nets (extra, SURVEY.md 8(d) iii); 6 / 6b / 6c: the paper's own performance model
# (KS with inertia, Fig. 6c) at its radii P = 2 / 4 / 6 (extras)
PER_CONFIG = ("1", "1b", "2", "3a", "3b", "4", "5", "6", "6b", "6c")
# RK4 steps per bench step (= per net_integrate call)
BENCH_RK4 = {"6": 10, "6b": 10, "6c": 10, "1": 1000, "1b": 1000, "2": 200, "3a": 10, "3b": 10, "4": 100, "5": 10}


def ntot(w):
    """Elements of all replicas of the workload (batch > 1: independent nets integrated together)."""
    return w.n * getattr(w, "batch", 1)


# ------------------------------------------------------------------ inputs
def make_inputs(w, seed=1):
    """Seeded synthetic inputs of DESIGN.md "Input recipe" (numpy only; HH gates are set to
    their steady state by the consumer)."""
    import numpy as np
    from paper_2410_19075_b200 import configs, inputs
    dt = np.float32 if w.dtype == "f32" else np.float64
    elem = None
    if w.model == configs.KS:
        y0 = inputs.ks_phases(ntot(w), seed).reshape(1, -1)
        if w.extra.get("omega") == "lorentzian":
            elem = inputs.lorentzian_omega(ntot(w), seed, w.extra["gamma"], w.extra["omega_max"])
    elif w.model == configs.KSI:
        y0 = np.stack([inputs.ks_phases(ntot(w), seed), 0.05 * inputs.fhn_circle(ntot(w), seed)[0]])
    elif w.model == configs.FHN:
        y0 = inputs.fhn_circle(ntot(w), seed)
    else:
        V = inputs.hh_voltage(ntot(w), seed)
        y0 = np.zeros((4, ntot(w)))
        y0[0] = V
        elem = inputs.hh_current(ntot(w), seed)
    return np.ascontiguousarray(y0.astype(dt)), None if elem is None else elem.astype(dt)


# ------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, device_index):
        self.samples, self.mask, self.max_mhz, self.ok = [], 0, None, False
        self._stop = threading.Event()
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = "GPU-" + str(torch.cuda.get_device_properties(device_index).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:      # no NVML: report that, never fake a clock
            self.err = repr(e)

    def _one(self):
        try:
            self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
            self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            self._one()
            self._stop.wait(0.02)

    def __enter__(self):
        if self.ok:
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()
        return self

    def __exit__(self, *a):
        if self.ok:
            self._stop.set()
            self.t.join()
            self._one()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml_unavailable"]}
        s = sorted(self.samples)
        reasons = [n for b, n in self.REASONS.items() if self.mask & b]
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(s)}


# ------------------------------------------------------------------ our arm
def build_net(w, device, seed=1, method=None, y0_map=None):
    from paper_2410_19075_b200 import binding as B, configs
    y0, elem = make_inputs(w, seed)
    if y0_map is not None:
        y0 = y0_map(y0)
    net = B.Net.from_workload(w, device=device, method=B.METHOD_AUTO if method is None else method)
    net.set_state(y0)
    if elem is not None:
        net.set_param_array(B.PARAM_OMEGA if w.model in (configs.KS, configs.KSI) else B.PARAM_IEXT, elem)
    if w.model == configs.HH:
        net.hh_steady_gates()
        y0 = net.get_state()                # full initial state (gates included) for the e2e leg
    return net, y0


def measure(w, device, steps, warmup, e2e=True, seed=1, peaks=False):
    """Times `steps` bench steps (each = BENCH_RK4[cfg] RK4 steps) after `warmup` untimed ones.
    Returns device-resident ms, e2e ms, launches and byte counts."""
    import torch
    from paper_2410_19075_b200 import replicas
    net, y0 = build_net(w, device, seed)
    S = BENCH_RK4[w.cfg]
    stream = net.stream
    for _ in range(warmup):
        net.integrate(S, w.dt)
    net.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = net.counters()[0]
    with ClockSampler(torch.device(device).index or 0) as clk:
        replicas.barrier()
        torch.cuda.synchronize()
        ev0.record(stream)
        for _ in range(steps):
            net.integrate(S, w.dt)
        ev1.record(stream)
        torch.cuda.synchronize()
        replicas.barrier()
    ms = ev0.elapsed_time(ev1)
    launches = net.counters()[0] - l0
    method = net.counters()[1]
    out = dict(ms=ms, launches=launches, method=method, clocks=clk.summary(), rk4_per_step=S,
               launch_config=net.launch_config())
    if peaks:
        out["measured_peaks"] = net.probe_peaks()
    if e2e:
        host_in = torch.from_numpy(y0).pin_memory()
        host_out = torch.empty_like(host_in).pin_memory()
        # warm-up of the host path
        net.set_state(host_in)
        net.integrate(S, w.dt)
        net.get_state(host_out)
        replicas.barrier()
        torch.cuda.synchronize()
        ev0.record(stream)
        for _ in range(steps):
            net.set_state(host_in)          # H2D from pinned memory (C ABI, host pointer)
            net.integrate(S, w.dt)
            net.get_state(host_out)         # D2H of the step's result
        ev1.record(stream)
        torch.cuda.synchronize()
        replicas.barrier()
        out.update(e2e_ms=ev0.elapsed_time(ev1), h2d=host_in.numel() * host_in.element_size(),
                   d2h=host_out.numel() * host_out.element_size())
    # ring nets are bound by the dependent chain of a stage: probe its primitives (SURVEY.md 8(d) ii)
    from paper_2410_19075_b200 import configs as _cfgs
    if w.topo == _cfgs.RING and getattr(w, "batch", 1) == 1 and method == 2:
        try:
            out["latency"] = net.probe_latency()
        except Exception as exc:               # diagnostic only
            out["latency"] = {"error": str(exc)}
    # the same step with the workload's observables switched on (global / local order parameter and
    # mean phase velocity sampled every obs_every RK4 steps; reported separately)
    if e2e:
        net.integrate_observed(S, w.dt, w.obs_every)
        replicas.barrier()
        torch.cuda.synchronize()
        ev0.record(stream)
        for _ in range(steps):
            net.integrate_observed(S, w.dt, w.obs_every)     # includes the D2H of the 8 statistics
        ev1.record(stream)
        torch.cuda.synchronize()
        replicas.barrier()
        out.update(obs_ms=ev0.elapsed_time(ev1))
    net.close()
    del net
    torch.cuda.empty_cache()
    return out


def rewrite_error(w, device):
    """Error of the exact-in-mathematics rewrites of the coupling sum (run sums, prefix sums,
    factorised sine, blocked gathers), measured on the GPU itself at the full size of the workload
    (BASELINE.json item 3): max_v ||f_FAST - f_DIRECT||_inf / ||f_DIRECT||_inf of one
    right-hand side, in the seeded incoherent state and in a nearly coherent one.  DIRECT is the
    plain per-link form of Alg. 1 in the arithmetic type of the net."""
    import numpy as np
    from paper_2410_19075_b200 import binding as B, configs
    out = {}
    states = [("incoherent", None)]
    if w.model != configs.HH:                  # HH gates are set to their steady state of V by the library
        states.append(("coherent", lambda y: (y * 1e-2 + 0.3).astype(y.dtype)))
    for name, ymap in states:
        f = {}
        for method in (B.METHOD_FAST, B.METHOD_DIRECT):
            net, _ = build_net(w, device, method=method, y0_map=ymap)
            f[method] = net.eval_rhs().astype(np.float64)
            net.close()
            del net
        err = 0.0
        for v in range(f[B.METHOD_FAST].shape[0]):
            ref = np.abs(f[B.METHOD_DIRECT][v]).max()
            if w.model == configs.HH:
                ref = max(ref, 1.0)            # reading R11: gates start at steady state, f = 0 there
            err = max(err, float(np.abs(f[B.METHOD_FAST][v] - f[B.METHOD_DIRECT][v]).max() / ref))
        out[name] = err
    out["norm"] = "max over variables of ||f_FAST - f_DIRECT||_inf / ||f_DIRECT||_inf, one RHS at full size, on the GPU"
    return out


def ncu_traffic(cfg):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the stage kernel, from the
    committed `ncu --set full` capture of this build (profiles/ncu_traffic.csv: cfg, mean bytes
    per captured launch, launches captured; None when there is no line for this workload)."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for line in f:
                parts = [p.strip() for p in line.split(",")]
                if len(parts) >= 2 and parts[0] == cfg:
                    return float(parts[1])
    except Exception:
        pass
    return None


def roofline_object(w, m, steps):
    """roofline of the dominant kernel (the fused RHS+RK4 stage kernel; every launch in the timed
    region is one of its four stage instances)."""
    from paper_2410_19075_b200 import roofline as R
    pk = R.peaks()
    c = R.ceiling(w, pk)
    rk4 = steps * m["rk4_per_step"]
    sec = m["ms"] * 1e-3
    avg_launch_s = sec / max(1, m["launches"])
    if c["bound"] == "hbm":
        per_launch = R.bytes_per_osc_step(w) * ntot(w) * rk4 / max(1, m["launches"])
        achieved, peak, unit = per_launch / avg_launch_s / 1e9, pk["hbm_gbs"], "GB/s"
        peak_src = "MEASURED_PEAKS.json hbm_gbs" if pk["hbm_source"] == "measured" else "guide fallback"
    else:
        per_launch = c["ops"] * ntot(w) * rk4 / max(1, m["launches"])
        achieved, peak, unit = per_launch / avg_launch_s / 1e9, pk[c["pipe"] + "_ginstr_s"], "Ginstr/s"
        peak_src = ("148 SM x %d lanes x sm_max_mhz (%s)" %
                    (R.LANES[c["pipe"]], "issue slots, all pipes" if c["pipe"] == "issue" else c["pipe"] + " pipe"))
    value = ntot(w) * rk4 / sec
    return {"bound": c["bound"], "achieved": achieved, "peak": peak, "unit": unit,
            "frac": achieved / peak, "traffic": ncu_traffic(w.cfg),
            "kernel": "fused RHS+RK4 stage kernel",
            "frac_of_nominal_8tbs": (achieved / 8000.0 if c["bound"] == "hbm" else None),
            "avg_launch_us": avg_launch_s * 1e6, "peak_source": peak_src,
            "bytes_per_osc_step": R.bytes_per_osc_step(w),
            "survey_bytes_per_osc_step": R.survey_bytes_per_osc_step(w),
            "ops_per_osc_step": c["ops"], "ops_pipe": c["pipe"], "ops_source": c["ops_source"],
            "ceiling_osc_steps_per_s": c["osc_steps_per_s"],
            "frac_of_ceiling": value / c["osc_steps_per_s"],
            # the direct (one term per link) formulation beside it, so that the rewrite cannot
            # inflate the fraction: > 1 means the shipped form beats what the direct form could reach
            "direct_formulation": {"ops_per_osc_step": c["direct_ops"], "pipe": c["direct_pipe"],
                                   "ceiling_osc_steps_per_s": c["direct_osc_steps_per_s"]},
            "frac_direct_formulation": value / c["direct_osc_steps_per_s"]}


# ------------------------------------------------------------------ SURVEY.md 8(f) rows, measured
def measure_next_rows(device, steps):
    """The rows SURVEY.md 8(f) lists as next, each measured on a synthetic workload of the paper's
    shape (3D ball of radius 2 on 100^3 = 10^6 elements, fp64, the size of the paper's own performance
    tests) with the metric of the bench and the roofline of its formulation:
      dp5        adaptive Dormand-Prince 5(4) (net_integrate_adaptive) on the KS lattice: N x accepted
                 steps / s; bytes per attempt = 6 RHS evaluations (read state, write k: 2 words each)
                 + the stage combinations (sum_{s=1..6} (s + 2) words) + error norm (9) + commit (4);
      compressed the coupling matrix of Alg. 2 (net_compress_csr of the lattice's CSR, EXTRACT inside
                 the per-link kernels) beside the same net given as a lattice (offset table) and as
                 plain CSR, all on the per-link DIRECT form: the paper's "decompression increases
                 computing time 2-5 folds compared to uncompressed bit arrays";
      delay      eq. (2) with delay 5 dt and noise (NET_MODEL_FHN2), per-link form.
    The per-link forms are bound by the FP64 sines / the gathers of the direct formulation."""
    import numpy as np
    import torch
    from paper_2410_19075_b200 import binding as B, configs, inputs, roofline as R
    pk = R.peaks()
    out = {}
    n1, P = 100, 2
    n = n1 ** 3
    from dataclasses import replace
    w = replace(configs.get("3b", n1=n1), radius=P, name="KS 3D %d^3 radius %d f64" % (n1, P))
    y0, elem = make_inputs(w, 1)

    def run_fixed(net, rk4_steps, reps):
        for _ in range(3):
            net.integrate(rk4_steps, w.dt)
        net.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(net.stream)
        for _ in range(reps):
            net.integrate(rk4_steps, w.dt)
        ev1.record(net.stream)
        torch.cuda.synchronize()
        return n * rk4_steps * reps / (ev0.elapsed_time(ev1) * 1e-3)

    def ks_net(topo, method):
        net = B.Net(w.model, B.F64, n, topo, w.params, method=method, device=device)
        net.set_state(y0)
        net.set_param_array(B.PARAM_OMEGA, elem)
        return net

    lattice = dict(kind=B.TOPO_LATTICE, extent=w.extent, radius=P)
    # ---- Dormand-Prince 5(4)
    net = ks_net(lattice, B.METHOD_AUTO)
    net.integrate_adaptive(1.0, 1e-8, 1e-11, 0.05)      # warm-up and the controller settles
    net.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = net.time()[0]
    ev0.record(net.stream)
    info = net.integrate_adaptive(t0 + 10.0 * max(1, steps // 5), 1e-8, 1e-11, 0.05)
    ev1.record(net.stream)
    torch.cuda.synchronize()
    sec = ev0.elapsed_time(ev1) * 1e-3
    attempts = info["accepted"] + info["rejected"]
    words = 6 * 2 + sum(s + 2 for s in range(1, 7)) + 9 + 4
    gbs = attempts * n * words * 8 / sec / 1e9
    out["dp5"] = {"workload": w.name + ", rtol 1e-8, atol 1e-11", "value": n * info["accepted"] / sec, "unit": METRIC,
                  "accepted": info["accepted"], "rejected": info["rejected"], "ms_per_attempt": sec * 1e3 / max(1, attempts),
                  "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": gbs / pk["hbm_gbs"],
                               "bytes_per_element_and_attempt": words * 8,
                               "note": "state-sized vectors of the integrator only (58 words per element and attempt); the 6 "
                                       "RHS launches inside are the lattice kernels of config 3b; every evaluation also pays two "
                                       "layout copies (DESIGN.md section 5)"}}
    net.close()
    # ---- compressed matrix against the same topology as offset table and as plain CSR (all DIRECT)
    net = ks_net(lattice, B.METHOD_DIRECT)
    v_lat = run_fixed(net, 4, max(2, steps // 2))
    rp, ci = net.get_topology()
    net.close()
    t_c = time.perf_counter()
    cm = B.net_compress_csr(rp, ci)
    t_c = time.perf_counter() - t_c
    net = ks_net(dict(kind=B.TOPO_CSR, row_ptr=rp, col_idx=ci), B.METHOD_DIRECT)
    v_csr = run_fixed(net, 4, max(2, steps // 2))
    net.close()
    net = ks_net(dict(kind=B.TOPO_COMPRESSED, compressed=cm), B.METHOD_DIRECT)
    v_cmp = run_fixed(net, 4, max(2, steps // 2))
    net.close()
    v, dptr, dpos, c = cm.arrays()
    deg = len(ci) // n
    sine_ceiling = pk["fp64_ginstr_s"] * 1e9 / (4 * deg * R.SINE_FP64_INSTR)
    out["compressed"] = {"workload": w.name + " as a compressed coupling matrix (Alg. 2), per-link form", "value": v_cmp,
                         "unit": METRIC, "same_topology_as_offset_table": v_lat, "same_topology_as_csr": v_csr,
                         "slowdown_vs_csr": v_csr / v_cmp, "table_entries": int(len(dptr) - 1),
                         "compressed_bytes": int(4 * (len(v) + len(dpos) + len(c)) + 8 * len(dptr)),
                         "csr_bytes": int(4 * len(ci) + 8 * len(rp)), "host_compress_s": t_c,
                         "roofline": {"bound": "alu", "achieved": v_cmp * 4 * deg * R.SINE_FP64_INSTR / 1e9,
                                      "peak": pk["fp64_ginstr_s"], "unit": "Ginstr/s",
                                      "frac": v_cmp / sine_ceiling,
                                      "note": "direct formulation: one fp64 sine (~60 FP64-pipe instructions) per link and stage"}}
    # ---- eq. (2) with delay and noise (per-link form)
    th = inputs.fhn_circle(n, 1)
    P2 = dict(eps=0.05, a=0.5, sigma=0.3, I_app=0.0)
    for name, m, D in (("delay", 5, 0.05), ("no_delay", 0, 0.0)):
        net = B.Net(B.MODEL_FHN2, B.F64, n, lattice, dict(P2, D=D, seed=3), device=device, delay_steps=m)
        net.set_state(th)
        val = run_fixed(net, 4, max(2, steps // 2))
        net.close()
        if name == "delay":
            # per stage and element: deg gathers of the delayed x (midpoint stages: 4 history values per link)
            out["delay"] = {"workload": "eq. (2) FHN 3D %d^3 radius %d f64, delay 5 dt, noise" % (n1, P), "value": val, "unit": METRIC}
        else:
            out["delay"]["without_delay_and_noise"] = val
    out["delay"]["roofline"] = {"bound": "gathers (L1 / L2; lattice neighbours are local)", "unit": "gathers/s",
                                "achieved": out["delay"]["value"] * deg * (1 + 4 + 4 + 1),
                                "note": "per oscillator-step: deg x (1 + 4 + 4 + 1) history values gathered per link "
                                        "(stage 0 and 3 one slot, the midpoint stages two slots of x and dx/dt); compare with "
                                        "roofline.measured_peaks.l2_gather_gops x 1e9"}
    return out


# ------------------------------------------------------------------ CPU oracle arm
SAMPLE = {"1": dict(), "2": dict(n=16384), "3a": dict(n1=64), "3b": dict(n1=64),
          "4": dict(n=200_000), "5": dict(n1=160)}


def oracle_sample(cfg, seed=1):
    """The oracle, as it stands, on a bounded sample of workload `cfg`: same model, parameters,
    radius rule, dtype rounding and step on a smaller ring / lattice / graph (SAMPLE).
    Returns (sample workload, OracleNet, y0)."""
    import numpy as np
    from oracle import oracle as ora           # the one place bench.py may load oracle/
    from paper_2410_19075_b200 import configs
    w = configs.get(cfg, **SAMPLE[cfg])
    y0, elem = make_inputs(w, seed)
    y0 = y0.astype(np.float64)
    if w.topo == configs.RING:
        rp, ci = ora.topology_ring(w.n, w.radius)
    elif w.topo == configs.LATTICE:
        rp, ci = ora.topology_lattice(w.extent, w.radius)
    else:
        rp, ci = ora.topology_random_indegree(w.n, w.in_degree, w.topo_seed)
    p = w.params
    if w.model == configs.KS:
        om = np.full(w.n, p["omega0"]) if elem is None else elem.astype(np.float64)
        net = ora.OracleNet.ks(w.n, rp, ci, p["K"], p["alpha"], om)
    elif w.model == configs.FHN:
        net = ora.OracleNet.fhn(w.n, rp, ci, p["eps"], p["a"], p["sigma"], p["phi"])
    else:
        y0[1], y0[2], y0[3] = ora.hh_steady_gates(y0[0])
        net = ora.OracleNet.hh(w.n, rp, ci, elem.astype(np.float64), **p)
    return w, net, y0, ora.omp_threads()


def time_oracle(cfg, budget_s=20.0, rk4_steps=None):
    """oscillator-steps/s of the oracle on its sample; about budget_s of CPU work."""
    w, net, y0, cores = oracle_sample(cfg)
    t0 = time.perf_counter()
    y = net.rk4(y0, 1, w.dt)
    one = max(time.perf_counter() - t0, 1e-6)
    if rk4_steps is None:
        rk4_steps = int(max(1, min(w.n_steps, budget_s / one)))
    t0 = time.perf_counter()
    net.rk4(y, rk4_steps, w.dt)
    sec = time.perf_counter() - t0
    return dict(value=w.n * rk4_steps / sec, unit=METRIC, cores=cores, kind="oracle",
                sample="%s, %d RK4 steps, %.1f s (plain C fp64, direct neighbour sums, OpenMP over "
                       "elements)" % (w.name, rk4_steps, sec)), w, sec, rk4_steps


def run_reference(args):
    from paper_2410_19075_b200 import configs, replicas
    rank, _, ws = replicas.world()
    if rank != 0:
        return 0
    full = configs.get(args.config)
    w, net, y0, cores = oracle_sample(args.config)
    t0 = time.perf_counter()
    y = net.rk4(y0, 1, w.dt)
    one = max(time.perf_counter() - t0, 1e-6)
    # each bench step = a bounded number of RK4 steps of the sample (<= BENCH_RK4[cfg], ~<= 4 s)
    S = int(max(1, min(BENCH_RK4[full.cfg], 4.0 / one)))
    for _ in range(args.warmup):
        y = net.rk4(y, S, w.dt)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        y = net.rk4(y, S, w.dt)
    sec = time.perf_counter() - t0
    value = w.n * S * args.steps / sec
    sample = "%s, %d RK4 steps per bench step" % (w.name, S)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": METRIC,
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": sec * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": full.name, "cfg": full.cfg, "sample": sample},
            "cpu_baseline": {"value": value, "unit": METRIC, "cores": cores, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": METRIC, "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------ main
def line_for(w, m, steps, n_gpus, units_total=None, ms_max=None):
    """The JSON fields of one measured workload (headline or per_config entry)."""
    rk4 = steps * m["rk4_per_step"]
    ms = m["ms"] if ms_max is None else ms_max
    units = ntot(w) * rk4 * n_gpus if units_total is None else units_total
    out = {"workload": w.name, "cfg": w.cfg, "value": units / (ms * 1e-3), "unit": METRIC,
           "ms_per_step": ms / steps, "rk4_steps_per_step": m["rk4_per_step"],
           "dtype": w.dtype, "method": "FAST" if m["method"] == 2 else "DIRECT",
           "gpu_launches": m["launches"], "roofline": roofline_object(w, m, steps)}
    if "e2e_ms" in m:
        out["e2e"] = {"value": ntot(w) * rk4 * n_gpus / (m["e2e_ms"] * 1e-3), "unit": METRIC,
                      "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"]}
    if "latency" in m and "error" not in m["latency"]:
        from paper_2410_19075_b200 import configs as _cfgs
        L = m["latency"]
        stage_us = ms * 1e3 / (rk4 * 4)
        # dependent chain of one stage of the persistent ring kernel: scan of the fields, grid barrier,
        # one L2 round trip (totals + prefix values), scan of the totals (multi-CTA nets only), and for
        # KS one fp64 sincos of the new phase
        floor = L["block_scan_us"] + (L["fp64_sincos_us"] if w.model == _cfgs.KS else 0.0)
        if L["grid_barrier_us"] > 0:
            floor += L["grid_barrier_us"] + L["l2_round_trip_us"] + L["block_scan_us"]
        out["latency_model"] = dict(L, stage_floor_us=floor, stage_us=stage_us, frac=floor / stage_us,
                                    what="measured latencies of the primitives one stage chains (net_probe_latency); "
                                         "frac = their sum / measured time per RK4 stage")
    if "obs_ms" in m:
        out["with_observables"] = {"value": ntot(w) * rk4 * n_gpus / (m["obs_ms"] * 1e-3), "unit": METRIC,
                                   "obs_every": w.obs_every,
                                   "what": "net_integrate_observed: global and local order parameter, mean phase "
                                           "velocity sampled every obs_every RK4 steps, statistics read back"}
    return out


def run_ours(args):
    import torch
    from paper_2410_19075_b200 import binding, configs, replicas
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    binding.lib()                                   # fail loudly if liboscnet.so is missing
    rank, local_rank, ws = replicas.world()
    torch.cuda.set_device(local_rank)
    device = "cuda:%d" % local_rank
    if ws > 1:
        replicas.init("nccl")
    if args.next_rows:
        if rank == 0:
            print(json.dumps({"next_rows": measure_next_rows(device, args.steps)}), flush=True)
        return 0
    w = configs.get(args.config)
    m = measure(w, device, args.steps, args.warmup, e2e=True, peaks=True)
    rk4 = args.steps * m["rk4_per_step"]
    units, ms_max, value = replicas.aggregate(ntot(w) * rk4, m["ms"], device)
    _, e2e_ms_max, e2e_value = replicas.aggregate(ntot(w) * rk4, m["e2e_ms"], device)
    head = line_for(w, m, args.steps, ws, units, ms_max)
    line = {"metric": METRIC, "value": value, "unit": METRIC, "n_gpus": ws, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": w.dtype, "data": "synthetic",
            "config": {"workload": w.name, "cfg": w.cfg, "n": w.n, "dt": w.dt,
                       "rk4_steps_per_step": m["rk4_per_step"], "method": head["method"],
                       "parallelism": "replicas x%d (no data-path collective)" % ws,
                       "l2": ("state arrays larger than L2 (no flush needed)"
                              if w.n * w.nvar * (4 if w.dtype == "f32" else 8) > 126e6 else
                              "state smaller than L2 by definition of the workload; resident by design")},
            "clocks": m["clocks"],
            "e2e": {"value": e2e_value, "unit": METRIC, "h2d_bytes_per_step": m["h2d"],
                    "d2h_bytes_per_step": m["d2h"]},
            "gpu_launches": m["launches"], "roofline": head["roofline"]}
    line["config"]["tile"] = m["launch_config"]
    if "measured_peaks" in m:
        # net_probe_peaks: the ALU / shared-memory / L2-gather ceilings
        # measured on this device, beside the nominal unit counts x clock the fractions divide by
        from paper_2410_19075_b200 import roofline as R
        pk = R.peaks()
        line["roofline"]["measured_peaks"] = dict(
            m["measured_peaks"], nominal_fp32_ginstr_s=pk["fp32_ginstr_s"], nominal_fp64_ginstr_s=pk["fp64_ginstr_s"],
            nominal_mufu_ginstr_s=pk["mufu_ginstr_s"])
    if "with_observables" in head and ws == 1:
        line["with_observables"] = head["with_observables"]
    if "latency_model" in head and ws == 1:
        line["latency_model"] = head["latency_model"]
    if getattr(w, "batch", 1) > 1:
        line["config"]["batch"] = w.batch
    if rank == 0 and ws == 1 and not args.no_rewrite_error:
        line["rewrite_error"] = rewrite_error(w, device)
    if rank == 0 and ws == 1 and not args.no_per_config:
        per = []
        for cfg in PER_CONFIG:
            if cfg == w.cfg:
                continue
            wc = configs.get(cfg)
            k = max(3, min(args.steps, 10))
            mc = measure(wc, device, k, max(3, args.warmup), e2e=True)
            e = line_for(wc, mc, k, 1)
            e["clocks"] = mc["clocks"]
            e["tile"] = mc["launch_config"]
            if not args.no_rewrite_error:
                e["rewrite_error"] = rewrite_error(wc, device)
            per.append(e)
        line["per_config"] = per
        # the same facts in a compact table inside `roofline` (a key every record of the run keeps)
        bad = {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
        tab = {}
        for e in [dict(head, clocks=m["clocks"])] + per:
            r = e["roofline"]
            tab[e["cfg"]] = {"value": e["value"], "bound": r["bound"], "frac": r["frac_of_ceiling"],
                             "frac_direct_formulation": r["frac_direct_formulation"],
                             "us_per_launch": r["avg_launch_us"],
                             "with_observables": e.get("with_observables", {}).get("value"),
                             "sm_mhz": e["clocks"]["sm_mhz"],
                             "clocks_ok": not (bad & set(e["clocks"]["reasons"]))}
        line["roofline"]["per_config"] = tab
    if rank == 0 and ws == 1 and not args.no_per_config:
        line["next_rows"] = measure_next_rows(device, args.steps)
    if rank == 0 and ws == 1 and not args.no_cpu_baseline:
        cb, _, _, _ = time_oracle(w.cfg)
        line["cpu_baseline"] = cb
    if rank == 0:
        print(json.dumps(line), flush=True)
    if ws > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=HEADLINE, choices=list(PER_CONFIG))
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-rewrite-error", action="store_true")
    ap.add_argument("--next-rows", action="store_true",
                    help="measure only the SURVEY.md 8(f) rows (next_rows of the full line) and print them")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
