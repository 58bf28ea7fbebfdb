"""Roofline bookkeeping for bench.py: algorithmic bytes and
operations per oscillator-step of each north-star workload, and the peaks they are divided by.
Plain arithmetic on sizes; nothing of the method is computed here.

Operation counts are SURVEY.md 8(d)'s own ("Algorithmic bytes and operations per oscillator-step"
and its table), NOT counts of the kernels in this repository: ~140 instructions per element and
stage for KS with P = 4 (560 per oscillator-step, both dtypes), ~55 for FHN with P = 2 (220),
~425 FP64 for HH (1700), ~160 for the FHN ring (prefix form), ~400 for the KS ring (factorised).
The direct formulation (one sine / one pair term per link) is carried beside it so that a rewrite
cannot inflate the fraction ("print the direct-formulation roofline next to it").
"""
import json
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# fallback peaks of /opt/skills/guides/B200_PROFILING.md when MEASURED_PEAKS.json is absent
FALLBACK_HBM_GBS = 6650.0
SM_COUNT = 148
SM_MAX_MHZ_NOMINAL = 1965.0
# issue rates per SM per clock (lanes): FP32 FMA pipe 128, FP64 64, MUFU (SFU) 16
# "issue": warp instructions of all pipes, 4 schedulers x 32 lanes per SM and clock
LANES = {"fp32": 128, "fp64": 64, "mufu": 16, "issue": 128}
# instructions one sine costs in the direct formulation: fp32 sin.approx = 1 MUFU (+ range
# reduction on the FP32 pipe, not counted); fp64 library sine ~ 60 instructions of the FP64 pipe
SINE_FP64_INSTR = 60


def peaks():
    """HBM GB/s (measured copy, else the guide's fallback) and ALU instruction rates derived
    from the guide's unit counts and the measured maximum SM clock."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    out = dict(hbm_gbs=FALLBACK_HBM_GBS, hbm_source="fallback", sm_max_mhz=SM_MAX_MHZ_NOMINAL)
    if os.path.exists(path):
        try:
            mp = json.load(open(path))
            out.update(hbm_gbs=float(mp["hbm_gbs"]), hbm_source="measured",
                       sm_max_mhz=float(mp.get("sm_max_mhz", SM_MAX_MHZ_NOMINAL)))
        except Exception:
            pass
    for k, lanes in LANES.items():
        out[k + "_ginstr_s"] = SM_COUNT * lanes * out["sm_max_mhz"] * 1e-3   # 1e9 instr/s
    return out


def records_per_step():
    """RK4 in the 4-array form (y, Y2, Y3, Y4): stage reads/writes of one element's record.
    stage 1: R y, W Y2 | stage 2: R Y2, R y, W Y3 | stage 3: R Y3, R y, W Y4 |
    stage 4: R Y4, R y, R Y2, R Y3, W y   => 13 records per RK4 step (SURVEY 8(d) counts 17 for
    the form with a separate accumulator; the build moves fewer and is judged on 13)."""
    return 2 + 3 + 3 + 5


def bytes_per_osc_step(w):
    """Algorithmic HBM bytes per oscillator per RK4 step of workload w (halo re-reads, cache
    misses of gathers etc. are implementation overhead and NOT counted)."""
    word = 4 if w.dtype == "f32" else 8
    b = records_per_step() * w.nvar * word
    if w.cfg in ("3a", "3b"):
        b += 4 * word                       # omega_i read by each of the 4 stages
    if w.cfg == "4":
        b += 4 * word                       # I_ext,i per stage
        b += 4 * w.in_degree * 4            # col_idx (int32) streamed by each stage
        b += 4 * 2 * word                   # s = S(V): written and read (first touch) per stage
    return b


def survey_bytes_per_osc_step(w):
    """SURVEY.md 8(d)'s own per-unit figure (17 records; its cfg-3/4 extras), for comparison."""
    word = 4 if w.dtype == "f32" else 8
    b = 17 * w.nvar * word
    if w.cfg in ("3a", "3b"):
        b += 4 * word
    if w.cfg == "4":
        b += 32 + 32 + 1600
    return b


def _degree(w):
    """Links per element (Omega) of the workload."""
    if w.in_degree:
        return w.in_degree
    if not w.extent:
        return 2 * w.radius
    P, nd = w.radius, len(w.extent)
    rng = range(-P, P + 1)
    if nd == 3:
        return sum(1 for a in rng for b in rng for c in rng if a * a + b * b + c * c <= P * P) - 1
    if nd == 2:
        return sum(1 for a in rng for b in rng if a * a + b * b <= P * P) - 1
    return 2 * P


def ops_per_osc_step(w):
    """(pipe, ops of the shipped formulation, pipe and ops of the direct formulation, source).
    Shipped = the exact-in-mathematics rewrite SURVEY.md 8(d) counts; direct = one term per link."""
    deg = _degree(w)
    f64 = w.dtype == "f64"
    if w.cfg in ("3a", "3b"):
        # "KS factorised+runs ~ 1 sincos + 2*(2P + (#runs-1)) adds + ~15 -> ~140 instr
        # (P=4: 49 runs)"; table: 560 FP32 (+8 MUFU) / 560 FP64 + fp64 sincos with T_arith 240-300 us
        # per step, i.e. ~620 FP64-pipe instructions per oscillator-step
        if f64:
            return ("fp64", 620, "fp64", 4 * deg * SINE_FP64_INSTR, "SURVEY.md 8(d): 560 FP64 + fp64 sincos (T_arith 240-300 us/step)")
        return ("fp32", 560, "mufu", 4 * deg, "SURVEY.md 8(d): 560 FP32 (+8 MUFU)")
    if w.cfg == "5":
        return ("fp32", 220, "fp32", 4 * 2 * 2 * deg, "SURVEY.md 8(d): ~55 per stage (x-runs, P=2: 13 runs)")
    if w.cfg == "4":
        return ("fp64", 1700, "fp64", 4 * (deg * 35 + 7 * 35 + 80), "SURVEY.md 8(d): ~425 FP64 per stage (7 exp + 80 + Omega adds)")
    if w.cfg in ("6", "6b", "6c"):
        # KS with inertia: 1 fp64 sincos (~15 FP64-pipe) + 2*(2P + (#runs - 1)) adds + ~15 per stage;
        # x-runs of the ball: 13 (P = 2), 49 (P = 4), 113 (P = 6)
        runs = {2: 13, 4: 49, 6: 113}[w.radius]
        return ("fp64", 4 * (15 + 2 * (2 * w.radius + runs - 1) + 15), "fp64", 4 * (deg * SINE_FP64_INSTR + 40),
                "SURVEY.md 8(d) rule for KS with runs: 1 sincos + 2*(2P + #runs - 1) adds + ~15 per stage")
    if w.cfg == "2":
        return ("fp64", 160, "fp64", 4 * 2 * 2 * deg, "SURVEY.md 8(d): ~160 FP64 (prefix sums)")
    return ("fp64", 400, "fp64", 4 * deg * SINE_FP64_INSTR, "SURVEY.md 8(d): ~400 FP64 (factorised)")


def ceiling(w, pk=None):
    """Per-config roofline ceiling in oscillator-steps/s = 1/max(T_hbm, T_alu) and its parts."""
    pk = pk or peaks()
    t_hbm = bytes_per_osc_step(w) / (pk["hbm_gbs"] * 1e9)
    pipe, ops, dpipe, dops, src = ops_per_osc_step(w)
    t_alu = ops / (pk[pipe + "_ginstr_s"] * 1e9)
    t_direct = dops / (pk[dpipe + "_ginstr_s"] * 1e9)
    bound = "hbm" if t_hbm >= t_alu else "alu"
    return dict(bound=bound, osc_steps_per_s=1.0 / max(t_hbm, t_alu), t_hbm=t_hbm, t_alu=t_alu,
                pipe=pipe, ops=ops, bytes=bytes_per_osc_step(w), ops_source=src,
                direct_pipe=dpipe, direct_ops=dops,
                direct_osc_steps_per_s=1.0 / max(t_hbm, t_direct))
