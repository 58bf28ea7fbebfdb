"""Roofline bookkeeping for bench.py: algorithmic bytes and
operations per oscillator-step of each north-star workload, and the peaks they are divided by.
Plain arithmetic on sizes; nothing of the method is computed here."""
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


def ops_per_osc_step(w):
    """Arithmetic instructions per oscillator per RK4 step in the formulation that is shipped
    (pipe, count).  Estimates of DESIGN.md "Kernels"; used only to name the binding bound."""
    if w.cfg in ("3a", "3b"):
        # per stage: one sincos (fp32 ~40 instr, fp64 ~110), separable ball sum of (cos, sin):
        # x-runs 2*(2P+1) adds + 49 run combinations * 2, local field + stage update ~30
        per_stage = (40 if w.dtype == "f32" else 110) + 2 * 9 + 2 * 49 + 30
        return ("fp32" if w.dtype == "f32" else "fp64", 4 * per_stage)
    if w.cfg == "5":
        return ("fp32", 4 * (2 * 5 + 2 * 13 + 30))
    if w.cfg == "4":
        return ("fp64", 4 * (7 * 35 + 80 + w.in_degree))
    if w.cfg == "6":
        # DIRECT (per-link) form of Alg. 1: one fp64 sine (~60 instructions) per link and stage
        return ("fp64", 4 * (32 * 60 + 40))
    if w.cfg == "2":
        return ("fp64", 4 * 60)
    if w.cfg == "1b":
        # measured, not estimated (profiles/r01_split_ncu.md, cfg 1b): 275 instructions of all pipes
        # per element and stage, 72 of them on the FP64 pipe (sincos, scan, window sums, RK4) -- the
        # batch is bound by instruction issue (74 % of the slots), the FP64 pipe is 39 % busy
        return ("issue", 4 * 275)
    return ("fp64", 4 * (110 + 2 * 2 * w.radius))


def ceiling(w, pk=None):
    """Per-config roofline ceiling in oscillator-steps/s = 1/max(T_hbm, T_alu) and its parts."""
    pk = pk or peaks()
    t_hbm = bytes_per_osc_step(w) / (pk["hbm_gbs"] * 1e9)
    pipe, ops = ops_per_osc_step(w)
    t_alu = ops / (pk[pipe + "_ginstr_s"] * 1e9)
    bound = "hbm" if t_hbm >= t_alu else "alu"
    return dict(bound=bound, osc_steps_per_s=1.0 / max(t_hbm, t_alu), t_hbm=t_hbm, t_alu=t_alu,
                pipe=pipe, ops=ops, bytes=bytes_per_osc_step(w))
