#!/usr/bin/env python
"""Writes tests/golden/stats_cfg<id>_seed<seed>.json: the long-run statistics of reading R9
 of a BASELINE.json config AT FULL SIZE, computed by the CPU oracle alone.

    python tests/golden/make_stats_cache.py --cfg 3b [--steps 100] [--seed 1] [--threads 8]

Calls only oracle/ and the seeded input generators (paper_2410_19075_b200/inputs.py, configs.py --
plain data and random draws, none of the method's arithmetic).  It never loads the CUDA library.

SURVEY.md 8(c): "the full-length statistics run of the oracle is computed once and cached on disk
keyed by (config, seed); if the box has too few cores, the long-run oracle may switch to its own
independently written factorised/prefix neighbour sum after that variant has been shown equal to
the direct sum to 1e-13 (A11 norm) on a full-size single RHS -- say so in the report when used".
That is what --variant fast does (default for every config but 1): before the run it evaluates ONE
right-hand side at full size with both forms, refuses to continue if they differ by more than
1e-13, and stores the discrepancy it saw.  --steps shortens the run where the full length does not
fit the CPU budget of the build box; the file records both the length that was run and the
config's own, and the GPU test (tests/test_gpu_stats_cache.py) integrates exactly the recorded
length.  Nothing is shrunk silently.
"""
import argparse
import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg", required=True, choices=["1", "2", "3a", "3b", "4", "5"])
    ap.add_argument("--steps", type=int, default=0, help="RK4 steps to run (0 = the config's own length)")
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--variant", default=None, choices=["direct", "fast"])
    args = ap.parse_args()
    if args.threads:
        os.environ["OMP_NUM_THREADS"] = str(args.threads)

    import numpy as np
    import harness as H                      # make_inputs / make_oracle: oracle + generators only
    from oracle import oracle as ora
    from paper_2410_19075_b200 import configs

    w = configs.get(args.cfg)
    n_steps = args.steps or w.n_steps
    assert n_steps % w.obs_every == 0
    variant = args.variant or ("direct" if args.cfg == "1" else "fast")
    t0 = time.time()
    inp = H.make_inputs(w, seed=args.seed)
    net = H.make_oracle(w, inp)
    if w.topo == configs.RING:
        net.ring_P = w.radius
    t_build = time.time() - t0
    check = None
    if variant == "fast":
        t1 = time.time()
        fd, ff = net.rhs(inp["y0"]), net.rhs_fast(inp["y0"])
        check = max(float(np.abs(ff[v] - fd[v]).max() / np.abs(fd[v]).max()) for v in range(fd.shape[0])
                    if np.abs(fd[v]).max() > 0)
        print("fast vs direct, one full-size RHS: %.3e (%.1f s)" % (check, time.time() - t1), flush=True)
        if not check <= 1e-13:
            raise SystemExit("the accelerated variant differs from the direct sum by %.3e > 1e-13" % check)
        del fd, ff
    t1 = time.time()
    st = net.run_statistics(inp["y0"], n_steps, w.dt, w.obs_every, fast=(variant == "fast"))
    wall = time.time() - t1
    out = {
        "cfg": w.cfg, "workload": w.name, "n": w.n, "dtype_of_initial_state": w.dtype, "seed": args.seed,
        "dt": w.dt, "obs_every": w.obs_every, "n_steps": n_steps, "n_steps_of_config": w.n_steps,
        "full_length": n_steps == w.n_steps,
        "oracle_variant": variant,
        "fast_vs_direct_full_size_rhs": check,
        "stats": {k: st[k] for k in ("R_mean", "R_std", "Rloc_mean", "vel_mean", "vel_std", "n_samples")},
        "vel_sample": {"index": [0, w.n // 3, w.n // 2, w.n - 1],
                       "value": [float(st["vel"][i]) for i in (0, w.n // 3, w.n // 2, w.n - 1)]},
        "written_by": "tests/golden/make_stats_cache.py (oracle only)",
        "threads": ora.omp_threads(), "build_s": round(t_build, 1), "run_s": round(wall, 1),
    }
    path = os.path.join(HERE, "stats_cfg%s_seed%d.json" % (w.cfg, args.seed))
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print(json.dumps(out["stats"]), "->", path, "(%.0f s)" % wall)


if __name__ == "__main__":
    main()
