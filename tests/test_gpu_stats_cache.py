"""Long-run order-parameter statistics of the BASELINE.json configs AT FULL SIZE (north star:
"the long-run order-parameter statistics of each config must agree to 1e-3").

The expected values are tests/golden/stats_cfg<id>_seed1.json, written by
tests/golden/make_stats_cache.py from the CPU oracle alone (computed once, cached on
disk keyed by (config, seed)).  Each file records the length that was run (the config's own where
the build box could afford it, shorter otherwise -- `full_length` says which) and the oracle variant
used; the GPU integrates exactly that length through net_integrate_observed.

Tolerance 1e-3 * max(1, |ref|): absolute for the order parameters (they live in [0, 1]) and for
velocities below 1, relative above.
"""
import glob
import json
import os

import numpy as np
import pytest

import harness as H
from paper_2410_19075_b200 import binding as B, configs

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
FILES = sorted(glob.glob(os.path.join(GOLDEN, "stats_cfg*_seed*.json")))


def test_every_config_has_a_cache_file():
    have = {json.load(open(p))["cfg"] for p in FILES}
    assert have >= set(configs.ALL), "missing: %s" % (set(configs.ALL) - have)


@pytest.mark.parametrize("path", FILES, ids=[os.path.basename(p)[:-5] for p in FILES])
def test_full_size_long_run_statistics(path):
    ref = json.load(open(path))
    w = configs.get(ref["cfg"])
    assert w.n == ref["n"] and w.dt == ref["dt"] and w.obs_every == ref["obs_every"]
    if ref["oracle_variant"] == "fast":
        assert ref["fast_vs_direct_full_size_rhs"] <= 1e-13
    inp = H.make_inputs(w, seed=ref["seed"])
    net = H.make_gpu(w, inp)
    got = net.integrate_observed(ref["n_steps"], w.dt, w.obs_every)
    assert got["n_samples"] == ref["stats"]["n_samples"]
    for k in ("R_mean", "R_std", "Rloc_mean", "vel_mean", "vel_std"):
        r = ref["stats"][k]
        assert abs(got[k] - r) <= H.TOL_STATS * max(1.0, abs(r)), (k, got[k], r)
    vel = net.observable(B.OBS_MEAN_PHASE_VELOCITY)
    idx = np.array(ref["vel_sample"]["index"])
    tol = 1e-6 if w.dtype == "f64" else 5e-2
    assert np.abs(vel[idx] - np.array(ref["vel_sample"]["value"])).max() <= tol
    net.close()
