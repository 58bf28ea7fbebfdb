"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot run the full nets, so it computes SAMPLED outputs one by one:
  * single RHS at sampled rows (corners, edges, random interior): only those rows get their
    neighbour lists in the oracle (harness.make_oracle(rows=...));
  * lattices: the state after s RK4 steps at a sampled site depends only on the initial values
    within distance 4 s P of it (four stages per step, coupling radius P), so the oracle
    integrates the periodic sub-box of edge 2 * 4 s P + 1 cut out around the site -- the wrap of
    the small box touches only stage values the centre never uses -- and the centre must agree.
Tolerances are the north star's (harness.TOL_*).
"""
from dataclasses import replace

import numpy as np
import pytest

import harness as H
from paper_2410_19075_b200 import configs

pytestmark = pytest.mark.gpu


def sample_rows(w, rng, k=48):
    fixed = [0, 1, w.n - 1, w.n // 2]
    if w.topo == configs.LATTICE:
        nx, ny, nz = w.extent
        idx = lambda x, y, z: (z * ny + y) * nx + x
        fixed += [idx(nx - 1, 0, 0), idx(0, ny - 1, 0), idx(0, 0, nz - 1), idx(nx - 1, ny - 1, nz - 1),
                  idx(nx // 2, ny - 1, nz // 2), idx(1, 2, 3), idx(nx - 2, ny - 3, nz - 4)]
    return np.unique(np.concatenate([fixed, rng.integers(0, w.n, k)])).astype(np.int64)


@pytest.mark.parametrize("cfg", ["2", "3a", "3b", "4", "5"])
def test_full_size_rhs_sampled(cfg):
    w = configs.get(cfg)
    inp = H.make_inputs(w, seed=1)
    rows = sample_rows(w, np.random.default_rng(int(cfg[0])))
    net = H.make_gpu(w, inp)
    got = net.eval_rhs()
    assert np.isfinite(got).all()
    net.close()
    ref = H.make_oracle(w, inp, rows=rows).rhs(inp["y0"])
    # the norm of reading R11, its denominator taken over the sampled rows
    assert H.rel_maxnorm(got[:, rows], ref[:, rows], H.rhs_floor(w)) <= H.TOL_RHS[w.dtype]


def sub_box(w, arr, centre, half):
    """Values of a per-site array on the periodic cube of edge 2*half+1 around `centre`."""
    nx, ny, nz = w.extent
    cx, cy, cz = centre
    xs = (np.arange(-half, half + 1) + cx) % nx
    ys = (np.arange(-half, half + 1) + cy) % ny
    zs = (np.arange(-half, half + 1) + cz) % nz
    a = arr.reshape(arr.shape[:-1] + (nz, ny, nx))
    return np.ascontiguousarray(a[..., zs[:, None, None], ys[None, :, None], xs[None, None, :]]).reshape(arr.shape[:-1] + (-1,))


@pytest.mark.parametrize("cfg,steps", [("5", 2), ("3a", 1), ("3b", 1)])
def test_full_size_lattice_steps_sampled_sites(cfg, steps):
    w = configs.get(cfg)
    inp = H.make_inputs(w, seed=1)
    net = H.make_gpu(w, inp)
    net.integrate(steps, w.dt)
    got = net.get_state()
    net.close()
    nx, ny, nz = w.extent
    half = 4 * steps * w.radius
    edge = 2 * half + 1
    wb = replace(w, extent=(edge, edge, edge), n=edge ** 3, name=w.name + " sub-box")
    rng = np.random.default_rng(7)
    centres = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (nx // 2, 0, nz - 1), (3, ny - 2, nz // 2)]
    centres += [tuple(int(v) for v in rng.integers(0, nx, 3)) for _ in range(4)]
    mid = (half * edge + half) * edge + half
    worst = 0.0
    for c in centres:
        sub = dict(y0=sub_box(w, inp["y0"], c, half),
                   elem=None if inp["elem"] is None else sub_box(w, inp["elem"], c, half))
        ref = H.make_oracle(wb, sub).rk4(sub["y0"], steps, w.dt)
        i = (c[2] * ny + c[1]) * nx + c[0]
        worst = max(worst, H.traj_err(w, got[:, i:i + 1], ref[:, mid:mid + 1]))
    assert worst <= H.TOL_TRAJ[w.dtype]
