"""The five north-star workloads of BASELINE.json (``configs``), as plain data.

``get(cfg_id)`` returns the full-size description; ``get(cfg_id, n1=...)`` or
``n=...`` returns the same workload on a smaller lattice / ring / graph (same
model, parameters, radius rule and step) for parity tests and CPU samples.
No arithmetic of the method lives here.
"""
import math
from dataclasses import dataclass, field, replace

KS, FHN, HH, KSI, FHN2, HHS = 0, 1, 2, 3, 4, 5
RING, LATTICE, CSR, RANDOM_INDEGREE = 0, 1, 2, 3


@dataclass(frozen=True)
class Workload:
    cfg: str
    name: str
    model: int
    topo: int
    n: int
    dtype: str                      # "f32" | "f64"
    dt: float
    n_steps: int
    obs_every: int
    params: dict
    extent: tuple = ()              # lattice edge lengths (x fastest)
    radius: int = 0                 # ring: P neighbours each side; lattice: Euclidean radius
    in_degree: int = 0              # RANDOM_INDEGREE
    topo_seed: int = 1
    batch: int = 1                  # independent replicas integrated together (rings)
    extra: dict = field(default_factory=dict)

    @property
    def nvar(self):
        return {KS: 1, FHN: 2, HH: 4, KSI: 2, FHN2: 2, HHS: 5}[self.model]


_FHN2 = dict(eps=0.05, a=0.5, sigma=0.1, phi=math.pi / 2 - 0.1)
_FHN5 = dict(eps=0.05, a=0.5, sigma=0.2, phi=math.pi / 2 - 0.1)
_HH = dict(gNa=120.0, gK=36.0, gL=0.3, ENa=50.0, EK=-77.0, EL=-54.4, C=1.0,
           g_syn=0.1, E_syn=0.0, theta_syn=0.0, k_syn=2.0)


def get(cfg, n=None, n1=None, batch=None):
    cfg = str(cfg)
    if cfg == "1b":
        # extra, not a BASELINE.json config (SURVEY.md 8(d) iii): config 1 as a batch of independent
        # rings, one per CTA, 8 per SM -- where the FP64 pipe, not the latency of one tiny net, binds
        batch = batch or 148 * 8
        w = get("1", n=n)
        return replace(w, cfg="1b", name="KS ring N=%d P=64 f64 x %d independent nets" % (w.n, batch), batch=batch)
    if cfg == "1":
        n = n or 256
        return Workload("1", "KS ring N=%d P=64 f64" % n, KS, RING, n, "f64", 0.025, 1000, 1,
                        dict(K=1.0, alpha=math.pi / 2 - 0.05, omega0=0.0), radius=64)
    if cfg in ("6", "6b", "6c"):
        # extra, not a BASELINE.json config: the paper's own performance model (PAPER.md:327, :337-343,
        # Fig. 6c): Kuramoto-Sakaguchi with inertia on a 3D ball, m = 1, eps = 0.05, mu = 0.01,
        # alpha = 0.45, N1 = 100, at its three radii P = 2 / 4 / 6 (cfg 6 / 6b / 6c); K = mu * Omega with
        # Omega = 32 / 256 / 924 links, self link excluded (reading R4)
        n1 = n1 or 100
        P, deg = {"6": (2, 32), "6b": (4, 256), "6c": (6, 924)}[cfg]
        return Workload(cfg, "KS with inertia 3D %d^3 radius %d f64" % (n1, P), KSI, LATTICE, n1 ** 3, "f64",
                        0.05, 200, 10, dict(K=0.01 * deg, alpha=0.45, m=1.0, eps=0.05, omega0=0.0),
                        extent=(n1, n1, n1), radius=P)
    if cfg == "2":
        n = n or 65536
        R = int(math.floor(0.35 * n))          # reading R5
        return Workload("2", "FHN ring N=%d R=%d f64" % (n, R), FHN, RING, n, "f64", 0.01, 2000,
                        10, dict(_FHN2), radius=R)
    if cfg in ("3a", "3b", "3"):
        n1 = n1 or 200
        dt = "f64" if cfg == "3b" else "f32"
        return Workload("3b" if dt == "f64" else "3a",
                        "KS 3D %d^3 radius 4 %s" % (n1, dt), KS, LATTICE, n1 ** 3, dt, 0.05, 500,
                        10, dict(K=1.0, alpha=math.pi / 2 - 0.1, omega0=0.0),
                        extent=(n1, n1, n1), radius=4,
                        extra=dict(omega="lorentzian", gamma=0.01, omega_max=1.0))
    if cfg == "4":
        n = n or 1_000_000
        return Workload("4", "HH random CSR N=%d k=100 f64" % n, HH, RANDOM_INDEGREE, n, "f64",
                        0.01, 10000, 100, dict(_HH), in_degree=min(100, max(1, n - 1)))
    if cfg == "5":
        n1 = n1 or 464
        return Workload("5", "FHN 3D %d^3 radius 2 f32" % n1, FHN, LATTICE, n1 ** 3, "f32", 0.01,
                        200, 10, dict(_FHN5), extent=(n1, n1, n1), radius=2)
    raise KeyError(cfg)


ALL = ("1", "2", "3a", "3b", "4", "5")


def with_steps(w, n_steps, obs_every=None):
    return replace(w, n_steps=n_steps, obs_every=obs_every or w.obs_every)
