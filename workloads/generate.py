"""Input recipes (readings R11, R13-R15).

Synthetic stand-ins for the paper's DALIA models and datasets, which
are not available: regular g x g grids replace the FEM meshes, iid N(0,1) `y` replaces
the measurements.  Shapes follow BASELINE.json `configs[0..4]`.

Random numbers come from a counter-based generator (splitmix64 finaliser applied to
`stream_key + index`), so any element can be regenerated independently and the arrays
are bit-identical on every platform.  Normals use Box-Muller on two independent
uniform streams.  Nothing here knows about precision matrices.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

_U64 = np.uint64
_GOLD = _U64(0x9E3779B97F4A7C15)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 output function on an array of uint64 counters (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (x + _GOLD).astype(_U64)
        z = (z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)
        z = z ^ (z >> _U64(31))
    return z


def _stream_key(seed: int, stream: int) -> np.uint64:
    k = np.array([(seed * 4 + stream) & 0xFFFFFFFFFFFFFFFF], dtype=_U64)
    return _splitmix64(_splitmix64(k))[0]


def uniforms(seed: int, stream: int, n: int) -> np.ndarray:
    """n doubles in [0,1): (u >> 11) * 2^-53 of the counter-based stream (seed, stream)."""
    idx = np.arange(n, dtype=_U64)
    with np.errstate(over="ignore"):
        ctr = (idx * _GOLD + _stream_key(seed, stream)).astype(_U64)
    bits = _splitmix64(ctr)
    return (bits >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normals(seed: int, stream: int, n: int) -> np.ndarray:
    """n iid N(0,1) by Box-Muller: streams `stream` (radius) and `stream+16` (angle)."""
    u1 = uniforms(seed, stream, n)
    u2 = uniforms(seed, stream + 16, n)
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)


@dataclass(frozen=True)
class Model:
    """Shape descriptor of one synthetic spatio-temporal model (no numerical content)."""

    g: int            # grid side; ns = g*g spatial nodes
    k: int            # response variables (1 = univariate)
    nt: int           # time blocks (the paper's n)
    a: int            # arrow width = number of fixed effects (the paper's a, BASELINE's nb)
    h: float = 1.0    # grid spacing (reading R3)
    fixed_prec: float = 1e-3  # prior precision of the fixed effects (reading R5)

    @property
    def ns(self) -> int:
        return self.g * self.g

    @property
    def b(self) -> int:
        return self.k * self.ns

    @property
    def N(self) -> int:
        return self.nt * self.b + self.a

    @property
    def a_per_row(self) -> int:
        """Covariates per observation row: all `a` (univariate) or a/k (multivariate, R14)."""
        return self.a // self.k

    @property
    def d(self) -> int:
        """Hyperparameters: 3 per variable + k(k-1)/2 couplings + k noise precisions (R13)."""
        return 3 * self.k + self.k * (self.k - 1) // 2 + self.k


@dataclass
class Obs:
    """Gaussian observations y = A x + eps.  Row i of A has a 1 at latent
    (time[i], var[i], node[i]) and `cov[i, :]` in the fixed-effect columns
    var[i]*a_per_row .. var[i]*a_per_row + a_per_row - 1 (R14)."""

    var: np.ndarray    # int32 [m]
    node: np.ndarray   # int32 [m]
    time: np.ndarray   # int32 [m]
    cov: np.ndarray    # float64 [m, a_per_row]
    y: np.ndarray      # float64 [m]

    @property
    def m(self) -> int:
        return int(self.y.shape[0])


# name -> (Model, observations per variable, seed, fixed theta or None)
CONFIGS = {
    0: (Model(g=4, k=1, nt=6, a=2), 200, 1000, (0.1, -0.2, 0.3, 0.0)),
    1: (Model(g=20, k=1, nt=50, a=4), 20_000, 1001, None),
    2: (Model(g=48, k=1, nt=100, a=6), 200_000, 1002, None),
    3: (Model(g=32, k=3, nt=64, a=6), 50_000, 1003, None),
    4: (Model(g=64, k=1, nt=128, a=8), 1_000_000, 1004, None),
    # two stand-ins shaped like the extremes of the paper's model zoo (
    # not BASELINE.json configs): "WA1-like" = many time steps (b = 3072, nt = 512), "WA2-like" = very large
    # blocks (b = 12288, nt = 48; needs the carry store mode to fit 180 GB).  Both multivariate (k = 3, d = 15).
    5: (Model(g=32, k=3, nt=512, a=6), 400_000, 1005, None),
    6: (Model(g=64, k=3, nt=48, a=6), 300_000, 1006, None),
}
EXTREME_NAMES = {5: "WA1-like (long time axis)", 6: "WA2-like (large blocks)"}


def make_model(g: int, k: int, nt: int, a: int, h: float = 1.0, fixed_prec: float = 1e-3) -> Model:
    if a % k != 0:
        raise ValueError("a must be a multiple of k")
    return Model(g=g, k=k, nt=nt, a=a, h=h, fixed_prec=fixed_prec)


def draw_obs(model: Model, m_per_var: int, seed: int) -> Obs:
    """R11: sites uniform with replacement over ns*nt; covariates and y iid N(0,1)."""
    k, apr = model.k, model.a_per_row
    m = k * m_per_var
    site = np.floor(uniforms(seed, 0, m) * (model.ns * model.nt)).astype(np.int64)
    site = np.minimum(site, model.ns * model.nt - 1)
    var = np.repeat(np.arange(k, dtype=np.int32), m_per_var)
    cov = normals(seed, 1, m * apr).reshape(m, apr) if apr > 0 else np.zeros((m, 0))
    y = normals(seed, 2, m)
    return Obs(
        var=var,
        node=(site % model.ns).astype(np.int32),
        time=(site // model.ns).astype(np.int32),
        cov=np.ascontiguousarray(cov, dtype=np.float64),
        y=np.ascontiguousarray(y, dtype=np.float64),
    )


def draw_theta(model: Model, seed: int, sd: float = 0.3) -> np.ndarray:
    """theta ~ N(0, sd^2) on every component (BASELINE.json configs[1..4]; R15)."""
    return sd * normals(seed, 3, model.d)


def make_config(idx: int, nt: int | None = None, m_per_var: int | None = None):
    """-> (Model, Obs, theta) of BASELINE.json configs[idx].  `nt`/`m_per_var` override the
    size for bounded samples of the same workload (bench.py's cpu_baseline leg)."""
    model, mpv, seed, theta = CONFIGS[idx]
    if nt is not None:
        model = Model(g=model.g, k=model.k, nt=nt, a=model.a, h=model.h, fixed_prec=model.fixed_prec)
    if m_per_var is not None:
        mpv = m_per_var
    obs = draw_obs(model, mpv, seed)
    th = np.array(theta, dtype=np.float64) if theta is not None else draw_theta(model, seed)
    return model, obs, th


def make_w0():
    """Worked example W0: config-0 shapes, RNG-free observations."""
    model = CONFIGS[0][0]
    i = np.arange(200)
    pick = (37 * i + 11) % 96
    cov = np.stack([np.cos(0.7 * (i + 1) * (j + 1)) for j in range(2)], axis=1)
    y = np.sin(1.3 * (i + 1))
    obs = Obs(
        var=np.zeros(200, dtype=np.int32),
        node=(pick % 16).astype(np.int32),
        time=(pick // 16).astype(np.int32),
        cov=np.ascontiguousarray(cov, dtype=np.float64),
        y=np.ascontiguousarray(y, dtype=np.float64),
    )
    return model, obs, np.array([0.1, -0.2, 0.3, 0.0])


def uniform_design(model: Model, c: int = 1, seed: int = 7) -> Obs:
    """Pin P12: every (variable, node, time) observed exactly c times, zero covariates."""
    k, ns, nt = model.k, model.ns, model.nt
    var, node, time = np.meshgrid(np.arange(k), np.arange(ns), np.arange(nt), indexing="ij")
    var = np.tile(var.ravel(), c).astype(np.int32)
    node = np.tile(node.ravel(), c).astype(np.int32)
    time = np.tile(time.ravel(), c).astype(np.int32)
    m = var.shape[0]
    return Obs(var=var, node=node, time=time, cov=np.zeros((m, model.a_per_row)), y=normals(seed, 2, m))
