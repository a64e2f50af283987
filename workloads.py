"""Seeded synthetic inputs for the GAME hot path (shared by tests, bench and smoke).

This module only *makes inputs*: knowledge bases (X, t) shaped like BASELINE.json's
five configurations, which stand in for the paper's NGC1399 globular-cluster catalogue
(PAPER.md:120-122 -- not available here).  It holds none of the method's code: it does not
import ``oracle`` or ``paper_1211_5481_b200`` and neither imports anything from the other.
The labels need a hidden chromosome applied to an expansion of the features; that is part
of the *data recipe* in BASELINE.json and is evaluated with numpy library routines
(``numpy.polynomial.chebyshev.chebvander``, ``numpy.cos/sin``) in float64.

Recipe: ``numpy.random.Generator(numpy.random.Philox(seed))``,
seed = config index unless given; X ~ U[-1,1) (c0,c1,c3,c4) or U[-pi,pi) (c2) cast to
float32; hidden w* ~ N(0,1) (c2: N(0,0.3^2)); classification label =
1[sigmoid(w*.phi(x)) + N(0,0.05^2) > 0.5] as 0.0/1.0 float32; c2 target =
tanh(w*.phi(x)) + N(0,0.01^2) as float32.  phi is evaluated on the float32-rounded X.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

EXP_CHEBYSHEV, EXP_TRIG = 0, 1
ACT_IDENTITY, ACT_SIGMOID, ACT_TANH = 0, 1, 2


@dataclass(frozen=True)
class Config:
    name: str
    P: int
    N: int
    d: int                 # Chebyshev degree or number of harmonics K (trig)
    M: int
    expansion: int
    activation: int
    elite: int
    tournament: int
    p_cross: float
    p_mut: float
    sigma: float
    generations: int
    x_range: float         # X ~ U[-x_range, x_range)
    w_star_std: float
    noise_std: float
    seed: int
    shared: bool = False   # the paper's literal form: one coefficient per degree for all features (eq.(2))

    @property
    def family(self) -> int:
        return self.expansion | (self.activation << 8) | (int(self.shared) << 16)

    @property
    def G(self) -> int:
        return (1 if self.shared else self.N) * self.d * (2 if self.expansion == EXP_TRIG else 1) + 1


# BASELINE.json configs[0..3]; configs[4] is the (M,P) sweep built by c4().
CONFIGS = {
    "c0": Config("c0", 1_000, 4, 3, 64, EXP_CHEBYSHEV, ACT_SIGMOID, 2, 3, 0.9, 0.05, 0.1, 10, 1.0, 1.0, 0.05, 0),
    "c1": Config("c1", 100_000, 10, 6, 512, EXP_CHEBYSHEV, ACT_SIGMOID, 4, 3, 0.9, 0.05, 0.1, 100, 1.0, 1.0, 0.05, 1),
    "c2": Config("c2", 1_000_000, 16, 4, 1024, EXP_TRIG, ACT_TANH, 8, 4, 0.9, 0.02, 0.05, 50, float(np.pi), 0.3, 0.01, 2),
    "c3": Config("c3", 4_000_000, 32, 10, 4096, EXP_CHEBYSHEV, ACT_SIGMOID, 4, 3, 0.9, 0.05, 0.1, 20, 1.0, 1.0, 0.05, 3),
}

# The paper's own experiment shape, as a synthetic stand-in: 2100 patterns x 9 feature
# columns, polytrigo degree 8, B*N+1 = 19 chromosomes (eq.(4)), crossover 0.9, mutation 0.2, elitism 2,
# ranking selection, MSE threshold 0.001, thousands of iterations: the latency-bound regime.  Per-feature coefficients (D1).
PAPER_SHAPE = Config("n1", 2_100, 9, 8, 19, EXP_TRIG, ACT_SIGMOID, 2, 3, 0.9, 0.2, 0.1, 10_000, float(np.pi), 0.3, 0.05, 11)

# the same with the paper's shared coefficients: G = 2 * 8 + 1 = 17 genes (eq.(5))
PAPER_SHAPE_SHARED = replace(PAPER_SHAPE, name="n1s", shared=True, w_star_std=0.1)

C4_M = (256, 1024, 4096, 16384)
C4_P = (100_000, 1_000_000, 10_000_000)


def c4(M: int, P: int) -> Config:
    """One point of the fitness-kernel sweep (BASELINE.json configs[4]); no GA step."""
    return Config(f"c4_M{M}_P{P}", P, 20, 6, M, EXP_CHEBYSHEV, ACT_SIGMOID, 0, 1, 0.0, 0.0, 0.0, 0,
                  1.0, 1.0, 0.05, 4)


def scaled(cfg: Config, **kw) -> Config:
    """Same recipe at another size (parity slices, smoke)."""
    return replace(cfg, **kw)


def _design_matrix(cfg: Config, X64: np.ndarray) -> np.ndarray:
    """[rows, G] expansion of the data recipe, gene order [bias | per-feature block]."""
    rows = X64.shape[0]
    if cfg.expansion == EXP_CHEBYSHEV:
        V = np.polynomial.chebyshev.chebvander(X64, cfg.d)[..., 1:]        # [rows, N, d]
        blocks = V.reshape(rows, cfg.N * cfg.d)
    else:
        k = np.arange(1, cfg.d + 1, dtype=np.float64)
        kx = X64[..., None] * k                                            # [rows, N, K]
        blocks = np.concatenate([np.cos(kx), np.sin(kx)], axis=-1).reshape(rows, cfg.N * 2 * cfg.d)
    if cfg.shared:   # shared coefficients: the term of gene j is the sum over the features
        blocks = blocks.reshape(rows, cfg.N, -1).sum(axis=1)
    return np.concatenate([np.ones((rows, 1)), blocks], axis=1)


def make_kb(cfg: Config, seed: int | None = None, chunk: int = 65536):
    """Returns (X float32 [P,N], t float32 [P], w_star float64 [G])."""
    rng = np.random.Generator(np.random.Philox(cfg.seed if seed is None else seed))
    w_star = rng.standard_normal(cfg.G) * cfg.w_star_std
    X = np.empty((cfg.P, cfg.N), dtype=np.float32)
    t = np.empty(cfg.P, dtype=np.float32)
    for p0 in range(0, cfg.P, chunk):
        p1 = min(cfg.P, p0 + chunk)
        xb = rng.uniform(-cfg.x_range, cfg.x_range, size=(p1 - p0, cfg.N)).astype(np.float32)
        noise = rng.standard_normal(p1 - p0) * cfg.noise_std
        z = _design_matrix(cfg, xb.astype(np.float64)) @ w_star
        if cfg.activation == ACT_TANH:
            tb = np.tanh(z) + noise
        elif cfg.activation == ACT_SIGMOID:
            tb = ((1.0 / (1.0 + np.exp(-z)) + noise) > 0.5).astype(np.float64)
        else:
            tb = z + noise
        X[p0:p1] = xb
        t[p0:p1] = tb.astype(np.float32)
    return X, t, w_star


def uniform_population(M: int, G: int, seed: int) -> np.ndarray:
    """Genes ~ U[-1,1) float32 from numpy -- for fitness-only cases (c4) and
    tests that want a population independent of the method's own Philox init."""
    rng = np.random.Generator(np.random.Philox(seed))
    return rng.uniform(-1.0, 1.0, size=(M, G)).astype(np.float32)


def shard_patterns(P: int, world_size: int, rank: int):
    """Contiguous pattern range [p0, p1) of rank `rank` (multi-GPU pattern sharding)."""
    base, rem = divmod(P, world_size)
    p0 = rank * base + min(rank, rem)
    return p0, p0 + base + (1 if rank < rem else 0)
