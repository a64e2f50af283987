"""CPU oracle for the GAME hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes/numpy view of ``oracle/game_oracle.c`` (plain C, fp64 fitness,
bit-defined GA operators).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package; the CUDA path (``paper_1211_5481_b200``) never does and shares no code
with it.  See the header of ``game_oracle.c`` for citations and pins.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "game_oracle.c")
_LIB = os.path.join(_HERE, "libgame_oracle.so")

EXP_CHEBYSHEV, EXP_TRIG = 0, 1
SEL_TOURNAMENT, SEL_RANKING, SEL_ROULETTE = 0, 1, 2
ACT_IDENTITY, ACT_SIGMOID, ACT_TANH = 0, 1, 2


def family(expansion: int, activation: int, shared: bool = False) -> int:
    """shared = the paper's literal form: one coefficient per degree for ALL features (eq.(2))."""
    return expansion | (activation << 8) | (int(shared) << 16)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC",
               "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        f32p, f64p, u32p = C.POINTER(C.c_float), C.POINTER(C.c_double), C.POINTER(C.c_uint32)
        L = _lib
        L.oracle_num_genes.restype = C.c_int
        L.oracle_num_genes.argtypes = [C.c_int, C.c_int, C.c_int]
        L.oracle_paper_shapes.restype = None
        L.oracle_paper_shapes.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.oracle_expand.restype = None
        L.oracle_expand.argtypes = [C.c_int, C.c_int, C.c_int, f32p, f64p]
        L.oracle_output.restype = C.c_double
        L.oracle_output.argtypes = [C.c_int, C.c_int, C.c_int, f32p, f32p]
        L.oracle_eval_fitness.restype = C.c_int
        L.oracle_eval_fitness.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, f32p, f32p, f32p, f64p, f64p]
        L.oracle_philox4x32_10.restype = None
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_index.restype = C.c_uint32
        L.oracle_index.argtypes = [C.c_uint32, C.c_uint32]
        L.oracle_bernoulli_threshold.restype = C.c_uint64
        L.oracle_bernoulli_threshold.argtypes = [C.c_double]
        L.oracle_neg2ln_u1.restype = C.c_float
        L.oracle_neg2ln_u1.argtypes = [C.c_uint32]
        L.oracle_cos_angle.restype = C.c_float
        L.oracle_cos_angle.argtypes = [C.c_uint32]
        L.oracle_gauss.restype = C.c_float
        L.oracle_gauss.argtypes = [C.c_uint32, C.c_uint32]
        for name in ("oracle_neg2ln_u1_many", "oracle_cos_angle_many"):
            getattr(L, name).restype = None
            getattr(L, name).argtypes = [C.c_int64, u32p, f32p]
        L.oracle_gauss_many.restype = None
        L.oracle_gauss_many.argtypes = [C.c_int64, u32p, u32p, f32p]
        L.oracle_init_population.restype = None
        L.oracle_init_population.argtypes = [C.c_int, C.c_int, C.c_uint64, f32p]
        L.oracle_best_index.restype = C.c_int
        L.oracle_best_index.argtypes = [C.c_int, f32p]
        L.oracle_step.restype = C.c_int
        L.oracle_step.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_float,
                                  C.c_uint64, C.c_uint32, f32p, f32p, f32p]
        L.oracle_roulette_weight.restype = C.c_uint64
        L.oracle_roulette_weight.argtypes = [C.c_float]
        L.oracle_rank_from_word.restype = C.c_int
        L.oracle_rank_from_word.argtypes = [C.c_uint32, C.c_int]
        L.oracle_roulette_from_word.restype = C.c_int
        L.oracle_roulette_from_word.argtypes = [C.c_uint32, C.c_int, C.POINTER(C.c_uint64)]
        L.oracle_step_sel.restype = C.c_int
        L.oracle_step_sel.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_float,
                                      C.c_uint64, C.c_uint32, f32p, f32p, f32p]
        L.oracle_eval_rmse.restype = C.c_int
        L.oracle_eval_rmse.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, f32p, f32p, f32p, f64p]
        L.oracle_immigrate.restype = C.c_int
        L.oracle_immigrate.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint64, C.c_uint32, f32p]
        L.oracle_run_until.restype = C.c_int
        L.oracle_run_until.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, f32p, f32p,
                                       C.c_int, C.c_int, C.c_double, C.c_double, C.c_float,
                                       C.c_uint64, C.c_uint32, C.c_uint32, C.c_float, f32p, f32p, f32p, u32p]
        L.oracle_predict.restype = None
        L.oracle_predict.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, f32p, f32p, f64p]
        L.oracle_confusion.restype = None
        L.oracle_confusion.argtypes = [C.c_int64, f64p, f32p, C.c_double, C.POINTER(C.c_int64)]
        L.oracle_run.restype = C.c_int
        L.oracle_run.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, f32p, f32p,
                                 C.c_int, C.c_int, C.c_double, C.c_double, C.c_float,
                                 C.c_uint64, C.c_uint32, C.c_uint32, f32p, f32p, f32p]
    return _lib


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _p(a: np.ndarray, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def num_genes(N: int, d: int, fam: int) -> int:
    return lib().oracle_num_genes(N, d, fam)


def paper_shapes(N: int, d: int, B: int):
    nc, ng = C.c_int(), C.c_int()
    lib().oracle_paper_shapes(N, d, B, C.byref(nc), C.byref(ng))
    return nc.value, ng.value


def expand(N: int, d: int, fam: int, x) -> np.ndarray:
    x = _f32(x)
    assert x.shape == (N,)
    phi = np.empty(num_genes(N, d, fam), dtype=np.float64)
    lib().oracle_expand(N, d, fam, _p(x, C.c_float), _p(phi, C.c_double))
    return phi


def output(N: int, d: int, fam: int, x, w) -> float:
    x, w = _f32(x), _f32(w)
    assert w.shape == (num_genes(N, d, fam),)
    return lib().oracle_output(N, d, fam, _p(x, C.c_float), _p(w, C.c_float))


def eval_fitness(d: int, fam: int, X, t, W, return_sse: bool = False):
    """F[m] (float64) of population W [M,G] on knowledge base X [P,N], t [P]."""
    X, t, W = _f32(X), _f32(t), _f32(W)
    P, N = X.shape
    M, G = W.shape
    assert t.shape == (P,) and G == num_genes(N, d, fam), (t.shape, G)
    F = np.empty(M, dtype=np.float64)
    S = np.empty(M, dtype=np.float64)
    rc = lib().oracle_eval_fitness(P, N, d, M, fam, _p(X, C.c_float), _p(t, C.c_float),
                                   _p(W, C.c_float), _p(F, C.c_double), _p(S, C.c_double))
    if rc:
        raise ValueError(f"oracle_eval_fitness failed: {rc}")
    return (F, S) if return_sse else F


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    assert c.shape == (4,) and k.shape == (2,)
    out = np.empty(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def index(w: int, n: int) -> int:
    return lib().oracle_index(w, n)


def bernoulli_threshold(p: float) -> int:
    return lib().oracle_bernoulli_threshold(p)


def neg2ln_u1(a: int) -> np.float32:
    return np.float32(lib().oracle_neg2ln_u1(a))


def cos_angle(b: int) -> np.float32:
    return np.float32(lib().oracle_cos_angle(b))


def gauss(a: int, b: int) -> np.float32:
    return np.float32(lib().oracle_gauss(a, b))


def _u32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.uint32)


def neg2ln_u1_many(a) -> np.ndarray:
    a = _u32(a)
    out = np.empty(a.shape, dtype=np.float32)
    lib().oracle_neg2ln_u1_many(a.size, _p(a, C.c_uint32), _p(out, C.c_float))
    return out


def cos_angle_many(b) -> np.ndarray:
    b = _u32(b)
    out = np.empty(b.shape, dtype=np.float32)
    lib().oracle_cos_angle_many(b.size, _p(b, C.c_uint32), _p(out, C.c_float))
    return out


def gauss_many(a, b) -> np.ndarray:
    a, b = _u32(a), _u32(b)
    assert a.shape == b.shape
    out = np.empty(a.shape, dtype=np.float32)
    lib().oracle_gauss_many(a.size, _p(a, C.c_uint32), _p(b, C.c_uint32), _p(out, C.c_float))
    return out


def init_population(M: int, G: int, seed: int) -> np.ndarray:
    W = np.empty((M, G), dtype=np.float32)
    lib().oracle_init_population(M, G, seed, _p(W, C.c_float))
    return W


def best_index(F) -> int:
    F = _f32(F)
    return lib().oracle_best_index(F.shape[0], _p(F, C.c_float))


def step(W, F, E: int, k: int, p_cross: float, p_mut: float, sigma: float, seed: int, gen: int) -> np.ndarray:
    W, F = _f32(W), _f32(F)
    M, G = W.shape
    assert F.shape == (M,)
    Wn = np.empty_like(W)
    rc = lib().oracle_step(M, G, E, k, p_cross, p_mut, sigma, seed, gen,
                           _p(W, C.c_float), _p(F, C.c_float), _p(Wn, C.c_float))
    if rc:
        raise ValueError(f"oracle_step failed: {rc}")
    return Wn


def run(d: int, fam: int, X, t, W, E: int, k: int, p_cross: float, p_mut: float, sigma: float,
        seed: int, gen0: int, n_gens: int):
    """Returns (final population, final fitness f32, best[0..n_gens])."""
    X, t = _f32(X), _f32(t)
    W = _f32(W).copy()
    P, N = X.shape
    M, G = W.shape
    assert G == num_genes(N, d, fam)
    F = np.empty(M, dtype=np.float32)
    best = np.empty(n_gens + 1, dtype=np.float32)
    rc = lib().oracle_run(P, N, d, M, fam, _p(X, C.c_float), _p(t, C.c_float), E, k, p_cross, p_mut,
                          sigma, seed, gen0, n_gens, _p(W, C.c_float), _p(F, C.c_float), _p(best, C.c_float))
    if rc:
        raise ValueError(f"oracle_run failed: {rc}")
    return W, F, best


def predict(d: int, fam: int, X, w) -> np.ndarray:
    """y[q] = act(w . phi(x_q)) in float64 for one chromosome (test / validation use case)."""
    X, w = _f32(X), _f32(w)
    Q, N = X.shape
    assert w.shape == (num_genes(N, d, fam),)
    y = np.empty(Q, dtype=np.float64)
    lib().oracle_predict(Q, N, d, fam, _p(X, C.c_float), _p(w, C.c_float), _p(y, C.c_double))
    return y


def confusion(y, t, threshold: float = 0.5):
    """(TP, FP, TN, FN) of the thresholded outputs against 0/1 targets."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    t = _f32(t)
    assert y.shape == t.shape
    counts = (C.c_int64 * 4)()
    lib().oracle_confusion(y.size, _p(y, C.c_double), _p(t, C.c_float), threshold, counts)
    return tuple(int(c) for c in counts)


def run_until(d: int, fam: int, X, t, W, E: int, k: int, p_cross: float, p_mut: float, sigma: float,
              seed: int, gen0: int, max_gens: int, threshold: float):
    """Run with the stop rule. Returns (final population, final fitness f32, best[0..done], done)."""
    X, t = _f32(X), _f32(t)
    W = _f32(W).copy()
    P, N = X.shape
    M, G = W.shape
    F = np.empty(M, dtype=np.float32)
    best = np.full(max_gens + 1, np.nan, dtype=np.float32)
    done = C.c_uint32()
    rc = lib().oracle_run_until(P, N, d, M, fam, _p(X, C.c_float), _p(t, C.c_float), E, k, p_cross, p_mut, sigma,
                                seed, gen0, max_gens, threshold, _p(W, C.c_float), _p(F, C.c_float),
                                _p(best, C.c_float), C.byref(done))
    if rc:
        raise ValueError(f"oracle_run_until failed: {rc}")
    return W, F, best[:done.value + 1], done.value


def roulette_weight(f: float) -> int:
    return lib().oracle_roulette_weight(float(f))


def rank_from_word(w: int, M: int) -> int:
    return lib().oracle_rank_from_word(w, M)


def roulette_from_word(w: int, weights) -> int:
    wt = np.ascontiguousarray(weights, dtype=np.uint64)
    return lib().oracle_roulette_from_word(w, wt.size, _p(wt, C.c_uint64))


def step_sel(W, F, E: int, k: int, selection: int, p_cross: float, p_mut: float, sigma: float, seed: int, gen: int):
    """One generation with tournament (0), ranking (1) or roulette (2) selection (reading R10)."""
    W, F = _f32(W), _f32(F)
    M, G = W.shape
    Wn = np.empty_like(W)
    rc = lib().oracle_step_sel(M, G, E, k, selection, p_cross, p_mut, sigma, seed, gen,
                               _p(W, C.c_float), _p(F, C.c_float), _p(Wn, C.c_float))
    if rc:
        raise ValueError(f"oracle_step_sel failed: {rc}")
    return Wn


def immigrate(Wn, E: int, R: int, seed: int, gen: int) -> np.ndarray:
    """Overwrite the last R child slots of a stepped population with fresh random chromosomes (R12)."""
    Wn = _f32(Wn).copy()
    M, G = Wn.shape
    rc = lib().oracle_immigrate(M, G, E, R, seed, gen, _p(Wn, C.c_float))
    if rc:
        raise ValueError(f"oracle_immigrate failed: {rc}")
    return Wn


def eval_rmse(d: int, fam: int, X, t, W) -> np.ndarray:
    """Root-mean-square error per chromosome."""
    X, t, W = _f32(X), _f32(t), _f32(W)
    P, N = X.shape
    M, G = W.shape
    F = np.empty(M, dtype=np.float64)
    rc = lib().oracle_eval_rmse(P, N, d, M, fam, _p(X, C.c_float), _p(t, C.c_float), _p(W, C.c_float), _p(F, C.c_double))
    if rc:
        raise ValueError(f"oracle_eval_rmse failed: {rc}")
    return F
