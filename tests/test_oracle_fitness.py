"""Pins of the oracle's expansion / output / fitness against things other than itself:
values the paper prints, closed forms, library routines, brute force, invariants.
CPU only (-m "not gpu")."""
import math
import os

import numpy as np
import pytest

import oracle
import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
CHEB, TRIG = oracle.EXP_CHEBYSHEV, oracle.EXP_TRIG
IDEN, SIGM, TANH = oracle.ACT_IDENTITY, oracle.ACT_SIGMOID, oracle.ACT_TANH
fam = oracle.family


def _kv(path):
    out = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        out[k] = v
    return out


# ---------------------------------------------------------------- shapes (paper / BASELINE)
def test_paper_worked_example_shapes():
    """N=11, d=3, B=2 -> 23 chromosomes x 7 genes."""
    g = _kv(os.path.join(GOLD, "paper_worked_example.txt"))
    nc, ng = oracle.paper_shapes(int(g["features"][0]), int(g["degree"][0]), int(g["B"][0]))
    assert nc == int(g["num_chromosomes"][0]) and ng == int(g["num_genes"][0])


def test_paper_gene_order_is_cos_block_then_sin_block():
    """PAPER.md:89 gene order [a0, a1..a3 (cos), b1..b3 (sin)]: with one feature and K=3 the
    oracle's per-feature layout must be exactly that."""
    g = _kv(os.path.join(GOLD, "paper_worked_example.txt"))
    assert g["gene_order"] == ["a0", "a1", "a2", "a3", "b1", "b2", "b3"]
    x = 0.7
    phi = oracle.expand(1, 3, fam(TRIG, IDEN), [x])
    xf = float(np.float32(x))
    expect = [1.0] + [math.cos(k * xf) for k in (1, 2, 3)] + [math.sin(k * xf) for k in (1, 2, 3)]
    np.testing.assert_allclose(phi, expect, rtol=0, atol=1e-15)


def test_baseline_gene_counts():
    for line in open(os.path.join(GOLD, "baseline_gene_counts.txt")):
        if line.startswith("#"):
            continue
        name, N, d, e, G = line.split()
        assert oracle.num_genes(int(N), int(d), fam(int(e), SIGM)) == int(G), name
    for name, cfg in wl.CONFIGS.items():
        assert oracle.num_genes(cfg.N, cfg.d, cfg.family) == cfg.G


def test_num_genes_rejects_bad_input():
    assert oracle.num_genes(0, 3, 0) < 0 and oracle.num_genes(3, 0, 0) < 0 and oracle.num_genes(3, 3, 7) < 0


# ---------------------------------------------------------------- Chebyshev closed forms
def test_chebyshev_cos_identity():
    """T_j(cos th) = cos(j th)  (north_star pin)."""
    d = 10
    for th in np.linspace(0.0, math.pi, 257):
        x = np.float32(math.cos(th))
        th_x = math.acos(float(x))            # angle of the float32-rounded argument
        phi = oracle.expand(1, d, fam(CHEB, IDEN), [x])
        expect = [1.0] + [math.cos(j * th_x) for j in range(1, d + 1)]
        # recurrence error grows ~ j^2 eps near the ends; 1e-12 is far above it and far
        # below any indexing / sign mistake
        np.testing.assert_allclose(phi, expect, rtol=0, atol=1e-12)


def test_chebyshev_special_values_and_explicit_polynomials():
    d = 7
    f = fam(CHEB, IDEN)
    np.testing.assert_array_equal(oracle.expand(1, d, f, [1.0]), np.ones(d + 1))
    np.testing.assert_array_equal(oracle.expand(1, d, f, [-1.0]), [1.0] + [(-1.0) ** j for j in range(1, d + 1)])
    np.testing.assert_array_equal(oracle.expand(1, d, f, [0.0])[1:5], [0.0, -1.0, 0.0, 1.0])
    for x in (0.3, -0.55, 0.999, 2.5):       # defined outside [-1,1] too (R2)
        xf = float(np.float32(x))
        phi = oracle.expand(1, 4, f, [x])
        expect = [1, xf, 2 * xf**2 - 1, 4 * xf**3 - 3 * xf, 8 * xf**4 - 8 * xf**2 + 1]
        np.testing.assert_allclose(phi, expect, rtol=1e-13, atol=1e-13)


def test_chebyshev_matches_numpy_chebvander_and_layout():
    """Library routine for the values + an independent statement of the gene layout
    g = 1 + i*d + (j-1)."""
    rng = np.random.default_rng(5)
    N, d = 5, 6
    x = rng.uniform(-1, 1, N).astype(np.float32)
    phi = oracle.expand(N, d, fam(CHEB, SIGM), x)
    V = np.polynomial.chebyshev.chebvander(x.astype(np.float64), d)    # [N, d+1]
    assert phi[0] == 1.0
    for i in range(N):
        for j in range(1, d + 1):
            assert abs(phi[1 + i * d + (j - 1)] - V[i, j]) < 1e-13, (i, j)


# ---------------------------------------------------------------- trig closed forms
def test_trig_special_values_and_layout():
    N, K = 3, 4
    f = fam(TRIG, TANH)
    phi0 = oracle.expand(N, K, f, [0.0] * N)
    expect0 = [1.0] + ([1.0] * K + [0.0] * K) * N
    np.testing.assert_array_equal(phi0, expect0)
    x = np.array([0.5, -1.25, 3.0], dtype=np.float32)
    phi = oracle.expand(N, K, f, x)
    for i in range(N):
        for k in range(1, K + 1):
            assert abs(phi[1 + i * 2 * K + (k - 1)] - math.cos(k * float(x[i]))) < 1e-15
            assert abs(phi[1 + i * 2 * K + K + (k - 1)] - math.sin(k * float(x[i]))) < 1e-15
    # half-period values: cos(k*pi) = (-1)^k up to the float32 rounding of pi
    xpi = np.float32(math.pi)
    ph = oracle.expand(1, K, f, [xpi])
    for k in range(1, K + 1):
        assert abs(ph[k] - (-1.0) ** k) < 1e-12
        assert abs(ph[K + k] - math.sin(k * float(xpi))) < 1e-15 and abs(ph[K + k]) < 1e-6


def test_trig_discrete_orthogonality():
    """mean_x cos(jx)cos(kx) = delta_jk/2, mean cos*sin = 0 on a uniform grid of 64 points."""
    K, n = 4, 64
    xs = (2 * math.pi * np.arange(n) / n - math.pi)
    Phi = np.stack([oracle.expand(1, K, fam(TRIG, IDEN), [x]) for x in xs])    # [n, 1+2K]
    gram = Phi.T @ Phi / n
    expect = np.diag([1.0] + [0.5] * (2 * K))
    # float32 rounding of the grid points perturbs the entries at the 1e-7 level
    np.testing.assert_allclose(gram, expect, rtol=0, atol=2e-6)


# ---------------------------------------------------------------- output, eq. (2)
def test_output_picks_single_gene_identity():
    """Out is linear in the genes (eq.(2)): a unit gene returns exactly phi_g."""
    N, d = 3, 4
    f = fam(CHEB, IDEN)
    x = np.array([0.25, -0.5, 0.75], dtype=np.float32)
    phi = oracle.expand(N, d, f, x)
    G = oracle.num_genes(N, d, f)
    for g in range(G):
        w = np.zeros(G, dtype=np.float32)
        w[g] = 1.0
        assert oracle.output(N, d, f, x, w) == phi[g]


def test_output_activations():
    N, d = 2, 2
    x = np.array([0.5, -0.25], dtype=np.float32)
    w = np.array([0.5, 1.0, -2.0, 0.25, 3.0], dtype=np.float32)
    # by hand: T1=x, T2=2x^2-1
    z = 0.5 + 1.0 * 0.5 + (-2.0) * (2 * 0.25 - 1) + 0.25 * (-0.25) + 3.0 * (2 * 0.0625 - 1)
    assert z == -0.6875
    assert oracle.output(N, d, fam(CHEB, IDEN), x, w) == z
    assert abs(oracle.output(N, d, fam(CHEB, SIGM), x, w) - 1 / (1 + math.exp(-z))) < 1e-16
    assert abs(oracle.output(N, d, fam(CHEB, TANH), x, w) - math.tanh(z)) < 1e-16


def test_shared_coefficient_model_from_precomputed_sums():
    """PAPER.md:54 eq.(2) shares a_j across features and PAPER.md:110 precomputes the per-pattern
    sums of sines and cosines.  Tying the genes across features in the per-feature layout must
    give a_0 + sum_j a_j C_j + sum_j b_j S_j with C_j = sum_i cos(j f_i), S_j = sum_i sin(j f_i)."""
    rng = np.random.default_rng(11)
    N, K, P = 11, 3, 40                       # the paper's example shape
    X = rng.uniform(-math.pi, math.pi, (P, N)).astype(np.float32)
    a0 = 0.3
    a = rng.uniform(-1, 1, K).astype(np.float32)
    b = rng.uniform(-1, 1, K).astype(np.float32)
    w = np.concatenate([[np.float32(a0)]] + [np.concatenate([a, b])] * N).astype(np.float32)
    X64 = X.astype(np.float64)
    k = np.arange(1, K + 1)
    Csum = np.cos(X64[:, :, None] * k).sum(axis=1)    # [P, K]
    Ssum = np.sin(X64[:, :, None] * k).sum(axis=1)
    out_shared = float(np.float32(a0)) + Csum @ a.astype(np.float64) + Ssum @ b.astype(np.float64)
    out = np.array([oracle.output(N, K, fam(TRIG, IDEN), X[p], w) for p in range(P)])
    np.testing.assert_allclose(out, out_shared, rtol=0, atol=1e-13)
    # and the MSE of that chromosome
    t = rng.normal(size=P).astype(np.float32)
    F = oracle.eval_fitness(K, fam(TRIG, IDEN), X, t, w[None, :])
    assert abs(F[0] - np.mean((out_shared - t.astype(np.float64)) ** 2)) < 1e-13


# ---------------------------------------------------------------- fitness closed forms
@pytest.mark.parametrize("expansion,d", [(CHEB, 3), (TRIG, 2)])
def test_zero_population_closed_forms(expansion, d):
    rng = np.random.default_rng(3)
    P, N, M = 77, 4, 5
    X = rng.uniform(-1, 1, (P, N)).astype(np.float32)
    G = oracle.num_genes(N, d, fam(expansion, SIGM))
    W = np.zeros((M, G), dtype=np.float32)
    labels = (rng.uniform(size=P) > 0.4).astype(np.float32)
    np.testing.assert_array_equal(oracle.eval_fitness(d, fam(expansion, SIGM), X, labels, W), 0.25)
    t = rng.normal(size=P).astype(np.float32)
    mt2 = np.mean(t.astype(np.float64) ** 2)
    for act in (TANH, IDEN):
        np.testing.assert_allclose(oracle.eval_fitness(d, fam(expansion, act), X, t, W), mt2, rtol=1e-15)


def test_bias_only_chromosome_closed_form():
    """w = (c,0,...): F = pi1 (1-s(c))^2 + (1-pi1) s(c)^2 with pi1 the label fraction."""
    rng = np.random.default_rng(4)
    P, N, d = 1000, 4, 3
    X = rng.uniform(-1, 1, (P, N)).astype(np.float32)
    t = (rng.uniform(size=P) > 0.3).astype(np.float32)
    pi1 = float(t.mean(dtype=np.float64))
    cs = np.array([-2.0, -0.5, 0.0, 0.75, 3.0], dtype=np.float32)
    W = np.zeros((len(cs), 13), dtype=np.float32)
    W[:, 0] = cs
    F = oracle.eval_fitness(d, fam(CHEB, SIGM), X, t, W)
    s = 1 / (1 + np.exp(-cs.astype(np.float64)))
    np.testing.assert_allclose(F, pi1 * (1 - s) ** 2 + (1 - pi1) * s**2, rtol=1e-13)


def test_generating_chromosome_has_zero_fitness_exact():
    """north_star pin: zero fitness for the generating chromosome on noiseless regression
    targets.  Dyadic features and integer genes make every term exact in binary32/64."""
    rng = np.random.default_rng(6)
    P, N, d = 64, 3, 3
    X = rng.choice(np.array([-1, -0.5, -0.25, 0, 0.25, 0.5, 1], dtype=np.float32), size=(P, N))
    G = N * d + 1
    W = rng.integers(-4, 5, size=(3, G)).astype(np.float32)
    V = np.polynomial.chebyshev.chebvander(X.astype(np.float64), d)[..., 1:].reshape(P, N * d)
    Phi = np.concatenate([np.ones((P, 1)), V], axis=1)
    t = (Phi @ W[1].astype(np.float64)).astype(np.float32)
    assert np.array_equal(t.astype(np.float64), Phi @ W[1].astype(np.float64))   # targets exact
    F = oracle.eval_fitness(d, fam(CHEB, IDEN), X, t, W)
    assert F[1] == 0.0 and F[0] > 0.0 and F[2] > 0.0


def test_generating_chromosome_noiseless_tanh_is_rounding_level():
    cfg = wl.scaled(wl.CONFIGS["c2"], P=500, noise_std=0.0, M=2)
    X, t, w_star = wl.make_kb(cfg)
    W = np.stack([w_star.astype(np.float32), np.zeros(cfg.G, dtype=np.float32)])
    F = oracle.eval_fitness(cfg.d, cfg.family, X, t, W)
    # targets are float32-rounded and the genes are float32-rounded copies of w*:
    # |error| <~ 1e-6 per pattern -> F <~ 1e-12; the zero chromosome is at mean(t^2)
    assert F[0] < 1e-11
    assert abs(F[1] - np.mean(t.astype(np.float64) ** 2)) < 1e-15


# ---------------------------------------------------------------- brute force / library
def _brute_force_fitness(N, d, expansion, act, X, t, W):
    """Independent pure-Python statement: explicit polynomials / math.cos, no recurrence,
    genes addressed through (feature, order) rather than a running index."""
    cheb = [lambda x: 1.0, lambda x: x, lambda x: 2 * x * x - 1, lambda x: 4 * x**3 - 3 * x,
            lambda x: 8 * x**4 - 8 * x * x + 1]
    P, M = len(X), len(W)
    F = []
    for m in range(M):
        acc = 0.0
        for p in range(P):
            z = float(W[m][0])
            for i in range(N):
                xi = float(X[p][i])
                for j in range(1, d + 1):
                    if expansion == CHEB:
                        z += float(W[m][1 + i * d + j - 1]) * cheb[j](xi)
                    else:
                        z += float(W[m][1 + i * 2 * d + j - 1]) * math.cos(j * xi)
                        z += float(W[m][1 + i * 2 * d + d + j - 1]) * math.sin(j * xi)
            y = 1 / (1 + math.exp(-z)) if act == SIGM else math.tanh(z) if act == TANH else z
            acc += (y - float(t[p])) ** 2
        F.append(acc / P)
    return np.array(F)


@pytest.mark.parametrize("expansion", [CHEB, TRIG])
@pytest.mark.parametrize("act", [IDEN, SIGM, TANH])
def test_fitness_brute_force_tiny(expansion, act):
    rng = np.random.default_rng(100 + 10 * expansion + act)
    P, N, d, M = 8, 2, 3, 4
    X = rng.uniform(-1, 1, (P, N)).astype(np.float32)
    t = rng.uniform(0, 1, P).astype(np.float32)
    G = oracle.num_genes(N, d, fam(expansion, act))
    W = rng.uniform(-1, 1, (M, G)).astype(np.float32)
    F = oracle.eval_fitness(d, fam(expansion, act), X, t, W)
    np.testing.assert_allclose(F, _brute_force_fitness(N, d, expansion, act, X, t, W), rtol=1e-13)


@pytest.mark.parametrize("name,P,M", [("c0", 1000, 64), ("c1", 700, 9), ("c2", 600, 7), ("c3", 300, 5)])
def test_fitness_matches_blas_on_library_design_matrix(name, P, M):
    """P-FIT-brute (library form): Phi from numpy's chebvander / cos / sin in float64,
    Phi @ W.T by BLAS dgemm, activation, mean."""
    cfg = wl.scaled(wl.CONFIGS[name], P=P, M=M)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(M, cfg.G, seed=9)
    F, S = oracle.eval_fitness(cfg.d, cfg.family, X, t, W, return_sse=True)
    X64 = X.astype(np.float64)
    if cfg.expansion == CHEB:
        blocks = np.polynomial.chebyshev.chebvander(X64, cfg.d)[..., 1:].reshape(P, -1)
    else:
        k = np.arange(1, cfg.d + 1)
        blocks = np.concatenate([np.cos(X64[..., None] * k), np.sin(X64[..., None] * k)], -1).reshape(P, -1)
    Phi = np.concatenate([np.ones((P, 1)), blocks], 1)
    Z = Phi @ W.astype(np.float64).T
    Y = 1 / (1 + np.exp(-Z)) if cfg.activation == SIGM else np.tanh(Z)
    ref = ((Y - t.astype(np.float64)[:, None]) ** 2).mean(0)
    np.testing.assert_allclose(F, ref, rtol=1e-12)
    np.testing.assert_allclose(S, ref * P, rtol=1e-12)


# ---------------------------------------------------------------- invariants
def test_identity_fitness_is_a_quadratic_form():
    """P-FIT-linear: F(w) = w'Aw - 2b'w + c with A = Phi'Phi/P (identity family), and
    superposition of outputs."""
    rng = np.random.default_rng(21)
    P, N, d = 50, 3, 2
    f = fam(CHEB, IDEN)
    G = oracle.num_genes(N, d, f)
    X = rng.uniform(-1, 1, (P, N)).astype(np.float32)
    t = rng.normal(size=P).astype(np.float32)
    Phi = np.stack([oracle.expand(N, d, f, X[p]) for p in range(P)])
    A = Phi.T @ Phi / P
    b = Phi.T @ t.astype(np.float64) / P
    c = np.mean(t.astype(np.float64) ** 2)
    W = rng.uniform(-1, 1, (6, G)).astype(np.float32)
    F = oracle.eval_fitness(d, f, X, t, W)
    W64 = W.astype(np.float64)
    quad = np.einsum("mg,gh,mh->m", W64, A, W64) - 2 * W64 @ b + c
    np.testing.assert_allclose(F, quad, rtol=1e-12)
    w1 = np.float32([0.5] * G)
    w2 = np.float32([-0.25 * (g % 3) for g in range(G)])
    o = lambda w: oracle.output(N, d, f, X[0], w)
    assert abs(o(w1 + w2) - (o(w1) + o(w2))) < 1e-15


def test_fitness_permutation_and_duplicates():
    cfg = wl.scaled(wl.CONFIGS["c0"], P=333, M=6)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(6, cfg.G, seed=1)
    W[4] = W[1]
    F = oracle.eval_fitness(cfg.d, cfg.family, X, t, W)
    assert F[4] == F[1]
    perm = np.array([5, 3, 1, 0, 2, 4])
    np.testing.assert_array_equal(oracle.eval_fitness(cfg.d, cfg.family, X, t, W[perm]), F[perm])
    # fitness of the hidden chromosome beats random ones on the classification recipe
    Xs, ts, w_star = wl.make_kb(cfg)
    Fs = oracle.eval_fitness(cfg.d, cfg.family, Xs, ts, np.vstack([w_star.astype(np.float32)[None], W]))
    assert Fs[0] == Fs.min() and Fs[0] < 0.1


def test_nan_propagates_to_that_chromosome_only():
    cfg = wl.scaled(wl.CONFIGS["c0"], P=50, M=3)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(3, cfg.G, seed=2)
    W[1, 5] = np.nan
    F = oracle.eval_fitness(cfg.d, cfg.family, X, t, W)
    assert np.isnan(F[1]) and np.isfinite(F[0]) and np.isfinite(F[2])


# ---------------------------------------------------------------- the input recipe itself
def test_workload_recipe_shapes_and_balance():
    cfg = wl.scaled(wl.CONFIGS["c1"], P=20000)
    X, t, w = wl.make_kb(cfg)
    assert X.dtype == np.float32 and t.dtype == np.float32 and X.shape == (20000, 10) and w.shape == (61,)
    assert X.min() >= -1 and X.max() <= 1 and set(np.unique(t)) == {0.0, 1.0}
    assert 0.2 < t.mean() < 0.8
    X2, t2, _ = wl.make_kb(cfg)
    assert np.array_equal(X, X2) and np.array_equal(t, t2)          # seeded
    c2 = wl.scaled(wl.CONFIGS["c2"], P=5000)
    X, t, _ = wl.make_kb(c2)
    assert abs(X).max() <= np.float32(math.pi) and abs(t).max() < 1.1
    assert wl.shard_patterns(10, 3, 0) == (0, 4) and wl.shard_patterns(10, 3, 2) == (7, 10)


# ------------------------------------------------------------------------------------------------ predict / confusion
def test_predict_is_the_model_behind_the_fitness():
    """mean((predict - t)^2) must be the (already pinned) fitness of that chromosome: ties the test / validation use
    case to eq.(2)-(3); and a numpy chebvander evaluation of the same outputs (library routine)."""
    import workloads as wl
    cfg = wl.scaled(wl.CONFIGS["c1"], P=400, M=6)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 21)
    F = oracle.eval_fitness(cfg.d, cfg.family, X, t, W)
    for m in range(cfg.M):
        y = oracle.predict(cfg.d, cfg.family, X, W[m])
        assert abs(np.mean((y - t.astype(np.float64)) ** 2) - F[m]) <= 1e-15
        z = wl._design_matrix(cfg, X.astype(np.float64)) @ W[m].astype(np.float64)
        assert np.max(np.abs(y - 1.0 / (1.0 + np.exp(-z)))) <= 1e-14


def test_confusion_counts_brute_force_and_identities():
    y = np.array([0.9, 0.2, 0.5, 0.51, 0.49, 1.0, 0.0, np.nan])
    t = np.array([1, 1, 1, 0, 0, 0, 0, 1], dtype=np.float32)
    # by hand at threshold 0.5: pred = [1,0,0,1,0,1,0,0] (y > thr; 0.5 and NaN are not above it)
    assert oracle.confusion(y, t, 0.5) == (1, 2, 2, 3)
    rng = np.random.default_rng(3)
    y = rng.uniform(size=1000); t = (rng.uniform(size=1000) > 0.4).astype(np.float32)
    tp, fp, tn, fn = oracle.confusion(y, t, 0.3)
    pred = y > 0.3
    assert (tp, fp, tn, fn) == (int(np.sum(pred & (t > 0.5))), int(np.sum(pred & (t <= 0.5))),
                                int(np.sum(~pred & (t <= 0.5))), int(np.sum(~pred & (t > 0.5))))
    assert tp + fp + tn + fn == 1000 and oracle.confusion(t.astype(np.float64), t, 0.5) == (int(t.sum()), 0, int(1000 - t.sum()), 0)


def test_rmse_closed_forms():
    """RMSE: W = 0 on 0/1 labels -> exactly 0.5; it is the Euclidean norm of the residual / sqrt(P)
    (numpy.linalg.norm, a library routine) and orders chromosomes exactly as the MSE does."""
    import workloads as wl
    cfg = wl.scaled(wl.CONFIGS["c1"], P=500, M=12)
    X, t, _ = wl.make_kb(cfg)
    assert np.all(oracle.eval_rmse(cfg.d, cfg.family, X, t, np.zeros((3, cfg.G), np.float32)) == 0.5)
    W = wl.uniform_population(cfg.M, cfg.G, 2)
    R = oracle.eval_rmse(cfg.d, cfg.family, X, t, W)
    for m in range(cfg.M):
        y = oracle.predict(cfg.d, cfg.family, X, W[m])
        assert abs(R[m] - np.linalg.norm(y - t) / np.sqrt(cfg.P)) <= 1e-14
    assert np.array_equal(np.argsort(R, kind="stable"), np.argsort(oracle.eval_fitness(cfg.d, cfg.family, X, t, W), kind="stable"))


# ------------------------------------------------------------------------------------------------ shared coefficients
def _golden_example():
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_worked_example.txt")
    return dict(l.split(None, 1) for l in open(path) if l.strip() and not l.startswith("#"))


def test_shared_mode_is_the_papers_worked_example_shape():
    """11 features, degree 3, polytrigo (B = 2) -> 7 genes [a0,a1,a2,a3,b1,b2,b3], 23 chromosomes."""
    ex = _golden_example()
    N, d = int(ex["features"]), int(ex["degree"])
    fam = oracle.family(oracle.EXP_TRIG, oracle.ACT_IDENTITY, shared=True)
    assert oracle.num_genes(N, d, fam) == int(ex["num_genes"]) == 7
    assert oracle.paper_shapes(N, d, int(ex["B"])) == (int(ex["num_chromosomes"]), int(ex["num_genes"]))
    assert oracle.num_genes(N, d, oracle.family(oracle.EXP_CHEBYSHEV, 0, shared=True)) == d + 1
    # gene order: a unit gene at position g picks out the documented term -- a_k -> sum_i cos(k x_i), b_k -> sum_i sin(k x_i)
    x = np.linspace(-2.5, 2.5, N).astype(np.float32)
    for g, name in enumerate(ex["gene_order"].split()):
        w = np.zeros(7, np.float32); w[g] = 1.0
        k = int(name[1])
        want = 1.0 if name == "a0" else float(np.sum((np.cos if name[0] == "a" else np.sin)(k * x.astype(np.float64))))
        assert abs(oracle.output(N, d, fam, x, w) - want) <= 1e-13, name


@pytest.mark.parametrize("expansion,act", [(0, 1), (1, 2), (1, 0)])
def test_shared_mode_equals_per_feature_model_with_tied_genes(expansion, act):
    """eq.(2) shares a_j across the features: the shared model must equal the per-feature model (BASELINE form, D1)
    whose genes are tied across features -- two code paths, one number."""
    rng = np.random.Generator(np.random.Philox(12))
    P, N, d, M = 300, 6, 4, 5
    X = rng.uniform(-1, 1, (P, N)).astype(np.float32)
    t = rng.uniform(0, 1, P).astype(np.float32)
    B = 2 if expansion == 1 else 1
    Ws = rng.uniform(-1, 1, (M, B * d + 1)).astype(np.float32)
    Wp = np.concatenate([Ws[:, :1]] + [Ws[:, 1:]] * N, axis=1)          # [a0 | block | block | ...]
    Fs = oracle.eval_fitness(d, oracle.family(expansion, act, shared=True), X, t, Ws)
    Fp = oracle.eval_fitness(d, oracle.family(expansion, act), X, t, Wp)
    assert np.max(np.abs(Fs - Fp) / Fp) <= 1e-12
