"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs (workloads.py).  Bars (BASELINE.json north_star): GA operators and population init
bit-exact; per-chromosome fitness within 1e-5 relative; best-fitness trajectories within 1e-4."""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

REL_TOL = 1e-5          # north_star: per-chromosome fitness relative error
ABS_FLOOR = 1e-10       # only matters where the reference fitness is ~0 (noiseless-regression pin)


@pytest.fixture(scope="module")
def game():
    import paper_1211_5481_b200 as g
    from paper_1211_5481_b200 import build
    build.build()
    g.lib()
    return g


def make(game, cfg, scheme=0):
    G = game.Game(cfg.P, cfg.N, cfg.d, cfg.M, cfg.expansion, cfg.activation, scheme=scheme)
    assert G.G == cfg.G
    G.set_ga_params(cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma)
    return G


def assert_fitness_close(F_gpu, F_ref, what=""):
    F_gpu = np.asarray(F_gpu, dtype=np.float64)
    err = np.abs(F_gpu - F_ref)
    bound = REL_TOL * np.abs(F_ref) + ABS_FLOOR
    worst = int(np.argmax(err - bound))
    assert np.all(err <= bound), (f"{what}: chromosome {worst}: gpu {F_gpu[worst]!r} ref {F_ref[worst]!r} "
                                   f"rel {err[worst] / max(abs(F_ref[worst]), 1e-300):.3e}")
    return float(np.max(err / np.maximum(np.abs(F_ref), 1e-300)))


SCHEMES = [1, 2]   # FFMA, F16X3

# (name, base config, overrides): several tiles + ragged tails in P (256-pattern tiles) and M (128-chromosome tiles)
FITNESS_CASES = [
    ("c0_full", "c0", {}),
    ("c0_ragged", "c0", dict(P=777, M=37)),
    ("c1_slice", "c1", dict(P=5000, M=200)),
    ("c1_one_pattern", "c1", dict(P=1, M=5)),
    ("c2_slice", "c2", dict(P=3000, M=130)),
    ("c3_slice", "c3", dict(P=1100, M=260)),
    ("c4_slice", "c4", dict(P=2049, M=129)),
    ("odd_shapes", "c1", dict(P=1537, N=9, d=5, M=131)),
    ("trig_odd", "c2", dict(P=700, N=5, d=3, M=33)),
    ("identity_cheb", "c1", dict(P=2000, M=64, activation=wl.ACT_IDENTITY)),
    ("tanh_cheb", "c1", dict(P=2000, M=64, activation=wl.ACT_TANH)),
    ("sigmoid_trig", "c2", dict(P=2000, M=64, activation=wl.ACT_SIGMOID)),
    ("d1", "c1", dict(P=1000, N=3, d=1, M=16)),
    # K extent too long for phi to stay resident in shared memory -> the kernel's streaming mode (25 K steps)
    ("stream_cheb", "c3", dict(P=1300, N=32, d=12, M=300)),
    ("stream_trig", "c2", dict(P=900, N=16, d=12, M=140)),
    # many chromosome tiles per unit with resident phi (reuse across 5 tile pairs), ragged everything
    ("resident_reuse", "c3", dict(P=2100, N=31, d=9, M=1111)),
    # more features than the old 32 / 16 limits (x is read straight from global memory)
    ("wide_cheb", "c3", dict(P=900, N=44, d=10, M=140)),
    ("wide_trig", "c2", dict(P=700, N=27, d=5, M=70)),
    ("stream_tail", "c3", dict(P=800, N=24, d=14, M=150)),       # streaming, 21 K steps: last stage holds 1 of 4 steps
    ("stream_tail_trig", "c2", dict(P=800, N=24, d=7, M=150)),   # streaming trig, 21 K steps
    ("huge_G_641", "c3", dict(P=600, N=64, d=10, M=70)),      # beyond the FFMA kernel's G <= 448: tensor path only
    # degrees far beyond a K step: a feature spans several k-groups, the producers enter items in mid-feature
    ("deg70_cheb", "c1", dict(P=1500, N=6, d=70, M=140)),
    ("deg100_cheb", "c1", dict(P=1500, N=10, d=100, M=140)),  # G = 1001, streaming
    ("deg300_cheb", "c3", dict(P=900, N=3, d=300, M=70)),
    ("deg100_trig", "c2", dict(P=900, N=3, d=100, M=70)),     # G = 601
]


def case_cfg(base, over):
    cfg = wl.c4(256, 100_000) if base == "c4" else wl.CONFIGS[base]
    return wl.scaled(cfg, **over)


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("name,base,over", FITNESS_CASES, ids=[c[0] for c in FITNESS_CASES])
def test_fitness_matches_oracle(game, name, base, over, scheme):
    cfg = case_cfg(base, over)
    if scheme == 1 and cfg.G > 448:
        pytest.skip("the FFMA kernel covers G <= 448")
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, seed=100 + cfg.seed)
    G = make(game, cfg, scheme)
    G.load_kb(X, t)
    G.set_population(W)
    G.eval_fitness()
    G.sync()
    assert G.scheme() == scheme
    F_ref = oracle.eval_fitness(cfg.d, cfg.family, X, t, W)
    assert_fitness_close(G.get_fitness(), F_ref, f"{name} scheme {scheme}")
    G.close()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_fitness_closed_forms_on_gpu(game, scheme):
    """W = 0 -> sigmoid fitness exactly 0.25 on 0/1 labels; generating chromosome on noiseless regression
    targets -> fitness ~ 0 (absolute floor); duplicate chromosomes -> identical fitness in any slot."""
    cfg = wl.scaled(wl.CONFIGS["c1"], P=3000, M=140)
    X, t, _ = wl.make_kb(cfg)
    G = make(game, cfg, scheme)
    G.load_kb(X, t)
    G.set_population(np.zeros((cfg.M, cfg.G), np.float32))
    G.eval_fitness(); G.sync()
    assert np.all(G.get_fitness() == np.float32(0.25))
    W = wl.uniform_population(cfg.M, cfg.G, 5)
    W[137] = W[3]; W[64] = W[3]
    G.set_population(W); G.eval_fitness(); G.sync()
    F = G.get_fitness()
    assert F[137] == F[3] == F[64]
    G.close()
    # noiseless regression, tanh / trig
    cfg = wl.scaled(wl.CONFIGS["c2"], P=2500, M=130, noise_std=0.0)
    X, t, w_star = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 6)
    W[7] = w_star.astype(np.float32)
    t = np.tanh(wl._design_matrix(cfg, X.astype(np.float64)) @ W[7].astype(np.float64)).astype(np.float32)
    G = make(game, cfg, scheme)
    G.load_kb(X, t); G.set_population(W); G.eval_fitness(); G.sync()
    F = G.get_fitness()
    assert F[7] <= 1e-10 + 1e-14, F[7]      # float32 rounding of t leaves ~1e-15
    assert_fitness_close(F, oracle.eval_fitness(cfg.d, cfg.family, X, t, W), "noiseless")
    G.close()


def test_fitness_is_deterministic_and_schemes_agree(game):
    cfg = wl.scaled(wl.CONFIGS["c3"], P=5000, M=300)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 9)
    out = {}
    for scheme in SCHEMES:
        G = make(game, cfg, scheme)
        G.load_kb(X, t); G.set_population(W)
        G.eval_fitness(); G.sync(); a = G.get_fitness()
        G.eval_fitness(); G.sync(); b = G.get_fitness()
        assert np.array_equal(a, b), "run-to-run bit stability"
        out[scheme] = a.astype(np.float64)
        G.close()
    assert np.max(np.abs(out[1] - out[2]) / out[1]) < 2e-6


@pytest.mark.parametrize("P", [600, 512])       # a ragged last tile, and whole tiles only (the packed epilogue path alone)
def test_nan_and_inf_propagate(game, P):
    cfg = wl.scaled(wl.CONFIGS["c0"], P=P, M=20)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 3)
    W[4, 2] = np.nan
    for scheme in SCHEMES:
        G = make(game, cfg, scheme)
        G.load_kb(X, t); G.set_population(W); G.eval_fitness(); G.sync()
        F = G.get_fitness()
        assert np.isnan(F[4]) and np.all(np.isfinite(np.delete(F, 4)))
        G.close()


# ------------------------------------------------------------------------------------------------ GA operators
@pytest.mark.parametrize("M,G_,seed", [(64, 13, 0), (512, 61, 1), (1000, 129, 2), (37, 1, 3), (130, 321, 2**40 + 17)])
def test_init_population_bit_exact(game, M, G_, seed):
    N, d = (G_ - 1, 1) if G_ > 1 else (1, 1)
    if G_ == 1:
        pytest.skip("G = 1 needs N*d = 0")
    G = game.Game(300, N, d, M, wl.EXP_CHEBYSHEV, wl.ACT_SIGMOID)
    G.init_population(seed); G.sync()
    W = G.get_population()
    assert np.array_equal(W.view(np.uint32), oracle.init_population(M, G_, seed).view(np.uint32))
    assert W.min() >= -1.0 and W.max() < 1.0
    G.close()


STEP_CASES = [
    # M, N, d, E, k, p_cross, p_mut, sigma, seed, gen
    (64, 4, 3, 2, 3, 0.9, 0.05, 0.1, 0, 0),
    (512, 10, 6, 4, 3, 0.9, 0.05, 0.1, 1, 7),
    (1024, 16, 8, 8, 4, 0.9, 0.02, 0.05, 2, 49),
    (4096, 32, 10, 4, 3, 0.9, 0.05, 0.1, 3, 19),
    (100, 5, 4, 0, 1, 0.0, 0.0, 0.0, 4, 1),
    (100, 5, 4, 99, 2, 1.0, 1.0, 0.5, 5, 2),
    (33, 2, 1, 1, 7, 0.5, 0.5, 1.0, 2**63 + 5, 2**31 + 3),
    (257, 7, 3, 3, 2, 1.0, 0.2, 0.1, 6, 123456),
]


@pytest.mark.parametrize("M,N,d,E,k,pc,pm,sigma,seed,gen", STEP_CASES)
def test_ga_step_bit_exact_on_given_fitness(game, M, N, d, E, k, pc, pm, sigma, seed, gen):
    """Same fitness vector and seed in, bit-identical next population out (north_star)."""
    rng = np.random.Generator(np.random.Philox(1000 + M))
    G = game.Game(300, N, d, M, wl.EXP_CHEBYSHEV, wl.ACT_SIGMOID)
    W = rng.uniform(-2, 2, size=(M, G.G)).astype(np.float32)
    F = rng.uniform(0, 1, size=M).astype(np.float32)
    F[rng.integers(0, M, size=max(1, M // 8))] = F[0]          # ties
    if M > 40:
        F[5] = np.nan; F[17] = np.inf; F[20] = -0.0; F[21] = 0.0
    G.set_ga_params(E, k, pc, pm, sigma)
    G.set_population(W); G.set_fitness(F)
    G.step(seed, gen); G.sync()
    Wn = G.get_population()
    ref = oracle.step(W, F, E, k, pc, pm, sigma, seed, gen)
    assert np.array_equal(Wn.view(np.uint32), ref.view(np.uint32)), \
        f"{np.count_nonzero(Wn.view(np.uint32) != ref.view(np.uint32))} genes differ"
    G.close()


def test_step_state_machine_on_gpu(game):
    cfg = wl.scaled(wl.CONFIGS["c0"], P=300)
    G = make(game, cfg)
    G.init_population(1)
    with pytest.raises(game.GameError) as e:
        G.step(1, 0)
    assert e.value.code == game.ERR_BAD_STATE
    X, t, _ = wl.make_kb(cfg)
    G.load_kb(X, t)
    G.eval_fitness(); G.step(1, 0)
    with pytest.raises(game.GameError):
        G.step(1, 1)           # fitness is stale after a step
    G.sync(); G.close()


# ------------------------------------------------------------------------------------------------ trajectories
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("base,over", [("c0", {}), ("c1", dict(P=4000, M=256, generations=12)),
                                       ("c2", dict(P=3000, M=128, generations=8))])
def test_lockstep_and_free_running_trajectory(game, base, over, scheme):
    """Lock-step: every generation the oracle steps on the GPU's fitness vector -> populations stay
    bit-identical and GPU fitness stays within 1e-5 of the oracle's fitness of the same population.
    Free-running: game_run's best-fitness trace within 1e-4 of the oracle's run."""
    import torch
    cfg = case_cfg(base, over)
    X, t, _ = wl.make_kb(cfg)
    seed, n = 1234 + cfg.seed, cfg.generations
    G = make(game, cfg, scheme)
    G.load_kb(X, t)
    G.init_population(seed); G.sync()
    W0 = G.get_population()
    assert np.array_equal(W0.view(np.uint32), oracle.init_population(cfg.M, cfg.G, seed).view(np.uint32))
    W = W0.copy()
    best_lock = []
    for g in range(n):
        G.eval_fitness(); G.sync()
        F_gpu = G.get_fitness()
        assert_fitness_close(F_gpu, oracle.eval_fitness(cfg.d, cfg.family, X, t, W), f"gen {g}")
        best_lock.append(F_gpu[oracle.best_index(F_gpu)])
        G.step(seed, g); G.sync()
        W = oracle.step(W, F_gpu, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, seed, g)
        assert np.array_equal(G.get_population().view(np.uint32), W.view(np.uint32)), f"population forked at gen {g}"
    # free-running on the device, one sync at the end
    G.set_population(W0)
    best = torch.full((n + 1,), float("nan"), dtype=torch.float32, device="cuda:0")
    G.run(seed, 0, n, best); G.sync()
    best = best.cpu().numpy()
    assert np.array_equal(best[:n], np.asarray(best_lock, np.float32)), "run() must replay the lock-step generations"
    _, _, best_ref = oracle.run(cfg.d, cfg.family, X, t, W0, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut,
                                cfg.sigma, seed, 0, n)
    dev = np.abs(best.astype(np.float64) - best_ref) / np.maximum(np.abs(best_ref), 1e-6)
    assert np.all(dev <= 1e-4), dev
    if cfg.elite >= 1:
        assert np.all(np.diff(best) <= 0), "best fitness must not get worse with elitism"
    G.close()


def test_checkpoint_resume_bit_exact(game):
    cfg = wl.scaled(wl.CONFIGS["c0"], P=500)
    X, t, _ = wl.make_kb(cfg)
    G = make(game, cfg); G.load_kb(X, t); G.init_population(5)
    G.run(5, 0, 6, None); G.sync()
    full = G.get_population()
    G.init_population(5); G.run(5, 0, 3, None); G.sync()
    ckpt = G.get_population()
    G.close()
    G2 = make(game, cfg); G2.load_kb(X, t); G2.set_population(ckpt)
    G2.run(5, 3, 3, None); G2.sync()
    assert np.array_equal(G2.get_population().view(np.uint32), full.view(np.uint32))
    G2.close()


@pytest.mark.parametrize("base", ["c1", "c2"])          # c2: tanh, i.e. with the calibration launches behind the upload
def test_generation_host_entry(game, base):
    """The host-buffer entry point = load + eval + step + download."""
    import torch
    cfg = wl.scaled(wl.CONFIGS[base], P=3000, M=150)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 11)
    G = make(game, cfg)
    Xh, th, Wh = (torch.from_numpy(a).pin_memory() for a in (X, t, W))
    Fh = torch.empty(cfg.M, dtype=torch.float32).pin_memory()
    Wn = torch.empty((cfg.M, cfg.G), dtype=torch.float32).pin_memory()
    game.game_generation_host(G.ctx, Xh.data_ptr(), th.data_ptr(), Wh.data_ptr(), Fh.data_ptr(), Wn.data_ptr(), 77, 3)
    F = Fh.numpy()
    assert_fitness_close(F, oracle.eval_fitness(cfg.d, cfg.family, X, t, W), "host entry")
    ref = oracle.step(W, F, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, 77, 3)
    assert np.array_equal(Wn.numpy().view(np.uint32), ref.view(np.uint32))
    assert G.launch_count() >= 3
    G.close()


# ------------------------------------------------------------------------------------------------ full sizes
def test_full_size_c1_all_chromosomes(game):
    """BASELINE.json configs[1] at full size, in the launch configuration bench.py times (AUTO scheme, persistent
    grid of CTA pairs): every chromosome against the oracle."""
    cfg = wl.CONFIGS["c1"]
    X, t, _ = wl.make_kb(cfg)
    G = make(game, cfg)
    G.load_kb(X, t); G.init_population(cfg.seed); G.eval_fitness(); G.sync()
    assert G.scheme() == game.SCHEME_F16X3
    W = G.get_population()
    assert_fitness_close(G.get_fitness(), oracle.eval_fitness(cfg.d, cfg.family, X, t, W), "c1 full size")
    G.close()


def test_full_size_c3_sampled_chromosomes(game):
    """BASELINE.json configs[3] (the headline workload) at full size P = 4e6, M = 4096: the oracle cannot finish the
    whole population, so sampled chromosomes (best, worst, first, last, two tile edges) are computed one by one."""
    cfg = wl.CONFIGS["c3"]
    X, t, _ = wl.make_kb(cfg)
    G = make(game, cfg)
    G.load_kb(X, t); G.init_population(cfg.seed); G.eval_fitness(); G.sync()
    assert G.scheme() == game.SCHEME_F16X3
    W, F = G.get_population(), G.get_fitness()
    assert np.all(np.isfinite(F)) and F.min() > 0
    rows = sorted({int(np.argmin(F)), int(np.argmax(F)), 0, cfg.M - 1, 127, 128})
    F_ref = oracle.eval_fitness(cfg.d, cfg.family, X, t, W[rows])
    assert_fitness_close(F[rows], F_ref, "c3 full size, sampled rows")
    # property that holds at any size: duplicated chromosomes get bit-identical fitness in any slot
    W[4000] = W[rows[0]]; W[77] = W[rows[0]]
    G.set_population(W); G.eval_fitness(); G.sync()
    F2 = G.get_fitness()
    assert F2[4000] == F2[77] == F2[rows[0]] == F[rows[0]]
    G.close()


def test_evolve_equals_eval_step_loop(game):
    cfg = wl.scaled(wl.CONFIGS["c1"], P=3000, M=300)
    X, t, _ = wl.make_kb(cfg)
    G = make(game, cfg); G.load_kb(X, t); G.init_population(9)
    for g in range(4):
        G.eval_fitness(); G.step(9, g)
    G.sync(); a = G.get_population()
    G.init_population(9)
    game.game_evolve(G.ctx, 9, 0, 4); G.sync()
    assert np.array_equal(G.get_population().view(np.uint32), a.view(np.uint32))
    G.close()


def test_generation_host_entry_pipelined_ranges(game):
    """A knowledge base >= 64 MB makes game_generation_host upload it in 8 pattern ranges on a copy stream, each
    evaluated as soon as it has landed (partial sums carried across the launches): same bars as everywhere else."""
    import torch
    cfg = wl.scaled(wl.CONFIGS["c3"], P=560_123, M=300)          # 72 MB of X, ragged last tile
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 12)
    G = make(game, cfg)
    G.X.zero_(); G.t.zero_()                                     # the device copy must come from the host buffers
    Xh, th, Wh = (torch.from_numpy(a).pin_memory() for a in (X, t, W))
    Fh = torch.empty(cfg.M, dtype=torch.float32).pin_memory()
    Wn = torch.empty((cfg.M, cfg.G), dtype=torch.float32).pin_memory()
    for rep in range(2):                                         # twice: the copy stream must wait for the previous eval
        game.game_generation_host(G.ctx, Xh.data_ptr(), th.data_ptr(), Wh.data_ptr(), Fh.data_ptr(), Wn.data_ptr(), 5, rep)
    F = Fh.numpy().copy()
    rows = [0, 1, 127, 128, 255, 256, 299]
    assert_fitness_close(F[rows], oracle.eval_fitness(cfg.d, cfg.family, X, t, W[rows]), "pipelined host entry")
    ref = oracle.step(W, F, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, 5, 1)
    assert np.array_equal(Wn.numpy().view(np.uint32), ref.view(np.uint32))
    assert torch.equal(G.X.cpu(), torch.from_numpy(X))
    G.close()


# ------------------------------------------------------------------------------------------------ test / validation use case
@pytest.mark.parametrize("base,over", [("c0", dict(P=777, M=16)), ("c1", dict(P=5001, M=16)), ("c2", dict(P=3000, M=16)),
                                       ("c3", dict(P=2047, M=16)), ("c1", dict(P=1000, M=16, activation=wl.ACT_IDENTITY))])
def test_predict_and_confusion_match_oracle(game, base, over):
    """game_predict / game_confusion: outputs of one chromosome on held-out patterns within 1e-5
    (relative to max(1, |y|): fp32 recurrences and a G-term fp32 dot product, |z| up to ~10) of the fp64 oracle; confusion counts bit-exact when both sides threshold the SAME fp32 outputs, and equal to
    the oracle's own counts wherever no output lies within the tolerance of the threshold."""
    import torch
    cfg = case_cfg(base, over)
    X, t, _ = wl.make_kb(cfg, seed=77)
    W = wl.uniform_population(cfg.M, cfg.G, 31)
    G = make(game, cfg)
    Xd, td = torch.from_numpy(X).cuda(), torch.from_numpy(t).cuda()
    Wd = torch.from_numpy(W).cuda()
    y = torch.empty(cfg.P, dtype=torch.float32, device="cuda")
    counts = torch.zeros(4, dtype=torch.int64, device="cuda")
    for m in (0, cfg.M - 1):
        game.game_predict(G.ctx, Wd[m].data_ptr(), Xd.data_ptr(), cfg.P, y.data_ptr())
        game.game_confusion(G.ctx, y.data_ptr(), td.data_ptr(), cfg.P, 0.5, counts.data_ptr())
        G.sync()
        y_gpu = y.cpu().numpy()
        y_ref = oracle.predict(cfg.d, cfg.family, X, W[m])
        scale = np.maximum(1.0, np.abs(y_ref))
        assert np.max(np.abs(y_gpu - y_ref) / scale) <= 1e-5
        got = tuple(int(c) for c in counts.cpu().numpy())
        assert got == oracle.confusion(y_gpu.astype(np.float64), t, 0.5)          # same fp32 outputs in -> bit-exact
        if np.min(np.abs(y_ref - 0.5)) > 2e-5:
            assert got == oracle.confusion(y_ref, t, 0.5)
        assert sum(got) == cfg.P
    G.close()


@pytest.mark.parametrize("N,d", [(130, 100), (600, 100)])
def test_predict_long_chromosomes(game, N, d):
    """game_predict with chromosomes beyond 48 KB (G = 13 001: staged in opted-in shared memory) and beyond what shared
    memory holds (G = 60 001: read through the caches): the trained model can be applied wherever training is accepted."""
    import torch
    Q = 700
    rng = np.random.Generator(np.random.Philox(90 + N))
    G = game.Game(8, N, d, 4, wl.EXP_CHEBYSHEV, wl.ACT_SIGMOID)
    fam = oracle.family(wl.EXP_CHEBYSHEV, wl.ACT_SIGMOID)
    assert G.G == N * d + 1
    X = rng.uniform(-1, 1, (Q, N)).astype(np.float32)
    w = (rng.uniform(-1, 1, G.G) / np.sqrt(G.G / 8.0)).astype(np.float32)
    y = torch.empty(Q, dtype=torch.float32, device="cuda")
    wd, Xd = torch.from_numpy(w).cuda(), torch.from_numpy(X).cuda()
    game.game_predict(G.ctx, wd.data_ptr(), Xd.data_ptr(), Q, y.data_ptr())
    G.sync()
    y_ref = oracle.predict(d, fam, X, w)
    assert np.max(np.abs(y.cpu().numpy() - y_ref)) <= 1e-5
    G.close()


# ------------------------------------------------------------------------------------------------ pattern sharding (N3)
@pytest.mark.parametrize("world", [2, 3])
def test_pattern_sharded_evaluation_single_device(game, world):
    """The multi-GPU path emulated on ONE device (ranks run one after the other, nothing waits on anything): each
    'rank' binds its contiguous shard of the patterns, game_eval_sse gives its partial sums, their sum goes through
    game_set_fitness_from_sse on every rank; fitness within 1e-5 of the oracle on the WHOLE knowledge base, and the
    GA step from it bit-identical on all ranks and to the oracle's."""
    import torch
    cfg = wl.scaled(wl.CONFIGS["c3"], P=3001, M=200)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 41)
    ranks, sse = [], torch.zeros(cfg.M, dtype=torch.float64, device="cuda")
    for r in range(world):
        p0, p1 = wl.shard_patterns(cfg.P, world, r)
        G = make(game, wl.scaled(cfg, P=p1 - p0))
        G.load_kb(X[p0:p1], t[p0:p1]); G.set_population(W)
        part = torch.empty(cfg.M, dtype=torch.float64, device="cuda")
        game.game_eval_sse(G.ctx, part.data_ptr()); G.sync()
        with pytest.raises(game.GameError):
            G.step(1, 0)                      # partial sums are not a fitness
        sse += part                           # the all-reduce
        ranks.append(G)
    F_ref, S_ref = oracle.eval_fitness(cfg.d, cfg.family, X, t, W, return_sse=True)
    assert np.max(np.abs(sse.cpu().numpy() - S_ref) / S_ref) <= 1e-5
    pops = []
    for G in ranks:
        game.game_set_fitness_from_sse(G.ctx, sse.data_ptr(), cfg.P, None)
        G.step(11, 4); G.sync()
        assert_fitness_close(G.get_fitness(), F_ref, "sharded fitness")
        pops.append(G.get_population())
    ref = oracle.step(W, ranks[0].get_fitness(), cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, 11, 4)
    for P_ in pops:
        assert np.array_equal(P_.view(np.uint32), ref.view(np.uint32))
    for G in ranks:
        G.close()


def test_evolve_sharded_world_of_one_matches_evolve(game):
    """game_evolve_sharded (the pattern-sharded generation loop inside the library: eval kernels, ncclAllReduce of M
    doubles on the library's stream, finalisation, GA step) on a communicator of ONE rank -- the only world this box
    has: NCCL is loaded, initialised and called in-stream, and the loop must reproduce game_run bit for bit."""
    import torch
    cfg = wl.scaled(wl.CONFIGS["c1"], P=3000, M=200)
    X, t, _ = wl.make_kb(cfg)
    n = 5
    A = make(game, cfg); A.load_kb(X, t); A.init_population(8)
    ref_best = torch.zeros(n + 1, dtype=torch.float32, device="cuda")
    A.run(8, 0, n, ref_best); A.sync()
    B = make(game, cfg); B.load_kb(X, t); B.init_population(8)
    try:
        ident = game.game_comm_unique_id()
    except game.GameError:
        pytest.skip("NCCL cannot be loaded in this process")
    game.game_comm_init(B.ctx, ident, 0, 1)
    best = torch.zeros(n, dtype=torch.float32, device="cuda")
    game.game_evolve_sharded(B.ctx, 8, 0, n, cfg.P, best.data_ptr()); B.sync()
    assert np.array_equal(B.get_population().view(np.uint32), A.get_population().view(np.uint32))
    assert np.array_equal(best.cpu().numpy(), ref_best.cpu().numpy()[:n])
    A.close(); B.close()


# ------------------------------------------------------------------------------------------------ out of core (N4)
@pytest.mark.parametrize("base,over,slot_rows,n_slots", [
    ("c3", dict(P=1_200_123, M=300), 50_176, 3),          # ring = 1/8 of the knowledge base; ragged last range and last tile
    ("c2", dict(P=300_000, M=520), 19_200, 2),            # tanh: the calibration launch runs on the first slot
    ("c1", dict(P=40_000, M=100), 65_536, 2),             # everything fits one slot
])
def test_streamed_out_of_core_evaluation_is_bit_identical(game, base, over, slot_rows, n_slots):
    """game_eval_fitness_streamed: the knowledge base stays in pinned HOST memory and passes through a ring
    of device buffers an eighth of its size; the fitness is bit-identical to the resident evaluation (same pattern tile ->
    CTA pair assignment, same order of the partial sums), twice in a row (ring re-use across calls), and the GA step runs on it."""
    import torch
    cfg = wl.scaled(wl.CONFIGS[base], **over)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 21)
    R = make(game, cfg); R.load_kb(X, t); R.set_population(W); R.eval_fitness(); R.sync()
    F_res = R.get_fitness()
    R.close()
    G = game.Game(cfg.P, cfg.N, cfg.d, cfg.M, cfg.expansion, cfg.activation, resident_kb=False)
    G.set_ga_params(cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma)
    assert G.X is None
    G.set_population(W)
    Xh, th = torch.from_numpy(X).pin_memory(), torch.from_numpy(t).pin_memory()
    Xr = torch.full((n_slots * slot_rows, cfg.N), float("nan"), dtype=torch.float32, device="cuda")
    tr = torch.full((n_slots * slot_rows,), float("nan"), dtype=torch.float32, device="cuda")
    assert Xr.numel() * 4 <= max(X.nbytes // 8 + 4 * 256 * cfg.N * n_slots, 2 * 65_536 * cfg.N * 4)
    for rep in range(2):
        game.game_eval_fitness_streamed(G.ctx, Xh.data_ptr(), th.data_ptr(), Xr.data_ptr(), tr.data_ptr(), slot_rows, n_slots)
        G.sync()
        assert np.array_equal(G.get_fitness().view(np.uint32), F_res.view(np.uint32)), f"pass {rep}"
    rows = sorted({0, min(127, cfg.M - 1), min(128, cfg.M - 1), cfg.M - 1})
    assert_fitness_close(F_res[rows], oracle.eval_fitness(cfg.d, cfg.family, X, t, W[rows]), "streamed vs oracle")
    G.step(5, 0); G.sync()
    ref = oracle.step(W, F_res, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, 5, 0)
    assert np.array_equal(G.get_population().view(np.uint32), ref.view(np.uint32))
    with pytest.raises(game.GameError) as e:          # a slot must hold one whole round of the persistent grid
        game.game_eval_fitness_streamed(G.ctx, Xh.data_ptr(), th.data_ptr(), Xr.data_ptr(), tr.data_ptr(), 256, n_slots)
    assert e.value.code == (game.ERR_INVALID_ARG if cfg.P > 256 * 74 else game.OK)
    G.close()


# ------------------------------------------------------------------------------------------------ the paper's fitness 1 - error
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("selection", [0, 1, 2])
def test_one_minus_mse_fitness(game, selection, scheme):
    """GAME_ERROR_ONE_MINUS_MSE (fitness = 1 - error, maximised): fitness_dev = 1 - MSE within 1e-5 of the
    oracle's; the best-fitness trace holds the MAXIMUM; the GA operators are those of the oracle on the error vector
    e = 1 - fitness (ONE fp32 subtraction, the same on both sides), bit for bit, for all three selection methods."""
    import torch
    cfg = wl.scaled(wl.CONFIGS["c1"], P=3000, M=150)
    X, t, _ = wl.make_kb(cfg)
    G = make(game, cfg, scheme); G.load_kb(X, t)
    game.game_set_error_metric(G.ctx, game.ERROR_ONE_MINUS_MSE)
    game.game_set_selection(G.ctx, selection)
    G.init_population(3); G.sync()
    W = G.get_population()
    best = torch.full((3,), float("nan"), dtype=torch.float32, device="cuda")
    G.run(3, 0, 0, best); G.sync()                      # one evaluation through the run loop: best[0]
    F = G.get_fitness()
    ref = 1.0 - oracle.eval_fitness(cfg.d, cfg.family, X, t, W)
    assert np.max(np.abs(F - ref) / ref) <= 1e-5
    assert best.cpu().numpy()[0] == F.max()
    err = (np.float32(1.0) - F).astype(np.float32)
    G.step(3, 0); G.sync()
    W1 = oracle.step_sel(W, err, cfg.elite, cfg.tournament, selection, cfg.p_cross, cfg.p_mut, cfg.sigma, 3, 0)
    assert np.array_equal(G.get_population().view(np.uint32), W1.view(np.uint32))
    # the stop rule is a learning-ERROR threshold: 1 - best <= threshold
    G.set_population(W)
    done = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    tr = torch.full((6,), float("nan"), dtype=torch.float32, device="cuda")
    game.game_run_until(G.ctx, 3, 0, 5, float(1.0 - F.max()) * 1.0000001, tr.data_ptr(), done.data_ptr()); G.sync()
    assert int(done.item()) == 0
    G.close()


# ------------------------------------------------------------------------------------------------ stop rule
@pytest.mark.parametrize("scheme", SCHEMES)
def test_run_until_stop_rule(game, scheme):
    """game_run_until: all generations are enqueued with no host sync; the device flag must freeze the
    population, the fitness and the best trace at the first generation whose best fitness <= threshold -- the same
    generation, population (bit-exact) and trace as the plain device run cut there, and as the oracle's stop rule."""
    import torch
    cfg = wl.scaled(wl.CONFIGS["c0"], P=600, M=48)
    X, t, _ = wl.make_kb(cfg)
    n, seed = 9, 21
    G = make(game, cfg, scheme); G.load_kb(X, t)
    G.init_population(seed)
    plain = torch.full((n + 1,), float("nan"), dtype=torch.float32, device="cuda")
    G.run(seed, 0, n, plain); G.sync()
    plain = plain.cpu().numpy()
    drops = [g for g in range(1, n + 1) if plain[g] < plain[g - 1]]
    assert drops
    g_stop = drops[len(drops) // 2]
    thr = float(plain[g_stop])
    for threshold, expect in ((thr, g_stop), (-1.0, n), (float("inf"), 0)):
        G.init_population(seed)
        best = torch.full((n + 1,), float("nan"), dtype=torch.float32, device="cuda")
        done = torch.full((1,), -7, dtype=torch.int32, device="cuda")
        game.game_run_until(G.ctx, seed, 0, n, threshold, best.data_ptr(), done.data_ptr()); G.sync()
        assert int(done.item()) == expect
        b = best.cpu().numpy()
        assert np.array_equal(b[:expect + 1], plain[:expect + 1]) and np.all(np.isnan(b[expect + 1:]))
        # population and fitness are those of generation `expect`
        G2 = make(game, cfg, scheme); G2.load_kb(X, t); G2.init_population(seed)
        G2.run(seed, 0, expect, None); G2.sync()
        assert np.array_equal(G.get_population().view(np.uint32), G2.get_population().view(np.uint32))
        assert np.array_equal(G.get_fitness(), G2.get_fitness())
        G.step(seed, 99); G.sync()            # the fitness is valid for the final population
        G2.close()
    # against the oracle's stop rule (free-running: same bar as the trajectories)
    W0 = oracle.init_population(cfg.M, cfg.G, seed)
    _, _, b_ref, done_ref = oracle.run_until(cfg.d, cfg.family, X, t, W0, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut,
                                             cfg.sigma, seed, 0, n, thr)
    assert done_ref == g_stop and np.all(np.abs(b_ref - plain[:g_stop + 1]) <= 1e-4 * np.abs(b_ref))
    G.close()


# ------------------------------------------------------------------------------------------------ ranking / roulette
@pytest.mark.parametrize("selection", [1, 2])
@pytest.mark.parametrize("M,N,d,E,pc,pm,sigma,seed,gen", [
    (64, 4, 3, 2, 0.9, 0.05, 0.1, 0, 0), (512, 10, 6, 4, 0.9, 0.2, 0.1, 1, 7), (4096, 32, 10, 2, 0.9, 0.2, 0.1, 3, 19),
    (1500, 7, 3, 0, 1.0, 0.0, 0.0, 2**40 + 1, 5), (33, 2, 1, 32, 0.5, 0.5, 1.0, 9, 2**31 + 3)])
def test_ga_step_ranking_roulette_bit_exact(game, selection, M, N, d, E, pc, pm, sigma, seed, gen):
    """The paper's own selection methods (crossover 0.9, mutation 0.2, elitism 2 are its settings):
    same fitness vector and seed in, bit-identical next population out."""
    rng = np.random.Generator(np.random.Philox(2000 + M + selection))
    G = game.Game(300, N, d, M, wl.EXP_CHEBYSHEV, wl.ACT_SIGMOID)
    W = rng.uniform(-2, 2, size=(M, G.G)).astype(np.float32)
    F = rng.uniform(0, 1.2, size=M).astype(np.float32)            # some fitness above 1: zero roulette weight
    F[rng.integers(0, M, size=max(1, M // 8))] = F[0]
    F[3] = np.nan; F[5] = np.inf; F[6] = -0.0; F[7] = 1e-30
    G.set_ga_params(E, 3, pc, pm, sigma)
    game.game_set_selection(G.ctx, selection)
    G.set_population(W); G.set_fitness(F)
    G.step(seed, gen); G.sync()
    ref = oracle.step_sel(W, F, E, 3, selection, pc, pm, sigma, seed, gen)
    Wn = G.get_population()
    assert np.array_equal(Wn.view(np.uint32), ref.view(np.uint32)), \
        f"{np.count_nonzero(Wn.view(np.uint32) != ref.view(np.uint32))} genes differ"
    if selection == 2:                                            # all weights zero -> uniform parents
        G.set_population(W); G.set_fitness(np.full(M, 2.0, np.float32)); G.step(seed, gen); G.sync()
        ref = oracle.step_sel(W, np.full(M, 2.0, np.float32), E, 3, selection, pc, pm, sigma, seed, gen)
        assert np.array_equal(G.get_population().view(np.uint32), ref.view(np.uint32))
    G.close()


@pytest.mark.parametrize("selection,M,E,R", [(0, 200, 2, 17), (1, 64, 2, 62), (2, 513, 0, 1), (0, 100, 4, 0)])
def test_ga_step_with_random_immigrants_bit_exact(game, selection, M, E, R):
    """Random replacement (R12): the last R child slots are fresh random chromosomes, everything else is
    the plain step; bit-exact against oracle.step_sel + oracle.immigrate."""
    rng = np.random.Generator(np.random.Philox(3000 + M))
    G = game.Game(300, 6, 4, M, wl.EXP_CHEBYSHEV, wl.ACT_SIGMOID)
    W = rng.uniform(-2, 2, size=(M, G.G)).astype(np.float32)
    F = rng.uniform(0, 1, size=M).astype(np.float32)
    G.set_ga_params(E, 3, 0.9, 0.2, 0.1)
    game.game_set_selection(G.ctx, selection)
    game.game_set_immigrants(G.ctx, R)
    with pytest.raises(game.GameError):
        game.game_set_immigrants(G.ctx, M - E + 1)
    G.set_population(W); G.set_fitness(F); G.step(31, 8); G.sync()
    ref = oracle.immigrate(oracle.step_sel(W, F, E, 3, selection, 0.9, 0.2, 0.1, 31, 8), E, R, 31, 8)
    assert np.array_equal(G.get_population().view(np.uint32), ref.view(np.uint32))
    G.close()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_rmse_metric(game, scheme):
    """game_set_error_metric(RMSE): fitness_dev = sqrt(MSE) within 1e-5 of the oracle's RMSE; the GA step on
    it is bit-exact (the operators only see a fitness vector)."""
    cfg = wl.scaled(wl.CONFIGS["c2"], P=2300, M=140)
    X, t, _ = wl.make_kb(cfg)
    W = wl.uniform_population(cfg.M, cfg.G, 14)
    G = make(game, cfg, scheme); G.load_kb(X, t); G.set_population(W)
    game.game_set_error_metric(G.ctx, game.ERROR_RMSE)
    G.eval_fitness(); G.sync()
    F = G.get_fitness()
    assert_fitness_close(F, oracle.eval_rmse(cfg.d, cfg.family, X, t, W), "rmse")
    G.step(3, 1); G.sync()
    ref = oracle.step(W, F, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, 3, 1)
    assert np.array_equal(G.get_population().view(np.uint32), ref.view(np.uint32))
    G.close()


@pytest.mark.parametrize("base,over,selection,immigrants", [
    ("c1", dict(P=1500, M=300), 0, 0), ("c3", dict(P=600, M=257), 1, 5), ("c2", dict(P=900, M=131), 2, 3),
    ("c0", dict(P=300, M=37), 0, 2)])
def test_step_keeps_w_images(game, base, over, selection, immigrants):
    """Inside a generation loop the GA step writes the W operand images of the tensor-core kernel itself (elites,
    children, immigrants), and the next evaluation runs no image pass.  The fitness it then computes must be
    bit-identical to the one computed from images rebuilt from scratch for the same population (set_population
    invalidates them), generation after generation; and it stays within 1e-5 of the oracle."""
    cfg = wl.scaled(wl.CONFIGS[base], **over)
    X, t, _ = wl.make_kb(cfg)
    G = make(game, cfg, game.SCHEME_F16X3); G.load_kb(X, t)
    game.game_set_selection(G.ctx, selection); game.game_set_immigrants(G.ctx, immigrants)
    H = make(game, cfg, game.SCHEME_F16X3); H.load_kb(X, t)       # every evaluation from rebuilt images
    G.init_population(9)
    for gen in range(4):
        n0 = G.launch_count()
        G.eval_fitness(); G.sync()
        cal = 4 if cfg.activation != wl.ACT_SIGMOID else 0        # regression activations: sample gather, calibration launch, cal_phi_kernel, calibrate_kernel
        assert G.launch_count() - n0 == (4 if gen == 0 else 2) + cal   # row scales + image pass only before the first generation
        F = G.get_fitness()
        W = G.get_population()
        H.set_population(W); H.eval_fitness(); H.sync()
        assert np.array_equal(F.view(np.uint32), H.get_fitness().view(np.uint32)), f"generation {gen}"
        G.step(21, gen); G.sync()
    assert_fitness_close(F, oracle.eval_fitness(cfg.d, cfg.family, X, t, W), "after three in-step image updates")
    G.close(); H.close()


@pytest.mark.parametrize("base,over,scheme,selection", [
    ("c0", {}, 2, 0), ("c1", dict(P=6000, M=300), 2, 1), ("c2", dict(P=2500, M=131), 2, 2), ("c1", dict(P=3000, M=64), 1, 0)])
def test_dependent_launch_chain_is_race_free(game, base, over, scheme, selection):
    """The generation's kernels run under programmatic dependent launch (csrc/pdl.cuh): each one is launched while its
    predecessor still runs and parks in griddepcontrol.wait.  A missing or misplaced wait would let a kernel read what its
    predecessor has not written yet, so 40 generations enqueued back to back must give the same populations, fitness
    vectors and best-fitness trace, bit for bit, as the same run with plain stream-ordered launches (game_set_option(GAME_OPT_PDL, 0)).  The same
    holds for the loop replayed from a CUDA graph of 16 generations (GAME_OPT_GRAPH, the default; seed and generation index in
    device memory): 40 = 2 replays + 8 plain generations + the final evaluation."""
    import torch
    cfg = wl.scaled(wl.CONFIGS[base], **over)
    X, t, _ = wl.make_kb(cfg)
    n = 40
    out = []
    for pdl, graph in (("0", "0"), ("1", "0"), ("1", "1"), ("0", "1")):      # plain launches / PDL chain / both replayed from a CUDA graph
        G = make(game, cfg, scheme); G.load_kb(X, t)
        game.game_set_option(G.ctx, game.OPT_PDL, int(pdl)); game.game_set_option(G.ctx, game.OPT_GRAPH, int(graph))
        game.game_set_selection(G.ctx, selection); game.game_set_immigrants(G.ctx, 2)
        best = torch.zeros(n + 1, dtype=torch.float32, device="cuda")
        G.init_population(17); G.run(17, 0, n, best); G.sync()
        out.append((G.get_population().view(np.uint32), G.get_fitness().view(np.uint32), best.cpu().numpy().view(np.uint32)))
        G.close()
    for other in out[1:]:
        for a, b in zip(out[0], other):
            assert np.array_equal(a, b)


def test_caller_rewrites_knowledge_base_on_the_stream(game):
    """include/game.h, game_load_kb: the caller may rewrite the borrowed X / t with work on the context's stream and evaluate
    again, with nothing but stream order in between.  On small grids (c0: 8 CTAs) the fitness kernel's phi producers start
    reading X before griddepcontrol.wait, which is only sound behind one of the library's own kernels -- so the first kernel
    of a public call must not do it.  Here the W images are already valid (no image pass ahead of the fitness kernel) and a
    device-side copy kernel fills X right before game_eval_fitness, on every activation (identity / tanh put the calibration
    launch first instead)."""
    import torch
    for act in (wl.ACT_SIGMOID, wl.ACT_TANH):
        cfg = wl.scaled(wl.CONFIGS["c0"], activation=act)
        X1, t1, _ = wl.make_kb(cfg)
        X2, t2, _ = wl.make_kb(cfg, seed=99)
        G = make(game, cfg, 2); G.load_kb(X1, t1)
        G.init_population(5); G.eval_fitness()                      # builds the W images; fitness over (X1, t1)
        X2d = torch.as_tensor(X2, device="cuda"); t2d = torch.as_tensor(t2, device="cuda")
        big = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
        for rep in range(3):
            src = (X2d, t2d) if rep % 2 == 0 else (torch.as_tensor(X1, device="cuda"), torch.as_tensor(t1, device="cuda"))
            big.zero_()                                             # keeps the stream busy: the copies below are still queued
            G.X.copy_(src[0]); G.t.copy_(src[1])                    # device-side kernels on the context's stream
            G.eval_fitness()                                        # population unchanged: the fitness kernel goes first
            G.sync()
            F_ref = oracle.eval_fitness(cfg.d, cfg.family, X2 if rep % 2 == 0 else X1, t2 if rep % 2 == 0 else t1, G.get_population())
            assert_fitness_close(G.get_fitness(), F_ref, f"act {act} rep {rep}")
        G.close()


# ------------------------------------------------------------------------------------------------ fused persistent loop
@pytest.mark.parametrize("base,over,selection,immigrants", [
    ("c0", {}, 0, 0), ("c0", dict(P=777, M=37), 1, 3), ("n1", {}, 1, 0), ("n1", dict(P=500, M=23), 2, 2),
    ("c1", dict(P=3001, M=50), 0, 0)])
def test_evolve_fused_lockstep_and_determinism(game, base, over, selection, immigrants):
    """game_evolve_fused (one persistent cooperative kernel).  Lock-step, one generation per call: the
    fitness it leaves in fitness_dev is within 1e-5 of the oracle's for the same population and the next population is
    bit-identical to the oracle's step on THAT fitness vector; n generations in one launch == n launches of one."""
    import torch
    cfg = wl.scaled(wl.PAPER_SHAPE if base == "n1" else wl.CONFIGS[base], **over)
    X, t, _ = wl.make_kb(cfg)
    seed, n = 5, 6
    G = make(game, cfg); G.load_kb(X, t)
    game.game_set_selection(G.ctx, selection); game.game_set_immigrants(G.ctx, immigrants)
    G.init_population(seed); G.sync()
    W = G.get_population()
    bests = []
    for g in range(n):
        game.game_evolve_fused(G.ctx, seed, g, 1, None); G.sync()
        F = G.get_fitness()
        assert_fitness_close(F, oracle.eval_fitness(cfg.d, cfg.family, X, t, W), f"fused gen {g}")
        bests.append(F[oracle.best_index(F)])
        W = oracle.immigrate(oracle.step_sel(W, F, cfg.elite, cfg.tournament, selection, cfg.p_cross, cfg.p_mut, cfg.sigma,
                                             seed, g), cfg.elite, immigrants, seed, g)
        assert np.array_equal(G.get_population().view(np.uint32), W.view(np.uint32)), f"population forked at gen {g}"
    with pytest.raises(game.GameError):
        G.step(seed, 0)                                    # the population is one step past its last fitness
    G.init_population(seed)
    best = torch.full((n,), float("nan"), dtype=torch.float32, device="cuda")
    game.game_evolve_fused(G.ctx, seed, 0, n, best.data_ptr()); G.sync()
    assert np.array_equal(G.get_population().view(np.uint32), W.view(np.uint32))
    assert np.array_equal(best.cpu().numpy(), np.asarray(bests, np.float32))
    G.close()


def test_evolve_fused_rejects_big_problems(game):
    G = game.Game(100_000, 10, 6, 512, wl.EXP_CHEBYSHEV, wl.ACT_SIGMOID)
    with pytest.raises(game.GameError) as e:
        game.game_evolve_fused(G.ctx, 1, 0, 1, None)
    assert e.value.code == game.ERR_UNSUPPORTED
    G.close()


# ------------------------------------------------------------------------------------------------ shared coefficients
@pytest.mark.parametrize("scheme", [1, 2])
@pytest.mark.parametrize("expansion,act,N,d,P,M", [(1, 0, 11, 3, 200, 23), (1, 1, 9, 8, 2100, 19), (0, 1, 7, 5, 1500, 40),
                                                    (1, 2, 16, 4, 3001, 130), (0, 2, 5, 33, 700, 300), (1, 1, 3, 32, 900, 70)])
def test_shared_coefficient_mode(game, expansion, act, N, d, P, M, scheme):
    """The paper's literal model (eq.(2),(5),(7): one coefficient per degree for all features; first case = its worked
    example 11 features, degree 3, 7 genes, 23 chromosomes): fitness, prediction, GA step and the fused loop."""
    import torch
    fam = oracle.family(expansion, act, shared=True)
    rng = np.random.Generator(np.random.Philox(50 + N))
    X = rng.uniform(-np.pi, np.pi, (P, N)).astype(np.float32) if expansion == 1 else rng.uniform(-1, 1, (P, N)).astype(np.float32)
    t = (rng.uniform(size=P) > 0.5).astype(np.float32)
    G = game.Game(P, N, d, M, expansion, act, shared=True, scheme=scheme)
    assert G.G == oracle.num_genes(N, d, fam) == (2 * d + 1 if expansion == 1 else d + 1)
    G.set_ga_params(2, 3, 0.9, 0.2, 0.1)
    G.load_kb(X, t); G.init_population(3); G.sync()
    W = G.get_population()
    G.eval_fitness(); G.sync()
    F = G.get_fitness()
    assert_fitness_close(F, oracle.eval_fitness(d, fam, X, t, W), "shared fitness")
    y = torch.empty(P, dtype=torch.float32, device="cuda")
    game.game_predict(G.ctx, G.current()[1].data_ptr(), G.X.data_ptr(), P, y.data_ptr()); G.sync()
    y_ref = oracle.predict(d, fam, X, W[1])
    assert np.max(np.abs(y.cpu().numpy() - y_ref) / np.maximum(1.0, np.abs(y_ref))) <= 1e-5
    G.step(3, 0); G.sync()
    W1 = oracle.step(W, F, 2, 3, 0.9, 0.2, 0.1, 3, 0)
    assert np.array_equal(G.get_population().view(np.uint32), W1.view(np.uint32))
    # fused loop, lock-step
    game.game_evolve_fused(G.ctx, 3, 1, 1, None); G.sync()
    F1 = G.get_fitness()
    assert_fitness_close(F1, oracle.eval_fitness(d, fam, X, t, W1), "shared fused fitness")
    W2 = oracle.step(W1, F1, 2, 3, 0.9, 0.2, 0.1, 3, 1)
    assert np.array_equal(G.get_population().view(np.uint32), W2.view(np.uint32))
    G.close()


# ------------------------------------------------------------------------------------------------ randomised shapes
def test_random_shapes_fitness_and_step(game):
    """Seeded sweep over odd shapes (P, N, d, M not multiples of any tile), both expansions, all activations, all three
    selection methods: fitness within 1e-5 of the oracle on the AUTO scheme, GA step bit-exact."""
    rng = np.random.Generator(np.random.Philox(2026))
    for trial in range(14):
        expansion = int(rng.integers(0, 2))
        act = int(rng.integers(0, 3))
        N = int(rng.integers(1, 41))
        d = int(rng.integers(1, 8 if expansion else 12))
        while N * d * (2 if expansion else 1) + 1 > 440:
            N -= 1
        P = int(rng.integers(1, 4000))
        M = int(rng.integers(2, 420))
        selection = int(rng.integers(0, 3))
        E = int(rng.integers(0, min(M, 6)))
        fam = oracle.family(expansion, act)
        X = rng.uniform(-1, 1, (P, N)).astype(np.float32) * (np.float32(np.pi) if expansion else np.float32(1))
        t = rng.uniform(0, 1, P).astype(np.float32)
        W = (rng.uniform(-1, 1, (M, oracle.num_genes(N, d, fam))) * (0.3 if act == 0 else 1.0)).astype(np.float32)
        G = game.Game(P, N, d, M, expansion, act)
        G.set_ga_params(E, 3, 0.9, 0.2, 0.1)
        game.game_set_selection(G.ctx, selection)
        G.load_kb(X, t); G.set_population(W); G.eval_fitness(); G.sync()
        F = G.get_fitness()
        what = f"trial {trial}: exp {expansion} act {act} P {P} N {N} d {d} M {M}"
        assert_fitness_close(F, oracle.eval_fitness(d, fam, X, t, W), what)
        G.step(trial, trial + 1); G.sync()
        ref = oracle.step_sel(W, F, E, 3, selection, 0.9, 0.2, 0.1, trial, trial + 1)
        assert np.array_equal(G.get_population().view(np.uint32), ref.view(np.uint32)), what
        G.close()


def test_random_shapes_tensor_path_wide(game):
    """Seeded sweep of the tensor-core kernel over the corners the fixed cases do not reach together: shared and
    per-feature coefficients, degrees far beyond a K step, streaming K extents, M and P around the tile edges.  Fitness
    within 1e-5 of the oracle for every activation up to G = 2401 (round 1 had to keep the identity output to G <= 1200: the
    truncating TMEM accumulation; K-chunk flush + calibration close it)."""
    import torch
    rng = np.random.Generator(np.random.Philox(4096))
    done = 0
    while done < 32:
        expansion = int(rng.integers(0, 2)); act = int(rng.integers(0, 3)); shared = bool(rng.integers(0, 3) == 0)
        if shared:
            N = int(rng.integers(1, 20)); d = int(rng.integers(1, 33 if expansion else 65))
        else:
            N = int(rng.integers(1, 60)); d = int(rng.integers(1, 30 if expansion else 80))
            while N * d * (2 if expansion else 1) > 2400:
                N = max(1, N // 2); d = max(1, d - 1)
        P = int(rng.choice([255, 256, 257, 700, 1500, 4000])) + int(rng.integers(0, 3))
        M = int(rng.choice([1, 2, 127, 128, 129, 255, 256, 257, 700, 1300])) + int(rng.integers(0, 2))
        Gn = (1 if shared else N) * d * (2 if expansion else 1) + 1
        if P * M * Gn > 3e8:
            continue
        fam = oracle.family(expansion, act, shared=shared)
        X = (rng.uniform(-np.pi, np.pi, (P, N)) if expansion else rng.uniform(-1, 1, (P, N))).astype(np.float32)
        t = (rng.uniform(size=P) > 0.5).astype(np.float32) if act == 1 else rng.uniform(-1, 1, P).astype(np.float32)
        scale = 1.0 / max(1.0, np.sqrt(Gn / 8.0) * (N if shared else 1) ** 0.5)
        W = (rng.uniform(-1, 1, (M, Gn)) * scale).astype(np.float32)
        G = game.Game(P, N, d, M, expansion, act, shared=shared, scheme=game.SCHEME_F16X3)
        G.load_kb(X, t); G.set_population(torch.from_numpy(W).cuda()); G.eval_fitness(); G.sync()
        F = G.get_fitness()
        G.close()
        assert_fitness_close(F, oracle.eval_fitness(d, fam, X, t, W),
                             f"exp={expansion} act={act} shared={shared} N={N} d={d} P={P} M={M} G={Gn}")
        done += 1
