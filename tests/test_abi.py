"""CPU-side checks of the C-ABI boundary (no GPU, no compute calls): the library builds for sm_100a,
loads, exports every symbol include/game.h declares, validates arguments, enforces the call-order state
machine, and fails loudly (GAME_ERR_CUDA) instead of falling back when there is no device."""
import ctypes as C
import os
import re

import pytest

import paper_1211_5481_b200 as game
from paper_1211_5481_b200 import build as game_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    game_build.build()
    return game.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "game.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(game_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_all_exported_and_bound(L):
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"libgame.so does not export {n}"
    assert sorted(game.SIGNATURES) == names, "binding and header disagree on the symbol list"
    for n in names:
        assert callable(getattr(game, n)), f"python binding lacks {n}"


def test_no_oracle_or_cpu_fallback_in_product():
    """The product path must not import or link the oracle (tests/, smoke and bench's cpu legs only)."""
    pkg = os.path.join(ROOT, "paper_1211_5481_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "game_oracle" not in src, f


def test_num_genes_matches_baseline_configs(L):
    # tests/golden/baseline_gene_counts.txt: BASELINE.json configs c0..c4 -> 13, 61, 129, 321, 121
    rows = [l.split() for l in open(os.path.join(ROOT, "tests", "golden", "baseline_gene_counts.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 5
    for name, N, d, expansion, G in rows:
        ctx = game.game_create(1000, int(N), int(d), 64, game.family(int(expansion), game.ACT_SIGMOID))
        assert game.game_num_genes(ctx) == int(G), name
        assert game.game_workspace_bytes(ctx) > 0
        game.game_destroy(ctx)


@pytest.mark.parametrize("args", [
    (0, 4, 3, 64, 0x0100), (10, 0, 3, 64, 0x0100), (10, 4, 0, 64, 0x0100), (10, 4, 3, 0, 0x0100),
    (10, 4, 3, 64, 0x0002), (10, 4, 3, 64, 0x0300), (10, 4, 3, 64, 0x20100),
])
def test_create_rejects_bad_shapes(L, args):
    ctx = C.c_void_p()
    assert L.game_create(C.byref(ctx), *args) == game.ERR_INVALID_ARG
    assert ctx.value is None


def test_create_unsupported_gene_count(L):
    ctx = C.c_void_p()
    assert L.game_create(C.byref(ctx), 10, 2, 200, 8, 0x0101) == game.ERR_UNSUPPORTED   # trig d > 128 and G = 801 > 448
    assert L.game_create(C.byref(ctx), 10, 10, 70, 8, 0x0100) == game.OK                # Chebyshev: any degree, G = 701
    game.game_destroy(ctx)
    assert L.game_create(C.byref(ctx), 10, 64, 10, 8, 0x0100) == game.OK                # G = 641: tensor-core kernel
    game.game_destroy(ctx)


def test_scheme_resolution(L):
    ctx = game.game_create(1000, 32, 10, 4096, 0x0100)
    assert game.game_get_scheme(ctx) == game.SCHEME_F16X3
    game.game_set_scheme(ctx, game.SCHEME_FFMA)
    assert game.game_get_scheme(ctx) == game.SCHEME_FFMA
    game.game_destroy(ctx)
    ctx = game.game_create(1000, 1, 200, 64, 0x0101)          # trig d > 128 (G = 401): tensor-core kernel does not cover it
    assert game.game_get_scheme(ctx) == game.SCHEME_FFMA
    with pytest.raises(game.GameError) as e:
        game.game_set_scheme(ctx, game.SCHEME_F16X3)
    assert e.value.code == game.ERR_UNSUPPORTED
    game.game_destroy(ctx)
    ctx = game.game_create(1000, 64, 10, 64, 0x0100)          # G = 641: only the tensor-core kernel covers it
    assert game.game_get_scheme(ctx) == game.SCHEME_F16X3
    with pytest.raises(game.GameError) as e:
        game.game_set_scheme(ctx, game.SCHEME_FFMA)
    assert e.value.code == game.ERR_UNSUPPORTED
    game.game_destroy(ctx)


def test_ga_param_validation_and_state_machine(L):
    ctx = game.game_create(1000, 4, 3, 64, 0x0100)
    for bad in [(-1, 3, .9, .05, .1), (64, 3, .9, .05, .1), (2, 0, .9, .05, .1), (2, 3, 1.5, .05, .1),
                (2, 3, .9, -0.1, .1), (2, 3, .9, .05, -1.0), (2, 3, .9, .05, float("nan")), (2, 3, float("nan"), .05, .1)]:
        with pytest.raises(game.GameError) as e:
            game.game_set_ga_params(ctx, *bad)
        assert e.value.code == game.ERR_INVALID_ARG, bad
    game.game_set_ga_params(ctx, 0, 1, 0.0, 1.0, 0.0)
    # call order: nothing bound yet
    for fn in (game.game_eval_fitness, lambda c: game.game_step(c, 1, 0), lambda c: game.game_init_population(c, 1),
               game.game_current_population, lambda c: game.game_run(c, 1, 0, 2, None)):
        with pytest.raises(game.GameError) as e:
            fn(ctx)
        assert e.value.code == game.ERR_BAD_STATE
    # alignment and workspace size
    with pytest.raises(game.GameError) as e:
        game.game_load_kb(ctx, 0x1004, 0x2000)
    assert e.value.code == game.ERR_INVALID_ARG
    with pytest.raises(game.GameError) as e:
        game.game_bind_state(ctx, 0x10000, 0x20000, 0x30000, 0x40000, 16)
    assert e.value.code == game.ERR_WORKSPACE
    with pytest.raises(game.GameError) as e:
        game.game_bind_state(ctx, 0x10000, 0x10000, 0x30000, 0x40000, 1 << 30)
    assert e.value.code == game.ERR_INVALID_ARG
    game.game_destroy(ctx)


def test_fails_loudly_without_a_device(L):
    """No CPU fallback: with (fake) buffers bound, a compute call on a box without a GPU is GAME_ERR_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    ctx = game.game_create(1000, 4, 3, 64, 0x0100)
    game.game_load_kb(ctx, 0x100000, 0x200000)
    game.game_bind_state(ctx, 0x300000, 0x400000, 0x500000, 0x600000, game.game_workspace_bytes(ctx))
    for fn in (game.game_eval_fitness, lambda c: game.game_init_population(c, 1)):
        with pytest.raises(game.GameError) as e:
            fn(ctx)
        assert e.value.code == game.ERR_CUDA
    with pytest.raises(game.GameError) as e:          # step needs a fitness first
        game.game_step(ctx, 1, 0)
    assert e.value.code == game.ERR_BAD_STATE
    game.game_destroy(ctx)
    with pytest.raises(RuntimeError):
        game.Game(1000, 4, 3, 64, 0, 1)


def test_shared_family_gene_counts(L):
    """The paper's literal form (eq.(5), 84-89): 11 features, degree 3, polytrigo -> 7 genes."""
    ctx = game.game_create(200, 11, 3, 23, game.family(game.EXP_TRIG, game.ACT_IDENTITY, shared=True))
    assert game.game_num_genes(ctx) == 7 and game.game_get_scheme(ctx) == game.SCHEME_F16X3
    game.game_set_scheme(ctx, game.SCHEME_FFMA)
    assert game.game_get_scheme(ctx) == game.SCHEME_FFMA
    game.game_destroy(ctx)
    ctx = game.game_create(200, 11, 40, 23, game.family(game.EXP_TRIG, game.ACT_IDENTITY, shared=True))   # 80 terms > 64
    assert game.game_num_genes(ctx) == 81 and game.game_get_scheme(ctx) == game.SCHEME_FFMA
    with pytest.raises(game.GameError):
        game.game_set_scheme(ctx, game.SCHEME_F16X3)
    game.game_destroy(ctx)
    ctx = game.game_create(200, 11, 3, 23, game.family(game.EXP_CHEBYSHEV, game.ACT_SIGMOID, shared=True))
    assert game.game_num_genes(ctx) == 4
    game.game_destroy(ctx)


def test_round2_entry_points_validate_arguments_without_a_device(L):
    """The entry points added in round 2 (out-of-core evaluation, sharded loop, metric, diagnostics): argument and state
    checks come before any device work, so they can be exercised here."""
    ctx = game.game_create(100_000, 8, 4, 300, game.family(game.EXP_CHEBYSHEV, game.ACT_SIGMOID))
    host = (C.c_float * 64)()
    p = C.addressof(host)
    p16 = (p + 15) & ~15
    # streamed evaluation: null pointers, slot size not a multiple of 256, slot count out of range, unaligned ring
    assert L.game_eval_fitness_streamed(ctx, None, p16, p16, p16, 512, 2) == game.ERR_INVALID_ARG
    assert L.game_eval_fitness_streamed(ctx, p16, p16, p16, p16, 500, 2) == game.ERR_INVALID_ARG
    assert L.game_eval_fitness_streamed(ctx, p16, p16, p16, p16, 512, 1) == game.ERR_INVALID_ARG
    assert L.game_eval_fitness_streamed(ctx, p16, p16, p16, p16, 512, 9) == game.ERR_INVALID_ARG
    assert L.game_eval_fitness_streamed(ctx, p16, p16, p16 + 4, p16, 512, 2) == game.ERR_INVALID_ARG
    assert L.game_eval_fitness_streamed(ctx, p16, p16, p16, p16, 512, 2) == game.ERR_BAD_STATE          # before game_bind_state
    # error metric: the paper's fitness 1 - MSE is accepted, anything else is not
    for metric, rc in ((game.ERROR_MSE, game.OK), (game.ERROR_RMSE, game.OK), (game.ERROR_ONE_MINUS_MSE, game.OK), (3, game.ERR_INVALID_ARG),
                       (-1, game.ERR_INVALID_ARG)):
        assert L.game_set_error_metric(ctx, metric) == rc
    # sharded loop: needs a communicator; the communicator needs bound buffers (their device)
    assert L.game_evolve_sharded(ctx, 1, 0, 2, 100_000, None) == game.ERR_BAD_STATE
    ident = (C.c_char * 128)()
    assert L.game_comm_init(ctx, None, 0, 1) == game.ERR_INVALID_ARG
    assert L.game_comm_init(ctx, ident, 2, 2) == game.ERR_INVALID_ARG
    assert L.game_comm_init(ctx, ident, 0, 1) in (game.ERR_BAD_STATE, game.ERR_UNSUPPORTED)            # not bound / no NCCL here
    assert L.game_comm_unique_id(None) == game.ERR_INVALID_ARG
    # diagnostics
    n = C.c_uint64(7)
    assert L.game_graph_replays(ctx, C.byref(n)) == game.OK and n.value == 0
    a, b, e = C.c_double(), C.c_double(), C.c_double()
    assert L.game_mma_stall(ctx, C.byref(a), C.byref(b), C.byref(e), None, 0) == game.ERR_BAD_STATE
    assert L.game_mma_stall(ctx, None, C.byref(b), C.byref(e), None, 0) == game.ERR_INVALID_ARG
    game.game_destroy(ctx)


def test_set_option_validation(L):
    """game_set_option: the documented switches (no environment variables are read), unknown options and bad values rejected."""
    ctx = game.game_create(1000, 10, 6, 64, game.family(game.EXP_CHEBYSHEV, game.ACT_TANH))
    for opt in (game.OPT_PDL, game.OPT_GRAPH, game.OPT_CALIBRATE):
        for v in (0, 1):
            assert L.game_set_option(ctx, opt, v) == game.OK
    assert L.game_set_option(ctx, game.OPT_UNIT_PAIRS, 2) == game.OK
    assert L.game_set_option(ctx, game.OPT_UNIT_PAIRS, 0) == game.OK
    assert L.game_set_option(ctx, game.OPT_UNIT_PAIRS, -1) == game.ERR_INVALID_ARG
    assert L.game_set_option(ctx, 99, 1) == game.ERR_INVALID_ARG and b"99" in L.game_last_error(ctx)
    assert L.game_set_option(None, game.OPT_PDL, 1) == game.ERR_INVALID_ARG
    game.game_destroy(ctx)
    src = open(os.path.join(ROOT, "paper_1211_5481_b200", "csrc", "game_api.cu")).read()
    assert "getenv" not in src
