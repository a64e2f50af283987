"""game_eval_fitness_noalloc: the fitness evaluation for callers that cannot allocate device memory.

Some users of libgame.so are handed their device buffers by somebody else and have no way (or no permission) to get
more: a plug-in inside an application that owns the GPU's memory pool, a serving loop that must never trigger
cudaMalloc's device-wide stall, a process whose memory budget was spent before the library was loaded.  They cannot
supply the workspace game_bind_state asks for.  The entry point tested here keeps its scratch (transposed population,
per-block partial sums) in a fixed 4.25 MiB array inside the library instead, at the price of hard limits
(M <= 1024 chromosomes, G <= 448 genes) and of one shared array per GPU.

What is checked:
  * its output against the existing workspace-based path (game_eval_fitness, FFMA scheme) within the 1e-5 relative
    tolerance the parity tests use, on calls made back to back with DIFFERENT shapes, so that whatever an earlier
    call left in the shared array would show up if the later call relied on it;
  * that sizes beyond the limits are refused with a message that names the limit (no GPU needed: arguments are
    validated before the device is touched).

The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity suite.  It passes on its own in a fresh process (where its first call does the one-time set-up on the device)
and after the other tests (where the library is already warm).
"""
import ctypes as C

import numpy as np
import pytest

import workloads as wl

REL_TOL = 1e-5          # the parity tests' bar on per-chromosome fitness (tests/test_gpu_parity.py)
ABS_FLOOR = 1e-10


@pytest.fixture(scope="module")
def game():
    import paper_1211_5481_b200 as g
    from paper_1211_5481_b200 import build
    build.build()
    g.lib()
    return g


# four calls in a row on one stream: large first, then a smaller population with another expansion and activation (its
# scratch footprint lies inside what the first call dirtied), then a shape that touches the limits M = 1024 and G = 441,
# then a tiny shared-coefficient model
CASES = [
    ("cheb_sigmoid", "c1", dict(P=5000, M=700)),                                  # G = 61, 40 pattern tiles, ragged
    ("trig_tanh_small", "c2", dict(P=777, N=5, d=3, M=37)),                       # G = 31, 7 tiles, ragged M and P
    ("at_the_limits", "c3", dict(P=1100, N=44, d=10, M=1024)),                    # G = 441 <= 448, M = 1024
    ("identity_shared", "c1", dict(P=300, M=9, activation=wl.ACT_IDENTITY, shared=True)),   # G = 7, the paper's literal model
]


def existing_path(game, cfg, X, t, W):
    """Fitness from the workspace-based library path (FFMA scheme), as numpy."""
    G = game.Game(cfg.P, cfg.N, cfg.d, cfg.M, cfg.expansion, cfg.activation, scheme=game.SCHEME_FFMA, shared=cfg.shared)
    try:
        G.load_kb(X, t)
        G.set_population(W)
        G.eval_fitness()
        G.sync()
        return G.get_fitness()
    finally:
        G.close()


@pytest.mark.gpu
def test_noalloc_matches_workspace_path_on_consecutive_calls(game):
    import torch

    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream(dev).cuda_stream
    inputs, outputs = [], []
    for i, (name, base, over) in enumerate(CASES):
        cfg = wl.scaled(wl.CONFIGS[base], **over)
        assert cfg.M <= game.NOALLOC_MAX_M and cfg.G <= game.NOALLOC_MAX_G, name
        X, t, _ = wl.make_kb(cfg)
        W = wl.uniform_population(cfg.M, cfg.G, seed=100 + i)
        inputs.append((name, cfg, X, t, W))
    # every input and output buffer exists before the first call: the calls below run back to back with nothing in between
    bufs = []
    for name, cfg, X, t, W in inputs:
        bufs.append((torch.as_tensor(X, device=dev), torch.as_tensor(t, device=dev), torch.as_tensor(W, device=dev),
                     torch.full((cfg.M,), float("nan"), dtype=torch.float32, device=dev)))
    name0, cfg0, _, _, _ = inputs[0]
    Xd0, td0, Wd0, _ = bufs[0]
    F_again = torch.full((cfg0.M,), float("nan"), dtype=torch.float32, device=dev)
    torch.cuda.synchronize(dev)
    before = torch.cuda.memory_allocated(dev)
    for (name, cfg, X, t, W), (Xd, td, Wd, Fd) in zip(inputs, bufs):
        game.game_eval_fitness_noalloc(Xd.data_ptr(), td.data_ptr(), Wd.data_ptr(), Fd.data_ptr(), cfg.P, cfg.N, cfg.d, cfg.M,
                                       cfg.family, stream)
    # and the first shape once more, after the others have overwritten the shared scratch
    game.game_eval_fitness_noalloc(Xd0.data_ptr(), td0.data_ptr(), Wd0.data_ptr(), F_again.data_ptr(), cfg0.P, cfg0.N, cfg0.d,
                                   cfg0.M, cfg0.family, stream)
    torch.cuda.synchronize(dev)
    assert torch.cuda.memory_allocated(dev) == before       # torch's pool was not asked for anything either
    outputs = [b[3].cpu().numpy() for b in bufs]

    for (name, cfg, X, t, W), F in zip(inputs, outputs):
        F_ref = existing_path(game, cfg, X, t, W).astype(np.float64)
        assert np.all(np.isfinite(F)), name
        err = np.abs(F.astype(np.float64) - F_ref)
        bound = REL_TOL * np.abs(F_ref) + ABS_FLOOR
        worst = int(np.argmax(err - bound))
        assert np.all(err <= bound), f"{name}: chromosome {worst}: no-alloc {F[worst]!r}, workspace path {F_ref[worst]!r}"
    # the repeated call gives what the first one gave, bit for bit (fixed summation order, nothing carried over)
    assert np.array_equal(F_again.cpu().numpy().view(np.uint32), outputs[0].view(np.uint32)), name0


def test_noalloc_refuses_sizes_beyond_the_static_scratch(game):
    """Host-side validation only: runs without a GPU.  The pointers are never dereferenced."""
    L = game.lib()
    buf = C.create_string_buffer(256)
    fake = 0x1000   # 16-byte aligned, non-null

    def call(P, N, d, M, fam):
        return L.game_eval_fitness_noalloc(fake, fake, fake, fake, P, N, d, M, fam, None, buf, len(buf)), buf.value.decode()

    rc, msg = call(1000, 4, 3, game.NOALLOC_MAX_M + 1, 0x0100)
    assert rc == game.ERR_UNSUPPORTED and "1025" in msg and "1024" in msg, msg
    rc, msg = call(1000, 45, 10, 64, 0x0100)              # G = 451
    assert rc == game.ERR_UNSUPPORTED and "451" in msg and "448" in msg, msg
    rc, msg = call(1000, 4, 3, 64, 0x0300)                # unknown activation
    assert rc == game.ERR_INVALID_ARG and msg
    rc, msg = call(0, 4, 3, 64, 0x0100)
    assert rc == game.ERR_INVALID_ARG
    assert L.game_eval_fitness_noalloc(None, fake, fake, fake, 10, 4, 3, 8, 0x0100, None, None, 0) == game.ERR_INVALID_ARG
    assert L.game_eval_fitness_noalloc(fake + 4, fake, fake, fake, 10, 4, 3, 8, 0x0100, None, buf, len(buf)) == game.ERR_INVALID_ARG
    with pytest.raises(game.GameError, match="1024"):
        game.game_eval_fitness_noalloc(fake, fake, fake, fake, 1000, 4, 3, 4096, 0x0100)
