"""paper_1211_5481_b200 -- thin Python binding of libgame.so (include/game.h).

Argument marshalling only: every step of the GAME hot path (feature expansion, fitness contraction,
activation, error reduction, GA operators, Philox RNG; arXiv:1211.5481) runs in the
CUDA kernels of ``csrc/``.  PyTorch is used for device memory and streams, nothing else.  There is no
CPU fallback: without the built library, or without a CUDA device, calls raise.

The functions mirror the C ABI one to one (same names); :class:`Game` bundles a context with the torch
tensors it borrows so that they stay alive while bound.
"""
from __future__ import annotations

import ctypes as C
import os

EXP_CHEBYSHEV, EXP_TRIG = 0, 1
ACT_IDENTITY, ACT_SIGMOID, ACT_TANH = 0, 1, 2
SCHEME_AUTO, SCHEME_FFMA, SCHEME_F16X3 = 0, 1, 2
SEL_TOURNAMENT, SEL_RANKING, SEL_ROULETTE = 0, 1, 2
ERROR_MSE, ERROR_RMSE, ERROR_ONE_MINUS_MSE = 0, 1, 2
OPT_PDL, OPT_GRAPH, OPT_CALIBRATE, OPT_UNIT_PAIRS = 0, 1, 2, 3
OK, ERR_INVALID_ARG, ERR_BAD_STATE, ERR_CUDA, ERR_WORKSPACE, ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgame.so")

# name -> (restype, argtypes); every symbol include/game.h declares
_VP, _F32P = C.c_void_p, C.c_void_p   # raw addresses (device or host) are passed as integers
SIGNATURES = {
    "game_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int64, C.c_int32, C.c_int32, C.c_int32, C.c_int32]),
    "game_destroy": (C.c_int, [_VP]),
    "game_num_genes": (C.c_int, [_VP, C.POINTER(C.c_int32)]),
    "game_workspace_bytes": (C.c_int, [_VP, C.POINTER(C.c_size_t)]),
    "game_set_stream": (C.c_int, [_VP, _VP]),
    "game_set_scheme": (C.c_int, [_VP, C.c_int32]),
    "game_get_scheme": (C.c_int, [_VP, C.POINTER(C.c_int32)]),
    "game_load_kb": (C.c_int, [_VP, _F32P, _F32P]),
    "game_bind_state": (C.c_int, [_VP, _F32P, _F32P, _F32P, _VP, C.c_size_t]),
    "game_set_ga_params": (C.c_int, [_VP, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_float]),
    "game_set_option": (C.c_int, [_VP, C.c_int32, C.c_int32]),
    "game_set_selection": (C.c_int, [_VP, C.c_int32]),
    "game_set_immigrants": (C.c_int, [_VP, C.c_int32]),
    "game_set_error_metric": (C.c_int, [_VP, C.c_int32]),
    "game_init_population": (C.c_int, [_VP, C.c_uint64]),
    "game_current_population": (C.c_int, [_VP, C.POINTER(C.c_void_p)]),
    "game_invalidate_fitness": (C.c_int, [_VP]),
    "game_assume_fitness": (C.c_int, [_VP]),
    "game_eval_fitness": (C.c_int, [_VP]),
    "game_step": (C.c_int, [_VP, C.c_uint64, C.c_uint32]),
    "game_run": (C.c_int, [_VP, C.c_uint64, C.c_uint32, C.c_uint32, _F32P]),
    "game_run_until": (C.c_int, [_VP, C.c_uint64, C.c_uint32, C.c_uint32, C.c_float, _F32P, _VP]),
    "game_evolve": (C.c_int, [_VP, C.c_uint64, C.c_uint32, C.c_uint32]),
    "game_evolve_fused": (C.c_int, [_VP, C.c_uint64, C.c_uint32, C.c_uint32, _F32P]),
    "game_sync": (C.c_int, [_VP]),
    "game_generation_host": (C.c_int, [_VP, _F32P, _F32P, _F32P, _F32P, _F32P, C.c_uint64, C.c_uint32]),
    "game_eval_fitness_streamed": (C.c_int, [_VP, _F32P, _F32P, _F32P, _F32P, C.c_int64, C.c_int32]),
    "game_eval_sse": (C.c_int, [_VP, _VP]),
    "game_set_fitness_from_sse": (C.c_int, [_VP, _VP, C.c_int64, _F32P]),
    "game_comm_unique_id": (C.c_int, [_VP]),
    "game_comm_init": (C.c_int, [_VP, _VP, C.c_int32, C.c_int32]),
    "game_evolve_sharded": (C.c_int, [_VP, C.c_uint64, C.c_uint32, C.c_uint32, C.c_int64, _F32P]),
    "game_predict": (C.c_int, [_VP, _F32P, _F32P, C.c_int64, _F32P]),
    "game_confusion": (C.c_int, [_VP, _F32P, _F32P, C.c_int64, C.c_float, _VP]),
    "game_launch_count": (C.c_int, [_VP, C.POINTER(C.c_uint64)]),
    "game_graph_replays": (C.c_int, [_VP, C.POINTER(C.c_uint64)]),
    "game_mma_stall": (C.c_int, [_VP, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double), _VP, C.c_int32]),
    "game_time_fitness_kernel": (C.c_int, [_VP, C.c_int32]),
    "game_fitness_kernel_ms": (C.c_int, [_VP, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]),
    "game_calibration_status": (C.c_int, [_VP, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]),
    "game_last_error": (C.c_char_p, [_VP]),
    "game_eval_fitness_noalloc": (C.c_int, [_F32P, _F32P, _F32P, _F32P, C.c_int64, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                            _VP, C.c_char_p, C.c_size_t]),
}
NOALLOC_MAX_M, NOALLOC_MAX_G = 1024, 448   # GAME_NOALLOC_MAX_M / _G of include/game.h

_lib = None


class GameError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"libgame error {code}: {message}")
        self.code = code


def lib() -> C.CDLL:
    """Load libgame.so (fails loudly if it has not been built: ``python -m paper_1211_5481_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1211_5481_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def family(expansion: int, activation: int, shared: bool = False) -> int:
    return expansion | (activation << 8) | (int(shared) << 16)


def _check(ctx, rc: int) -> None:
    if rc != OK:
        msg = lib().game_last_error(ctx)
        raise GameError(rc, msg.decode() if msg else "")


# ---- one-to-one wrappers (same names as the C ABI) -------------------------------------------------------
def game_create(P: int, N: int, d: int, M: int, fam: int):
    ctx = C.c_void_p()
    rc = lib().game_create(C.byref(ctx), P, N, d, M, fam)
    if rc != OK:
        raise GameError(rc, "game_create rejected the shapes")
    return ctx


def game_destroy(ctx) -> None:
    lib().game_destroy(ctx)


def game_num_genes(ctx) -> int:
    g = C.c_int32()
    _check(ctx, lib().game_num_genes(ctx, C.byref(g)))
    return g.value


def game_workspace_bytes(ctx) -> int:
    b = C.c_size_t()
    _check(ctx, lib().game_workspace_bytes(ctx, C.byref(b)))
    return b.value


def game_set_stream(ctx, cuda_stream: int) -> None:
    _check(ctx, lib().game_set_stream(ctx, cuda_stream))


def game_set_scheme(ctx, scheme: int) -> None:
    _check(ctx, lib().game_set_scheme(ctx, scheme))


def game_get_scheme(ctx) -> int:
    s = C.c_int32()
    _check(ctx, lib().game_get_scheme(ctx, C.byref(s)))
    return s.value


def game_load_kb(ctx, X_dev: int, t_dev: int) -> None:
    _check(ctx, lib().game_load_kb(ctx, X_dev, t_dev))


def game_bind_state(ctx, popA_dev: int, popB_dev: int, fitness_dev: int, workspace_dev: int, workspace_bytes: int) -> None:
    _check(ctx, lib().game_bind_state(ctx, popA_dev, popB_dev, fitness_dev, workspace_dev, workspace_bytes))


def game_set_ga_params(ctx, elite: int, tournament: int, p_cross: float, p_mut: float, sigma: float) -> None:
    _check(ctx, lib().game_set_ga_params(ctx, elite, tournament, p_cross, p_mut, sigma))


def game_set_error_metric(ctx, metric: int) -> None:
    _check(ctx, lib().game_set_error_metric(ctx, metric))


def game_set_immigrants(ctx, immigrants: int) -> None:
    _check(ctx, lib().game_set_immigrants(ctx, immigrants))


def game_set_option(ctx, option: int, value: int) -> None:
    _check(ctx, lib().game_set_option(ctx, option, value))


def game_set_selection(ctx, selection: int) -> None:
    _check(ctx, lib().game_set_selection(ctx, selection))


def game_init_population(ctx, seed: int) -> None:
    _check(ctx, lib().game_init_population(ctx, seed))


def game_current_population(ctx) -> int:
    p = C.c_void_p()
    _check(ctx, lib().game_current_population(ctx, C.byref(p)))
    return p.value


def game_invalidate_fitness(ctx) -> None:
    _check(ctx, lib().game_invalidate_fitness(ctx))


def game_assume_fitness(ctx) -> None:
    _check(ctx, lib().game_assume_fitness(ctx))


def game_eval_fitness(ctx) -> None:
    _check(ctx, lib().game_eval_fitness(ctx))


def game_step(ctx, seed: int, gen: int) -> None:
    _check(ctx, lib().game_step(ctx, seed, gen))


def game_run(ctx, seed: int, gen0: int, n_gens: int, best_fitness_dev: int | None) -> None:
    _check(ctx, lib().game_run(ctx, seed, gen0, n_gens, best_fitness_dev))


def game_run_until(ctx, seed: int, gen0: int, max_gens: int, threshold: float, best_fitness_dev: int,
                   gens_done_dev: int) -> None:
    _check(ctx, lib().game_run_until(ctx, seed, gen0, max_gens, threshold, best_fitness_dev, gens_done_dev))


def game_evolve(ctx, seed: int, gen0: int, n_gens: int) -> None:
    _check(ctx, lib().game_evolve(ctx, seed, gen0, n_gens))


def game_evolve_fused(ctx, seed: int, gen0: int, n_gens: int, best_fitness_dev: int | None = None) -> None:
    _check(ctx, lib().game_evolve_fused(ctx, seed, gen0, n_gens, best_fitness_dev))


def game_sync(ctx) -> None:
    _check(ctx, lib().game_sync(ctx))


def game_generation_host(ctx, X_host: int, t_host: int, W_host: int, F_host: int | None, W_next_host: int | None,
                         seed: int, gen: int) -> None:
    _check(ctx, lib().game_generation_host(ctx, X_host, t_host, W_host, F_host, W_next_host, seed, gen))


def game_eval_fitness_streamed(ctx, X_host: int, t_host: int, X_ring_dev: int, t_ring_dev: int, slot_rows: int, n_slots: int) -> None:
    _check(ctx, lib().game_eval_fitness_streamed(ctx, X_host, t_host, X_ring_dev, t_ring_dev, slot_rows, n_slots))


def game_eval_sse(ctx, sse_dev: int) -> None:
    _check(ctx, lib().game_eval_sse(ctx, sse_dev))


def game_set_fitness_from_sse(ctx, sse_dev: int, P_total: int, best_fitness_dev: int | None = None) -> None:
    _check(ctx, lib().game_set_fitness_from_sse(ctx, sse_dev, P_total, best_fitness_dev))


def game_comm_unique_id() -> bytes:
    buf = C.create_string_buffer(128)
    rc = lib().game_comm_unique_id(buf)
    if rc != OK:
        raise GameError(rc, "game_comm_unique_id: NCCL unavailable")
    return buf.raw


def game_comm_init(ctx, id128: bytes, rank: int, world: int) -> None:
    buf = C.create_string_buffer(bytes(id128), 128)
    _check(ctx, lib().game_comm_init(ctx, buf, rank, world))


def game_evolve_sharded(ctx, seed: int, gen0: int, n_gens: int, P_total: int, best_fitness_dev: int | None = None) -> None:
    _check(ctx, lib().game_evolve_sharded(ctx, seed, gen0, n_gens, P_total, best_fitness_dev))


def game_predict(ctx, w_dev: int, X_dev: int, Q: int, y_dev: int) -> None:
    _check(ctx, lib().game_predict(ctx, w_dev, X_dev, Q, y_dev))


def game_confusion(ctx, y_dev: int, t_dev: int, Q: int, threshold: float, counts_dev: int) -> None:
    _check(ctx, lib().game_confusion(ctx, y_dev, t_dev, Q, threshold, counts_dev))


def game_launch_count(ctx) -> int:
    n = C.c_uint64()
    _check(ctx, lib().game_launch_count(ctx, C.byref(n)))
    return n.value


def game_mma_stall(ctx, raw=None):
    """(a_full, b_full, acc_empty) wait shares of the MMA warp in the last tensor-core fitness launch; `raw`: optional
    numpy int64 array that receives the per-CTA records."""
    a, b, e = C.c_double(), C.c_double(), C.c_double()
    _check(ctx, lib().game_mma_stall(ctx, C.byref(a), C.byref(b), C.byref(e), None if raw is None else raw.ctypes.data,
                                     0 if raw is None else raw.size))
    return a.value, b.value, e.value


def game_graph_replays(ctx) -> int:
    n = C.c_uint64()
    _check(ctx, lib().game_graph_replays(ctx, C.byref(n)))
    return n.value


def game_time_fitness_kernel(ctx, enable: bool) -> None:
    _check(ctx, lib().game_time_fitness_kernel(ctx, int(enable)))


def game_fitness_kernel_ms(ctx):
    ms, n = C.c_double(), C.c_uint64()
    _check(ctx, lib().game_fitness_kernel_ms(ctx, C.byref(ms), C.byref(n)))
    return ms.value, n.value


def game_calibration_status(ctx):
    """(active, rows_rejected) of the tensor-core scheme's per-row calibration; see include/game.h."""
    a, r = C.c_int32(), C.c_int32()
    _check(ctx, lib().game_calibration_status(ctx, C.byref(a), C.byref(r)))
    return bool(a.value), r.value


def game_last_error(ctx) -> str:
    msg = lib().game_last_error(ctx)
    return msg.decode() if msg else ""


def game_eval_fitness_noalloc(X_dev: int, t_dev: int, W_dev: int, fitness_dev: int, P: int, N: int, d: int, M: int, fam: int,
                              cuda_stream: int | None = None) -> None:
    """MSE fitness of W_dev[M][G] over X_dev[P][N], t_dev[P] into fitness_dev[M] without a context, a workspace or any
    device allocation: the scratch is a fixed 4.25 MiB array inside libgame.so (M <= 1024, G <= 448; one per GPU, shared
    by all calls, so keep the calls for a device on one stream).  Meant for callers who are handed their buffers and
    cannot allocate -- see include/game.h.  Raises GameError with the library's message (limits included)."""
    buf = C.create_string_buffer(256)
    rc = lib().game_eval_fitness_noalloc(X_dev, t_dev, W_dev, fitness_dev, P, N, d, M, fam, cuda_stream, buf, len(buf))
    if rc != OK:
        raise GameError(rc, buf.value.decode())


# ---- convenience: a context plus the torch tensors it borrows ---------------------------------------------
class Game:
    """Owns the device tensors a ``game_ctx`` borrows (knowledge base, two populations, fitness, workspace).

    Marshalling only -- every method is one C-ABI call (plus torch copies for upload / download).
    """

    def __init__(self, P: int, N: int, d: int, M: int, expansion: int, activation: int, device="cuda:0",
                 scheme: int = SCHEME_AUTO, shared: bool = False, resident_kb: bool = True):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1211_5481_b200 needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.device = torch.device(device)
        self.P, self.N, self.d, self.M = P, N, d, M
        self.ctx = game_create(P, N, d, M, family(expansion, activation, shared))
        self.G = game_num_genes(self.ctx)
        with torch.cuda.device(self.device):
            # resident_kb = False: the knowledge base stays in host memory (game_eval_fitness_streamed), nothing of size P
            # is allocated on the device
            self.X = torch.empty((P, N), dtype=torch.float32, device=self.device) if resident_kb else None
            self.t = torch.empty((P,), dtype=torch.float32, device=self.device) if resident_kb else None
            self.pop = [torch.zeros((M, self.G), dtype=torch.float32, device=self.device) for _ in range(2)]
            self.fitness = torch.zeros((M,), dtype=torch.float32, device=self.device)
            self.ws_bytes = game_workspace_bytes(self.ctx)
            self.workspace = torch.empty((self.ws_bytes,), dtype=torch.uint8, device=self.device)
            game_set_stream(self.ctx, torch.cuda.current_stream(self.device).cuda_stream)
        if resident_kb:
            game_load_kb(self.ctx, self.X.data_ptr(), self.t.data_ptr())
        game_bind_state(self.ctx, self.pop[0].data_ptr(), self.pop[1].data_ptr(), self.fitness.data_ptr(),
                        self.workspace.data_ptr(), self.ws_bytes)
        if scheme != SCHEME_AUTO:
            game_set_scheme(self.ctx, scheme)

    def close(self) -> None:
        if getattr(self, "ctx", None) is not None:
            self.torch.cuda.synchronize(self.device)
            game_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # knowledge base / population transfer (plain torch copies into the borrowed buffers)
    def load_kb(self, X, t) -> None:
        torch = self.torch
        self.X.copy_(torch.as_tensor(X, dtype=torch.float32).reshape(self.P, self.N), non_blocking=False)
        self.t.copy_(torch.as_tensor(t, dtype=torch.float32).reshape(self.P), non_blocking=False)
        game_invalidate_fitness(self.ctx)

    def current(self):
        ptr = game_current_population(self.ctx)
        return self.pop[0] if ptr == self.pop[0].data_ptr() else self.pop[1]

    def set_population(self, W) -> None:
        torch = self.torch
        self.current().copy_(torch.as_tensor(W, dtype=torch.float32).reshape(self.M, self.G))
        game_invalidate_fitness(self.ctx)

    def get_population(self):
        return self.current().detach().cpu().numpy().copy()

    def set_fitness(self, F) -> None:
        torch = self.torch
        self.fitness.copy_(torch.as_tensor(F, dtype=torch.float32).reshape(self.M))
        game_assume_fitness(self.ctx)

    def get_fitness(self):
        return self.fitness.detach().cpu().numpy().copy()

    # the C-ABI calls
    def set_ga_params(self, elite, tournament, p_cross, p_mut, sigma) -> None:
        game_set_ga_params(self.ctx, elite, tournament, p_cross, p_mut, sigma)

    def set_scheme(self, scheme: int) -> None:
        game_set_scheme(self.ctx, scheme)

    def scheme(self) -> int:
        return game_get_scheme(self.ctx)

    def init_population(self, seed: int) -> None:
        game_init_population(self.ctx, seed)

    def eval_fitness(self) -> None:
        game_eval_fitness(self.ctx)

    def step(self, seed: int, gen: int) -> None:
        game_step(self.ctx, seed, gen)

    def run(self, seed: int, gen0: int, n_gens: int, best=None) -> None:
        game_run(self.ctx, seed, gen0, n_gens, None if best is None else best.data_ptr())

    def sync(self) -> None:
        game_sync(self.ctx)

    def launch_count(self) -> int:
        return game_launch_count(self.ctx)
