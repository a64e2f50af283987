"""N > 1 host logic on CPU (gloo, world_size 2): max-over-ranks timing, whole-job value, the replica
knowledge-base seeds, the pattern-shard helper, and the reference arm under torchrun (rank 0 prints, the
other ranks exit 0 without work)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")
    cfg = wl.scaled(wl.CONFIGS["c0"], P=64)
    X, _, _ = wl.make_kb(cfg, seed=cfg.seed + 1000 * rank)
    sums = torch.tensor([float(X.sum())], dtype=torch.float64)
    gathered = [torch.zeros_like(sums) for _ in range(world)]
    dist.all_gather(gathered, sums)
    if rank == 0:
        json.dump({"ms": ms, "value": bench.job_value(1000, 64, 4, world, ms), "sums": [float(g) for g in gathered]},
                  open(out, "w"))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_gloo(tmp_path):
    out = str(tmp_path / "r.json")
    mp.spawn(_worker, args=(2, 29533, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["ms"] == 15.0                                   # slowest rank
    assert r["value"] == 1000 * 64 * 4 * 2 / 15e-3           # units of ALL ranks / max time
    assert r["sums"][0] != r["sums"][1]                      # every replica has its own knowledge base


def test_shard_patterns_partition():
    for P, w in [(10, 3), (1000, 2), (7, 8), (4_000_000, 8)]:
        edges = [wl.shard_patterns(P, w, r) for r in range(w)]
        assert edges[0][0] == 0 and edges[-1][1] == P
        assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
        sizes = [b - a for a, b in edges]
        assert max(sizes) - min(sizes) <= 1


def test_reference_arm_under_torchrun_rank0_only():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
           "127.0.0.1", "--master-port", "29534", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--workload", "c0", "--steps", "2", "--warmup", "1"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["n_gpus"] == 2 and j["value"] > 0 and j["cpu_baseline"]["kind"] == "oracle"
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["gpu_launches"] == 0


def _shard_worker(rank, world, port, out):
    """Pattern-sharded generation on CPU: every rank evaluates the oracle's SSE on its shard, one all-reduce (gloo) of M
    doubles, every rank steps the GA on the same all-reduced fitness."""
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = wl.scaled(wl.CONFIGS["c1"], P=1001, M=40)
    X, t, _ = wl.make_kb(cfg)                                     # same seed on every rank = one global knowledge base
    W = oracle.init_population(cfg.M, cfg.G, 5)
    p0, p1 = wl.shard_patterns(cfg.P, world, rank)
    _, sse = oracle.eval_fitness(cfg.d, cfg.family, X[p0:p1], t[p0:p1], W, return_sse=True)
    tot = torch.from_numpy(sse.copy())
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    F = (tot.numpy() / cfg.P).astype(np.float32)
    Wn = oracle.step(W, F, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, 5, 0)
    gathered = [torch.zeros(Wn.shape, dtype=torch.float32) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(Wn.copy()))
    if rank == 0:
        F_full = oracle.eval_fitness(cfg.d, cfg.family, X, t, W)
        json.dump({"same_pop": all(torch.equal(g, gathered[0]) for g in gathered),
                   "max_rel": float(np.max(np.abs(tot.numpy() / cfg.P - F_full) / F_full))}, open(out, "w"))
    dist.barrier()
    dist.destroy_process_group()


def test_pattern_sharded_generation_gloo(tmp_path):
    out = str(tmp_path / "s.json")
    mp.spawn(_shard_worker, args=(2, 29535, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["same_pop"] and r["max_rel"] <= 1e-13


def _lib_shard_worker(rank, world, port, out):
    """Pattern-sharded generations driven through the LIBRARY's entry points (game_eval_sse -> all-reduce ->
    game_set_fitness_from_sse -> game_step), two processes on the one GPU of the box; the all-reduce goes through gloo on
    a CPU copy (two ranks cannot share one GPU under NCCL), so no kernel ever waits on another rank's kernel."""
    import oracle
    import paper_1211_5481_b200 as game
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = wl.scaled(wl.CONFIGS["c3"], P=5003, M=200)
    X, t, _ = wl.make_kb(cfg)                                     # same seed on every rank = one global knowledge base
    p0, p1 = wl.shard_patterns(cfg.P, world, rank)
    G = game.Game(p1 - p0, cfg.N, cfg.d, cfg.M, cfg.expansion, cfg.activation)
    G.set_ga_params(cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma)
    G.load_kb(X[p0:p1], t[p0:p1])
    G.init_population(5)
    W = oracle.init_population(cfg.M, cfg.G, 5)
    sse = torch.zeros(cfg.M, dtype=torch.float64, device="cuda")
    ok, worst = True, 0.0
    for gen in range(3):
        game.game_eval_sse(G.ctx, sse.data_ptr()); G.sync()
        host = sse.cpu()
        dist.all_reduce(host, op=dist.ReduceOp.SUM)
        sse.copy_(host)
        game.game_set_fitness_from_sse(G.ctx, sse.data_ptr(), cfg.P, None)
        G.sync()
        F = G.get_fitness()
        F_ref = oracle.eval_fitness(cfg.d, cfg.family, X, t, W)
        worst = max(worst, float(np.max(np.abs(F - F_ref) / F_ref)))
        G.step(5, gen); G.sync()
        W = oracle.step(W, F, cfg.elite, cfg.tournament, cfg.p_cross, cfg.p_mut, cfg.sigma, 5, gen)
        ok = ok and np.array_equal(G.get_population().view(np.uint32), W.view(np.uint32))
    pops = [torch.zeros(W.shape, dtype=torch.float32) for _ in range(world)]
    dist.all_gather(pops, torch.from_numpy(G.get_population()))
    if rank == 0:
        json.dump({"lockstep": bool(ok), "same_pop": all(torch.equal(p_, pops[0]) for p_ in pops), "max_rel": worst}, open(out, "w"))
    G.close()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.gpu
def test_library_sharded_generations_two_processes_one_gpu(tmp_path):
    out = str(tmp_path / "ls.json")
    mp.spawn(_lib_shard_worker, args=(2, 29536, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["lockstep"] and r["same_pop"] and r["max_rel"] <= 1e-5
