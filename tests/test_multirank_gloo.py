"""N > 1 host logic on CPU: two gloo ranks, independent per-rank problems, max-over-ranks timing."""
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2107_08145_b200 import inputs, multi

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        r, lr, w = multi.env_ranks()
        assert (r, lr, w) == (rank, rank, world)
        inp = inputs.make_config(1, grid=(8, 8, 6), seed_offset=multi.rank_seed_offset(rank))
        local_ms = 10.0 * (rank + 1)                       # rank 1 is the slow one
        agg = multi.aggregate(local_ms, float(inp.updates), world)
        # every rank must see the same job-level numbers
        chk = torch.tensor([agg["ms"], agg["value"], float(inp.T.sum())], dtype=torch.float64)
        gathered = [torch.zeros_like(chk) for _ in range(world)]
        dist.all_gather(gathered, chk)
        if rank == 0:
            out.put([g.tolist() for g in gathered] + [inp.updates])
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_weak_scaling_aggregate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    g0, g1, upd = res
    assert g0[0] == g1[0] == 20.0                            # max over ranks
    assert np.isclose(g0[1], 2 * upd / 20.0e-3) and g0[1] == g1[1]   # units of all ranks / slowest time
    assert g0[2] != g1[2]                                    # different atmospheres per rank


def test_single_rank_needs_no_process_group():
    assert multi.max_over_ranks(3.5, 1) == 3.5
    assert multi.aggregate(2.0, 100.0, 1) == {"ms": 2.0, "value": 100.0 / 2e-3}


def test_reference_arm_other_ranks_exit_without_work():
    assert multi.reference_arm_runs_here(0) and not multi.reference_arm_runs_here(1)
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n_units, n = 12, 64
        mine = multi.shard_units(n_units, rank, world)
        # a mocked solve: unit u contributes the field (u + 1) * base to Q and owns slice u of "I_top"
        base = torch.arange(n, dtype=torch.float64)
        Q = torch.zeros(n, dtype=torch.float64)
        I = torch.zeros(n_units, n, dtype=torch.float64)
        for u in mine:
            Q += (u + 1) * base
            I[u] = (u + 1) + base
        multi.allreduce_sum(world, Q, I, None)
        lst = [None] * world
        dist.all_gather_object(lst, mine)
        if rank == 0:
            out.put((Q.tolist(), I.tolist(), lst))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_band_octant_sharding():
    """the ranks' unit lists are disjoint and cover all units; one sum all-reduce of the partial
    heating (and of the disjoint I_top slices) gives the single-rank result."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    Q, I, lst = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(lst[0] + lst[1]) == list(range(12)) and not set(lst[0]) & set(lst[1])
    base = np.arange(64, dtype=np.float64)
    assert np.array_equal(np.array(Q), sum(u + 1 for u in range(12)) * base)
    assert np.array_equal(np.array(I), np.array([(u + 1) + base for u in range(12)]))
    for world in (1, 3, 5, 12, 16):
        cover = sorted(u for r in range(world) for u in multi.shard_units(12, r, world))
        assert cover == list(range(12))
