"""world_size-2 gloo test (CPU) of the N > 1 host logic of bench.py: the path shards over walkers
with the table replicated and no data-path collective, so what the ranks share
is (i) the seeded recipe that gives every rank its own walkers, (ii) the max-over-ranks timing
reduction and (iii) the whole-job aggregate."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    import workloads
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = workloads.CONFIGS["small"]
        pos = workloads.positions(cfg, rank=rank)
        # every rank sees every rank's checksum: own walkers per rank, same recipe
        mine = torch.tensor([float(pos.sum()), float(pos.shape[0])], dtype=torch.float64)
        gathered = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(gathered, mine)
        sums = [float(g[0]) for g in gathered]
        assert len(set(sums)) == world, "ranks must draw different walkers"
        assert all(int(g[1]) == cfg.M for g in gathered), "weak scaling: same positions per rank"
        assert np.array_equal(pos, workloads.positions(cfg, rank=rank)), "recipe is deterministic per rank"
        # the slowest rank's time is the job's time, on every rank
        ms = bench.max_over_ranks(dist, 1.0 + 2.0 * rank, "cpu")
        assert ms == 1.0 + 2.0 * (world - 1)
        value = bench.whole_job_value(cfg.M, cfg.norb, world, ms)
        assert value == cfg.M * cfg.norb * world / (ms * 1e-3)
        dist.barrier()
        with open(os.path.join(out_dir, f"ok{rank}"), "w") as fh:
            fh.write(repr(value))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    vals = [open(tmp_path / f"ok{r}").read() for r in range(world)]
    assert vals[0] == vals[1]


def _orbital_worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import oracle
    import workloads
    from paper_1204_1121_b200 import sharding
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # orbital split (SURVEY.md §8e ii): every rank holds some columns of the table, sees all positions
        grid, L, M = (6, 5, 7), 38, 25                       # 38 orbitals: shards of 20 and 18 (units of 4)
        A, c, pos = workloads.small_case(grid, L, M, ((5.0, 0.3, -0.2), (1.1, 4.0, 0.7), (-0.6, 0.9, 6.0)), seed=7)
        lo, hi = sharding.orbital_range(L, rank, world)
        mine = sharding.table_shard(c, rank, world)
        assert mine.shape[-1] == hi - lo and np.array_equal(mine, c[..., lo:hi])
        # the CPU oracle stands in for the single-GPU evaluator of the shard (no GPU in this test)
        val, grad, lap, _ = oracle.eval_fast(A, grid, mine, pos)
        full_val = sharding.gather_orbitals(torch.from_numpy(val), L, dist)
        full_grad = sharding.gather_orbitals(torch.from_numpy(grad), L, dist)
        ref_val, ref_grad, _, _ = oracle.eval_fast(A, grid, c, pos)
        assert full_val.shape == (M, L) and full_grad.shape == (M, 3, L)
        assert np.array_equal(full_val.numpy(), ref_val) and np.array_equal(full_grad.numpy(), ref_grad)
        with open(os.path.join(out_dir, f"orb{rank}"), "w") as fh:
            fh.write("ok")
    finally:
        dist.destroy_process_group()


def test_orbital_split_two_ranks_gloo(tmp_path):
    world = 2
    mp.spawn(_orbital_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"orb{r}").exists() for r in range(world))


def test_orbital_ranges_cover_the_axis():
    from paper_1204_1121_b200 import sharding
    for norb, world, mult in [(768, 8, 4), (38, 2, 4), (5, 3, 4), (1536, 7, 2), (3, 4, 4)]:
        r = [sharding.orbital_range(norb, k, world, mult) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == norb
        assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
        assert all(lo % mult == 0 for lo, hi in r if lo < norb)


def test_single_process_reduction_is_identity():
    import bench
    assert bench.max_over_ranks(None, 3.5, "cpu") == 3.5
