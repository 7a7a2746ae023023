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


def test_single_process_reduction_is_identity():
    import bench
    assert bench.max_over_ranks(None, 3.5, "cpu") == 3.5
