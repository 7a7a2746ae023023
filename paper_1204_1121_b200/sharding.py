"""Multi-GPU partitionings of the orbital evaluation.  Host logic only: every
(position, orbital) pair is independent, so sharding is a choice of who holds what.

  walkers   replicate the table, give every rank its own walkers: no data-path collective at all —
            the paper's own scaling model (MPI over configurations, one GPU per node,
            PAPER.md:25-27).  bench.py --gpus N runs this way; nothing is needed from this module.
  orbitals  rank r holds the columns [lo_r, hi_r) of the table (`orbital_range`, `table_shard`) and
            evaluates them at ALL positions with an ordinary single-GPU handle; if a consumer
            needs whole rows, `gather_orbitals` concatenates the shards along the orbital axis
            with one all-gather (NCCL over NVLink on GPUs; gloo in the CPU tests).  Only needed
            when the table outgrows one GPU's memory (the largest config here is 6.3 GB of 180 GB).

Argument marshalling and one torch.distributed call; no arithmetic of the method.
"""
import torch


def orbital_range(norb, rank, world, multiple=4):
    """Columns [lo, hi) of rank `rank`: contiguous, as even as possible in units of `multiple`
    orbitals (4 = one 128-bit lane quad; use an even multiple for complex orbitals, whose real and
    imaginary channels are adjacent columns)."""
    assert 0 <= rank < world and multiple >= 1
    units = -(-int(norb) // multiple)
    base, extra = divmod(units, world)
    lo_u = rank * base + min(rank, extra)
    hi_u = lo_u + base + (1 if rank < extra else 0)
    return min(lo_u * multiple, norb), min(hi_u * multiple, norb)


def table_shard(coeffs, rank, world, multiple=4):
    """The columns of `coeffs` [n1][n2][n3][L] (numpy or torch) that rank `rank` holds, contiguous."""
    lo, hi = orbital_range(coeffs.shape[-1], rank, world, multiple)
    part = coeffs[..., lo:hi]
    return part.contiguous() if isinstance(part, torch.Tensor) else part.copy()


def gather_orbitals(local, norb, dist, multiple=4, group=None):
    """All-gather of per-rank outputs along the orbital axis: `local` [..., hi_r - lo_r] on every
    rank -> [..., norb] on every rank.  Shards may differ in width: they are padded to the widest
    for the collective and trimmed afterwards."""
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    ranges = [orbital_range(norb, r, world, multiple) for r in range(world)]
    assert local.shape[-1] == ranges[rank][1] - ranges[rank][0]
    width = max(hi - lo for lo, hi in ranges)
    padded = local.new_zeros((*local.shape[:-1], width))
    padded[..., :local.shape[-1]] = local
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded.contiguous(), group=group)
    return torch.cat([p[..., :hi - lo] for p, (lo, hi) in zip(parts, ranges)], dim=-1)
