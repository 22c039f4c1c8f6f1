"""Multi-GPU layout of the path: material points are independent, so the
centre list is cut into contiguous equal-count slabs, one per rank; the ion cloud is replicated (every rank
ingests the same array) and there is NO collective on the data path.  Signatures stay sharded on the rank
that computed them; only small per-material-point arrays (counts) are worth gathering.

Host logic only -- the arithmetic of the method lives in the CUDA library."""
from __future__ import annotations


def shard_range(M: int, rank: int, world: int) -> tuple[int, int]:
    """[begin, end) of the material points owned by `rank`: slabs differ by at most one point."""
    if world < 1 or not (0 <= rank < world) or M < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(M, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def run_sharded(plan, xyz, types, centres, sig_local, counts_local=None, rank: int = 0, world: int = 1, stream=None):
    """Run the hot path for this rank's slab of `centres` (a device tensor holding ALL centres).
    `sig_local` / `counts_local` are sized for the slab.  Returns (begin, end)."""
    b, e = shard_range(int(centres.shape[0]), rank, world)
    plan.apx_run(xyz, types, centres[b:e], sig_local, counts_local, stream=stream)
    return b, e


def gather_counts(counts_local, M: int, rank: int, world: int):
    """all_gather the per-material-point ion counts (4 B each) of every rank into one [M] tensor, in order.
    Uses the default process group (NCCL on GPUs, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    if world == 1:
        return counts_local.clone()
    sizes = [shard_range(M, r, world)[1] - shard_range(M, r, world)[0] for r in range(world)]
    pad = max(sizes)
    buf = torch.zeros(pad, dtype=counts_local.dtype, device=counts_local.device)
    buf[: counts_local.numel()] = counts_local
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    return torch.cat([o[:n] for o, n in zip(out, sizes)])
