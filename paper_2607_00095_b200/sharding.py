"""Host-side multi-GPU plumbing: one process per GPU, samples sharded across ranks.

Samples are independent blocks of the KKT system (runtime linear in the number of
samples, L750), so the path shards over the batch with NO data-path collective: each rank projects its
own contiguous slice.  `torch.distributed` carries only bookkeeping — the barrier around the timed region,
the max-over-ranks of the device time, the sum of projected samples and the AND of the converged flags.
Backend-agnostic (NCCL on GPUs, gloo in the CPU tests); holds no projection arithmetic.
"""
from __future__ import annotations

from typing import Optional, Tuple


def shard_range(total: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous slice [lo, hi) of `total` samples owned by `rank`; sizes differ by at most one and the
    first `total % world` ranks get the extra sample.  Empty slices are legal (total < world)."""
    if world < 1 or not (0 <= rank < world) or total < 0:
        raise ValueError(f"bad shard request total={total} rank={rank} world={world}")
    base, extra = divmod(total, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def rank_seed(seed: int, rank: int) -> int:
    """Seed of rank `rank`'s synthetic batch in the weak-scaling bench (rank 0 keeps the config's seed)."""
    return int(seed) + 1000 * int(rank)


def reduce_timing(dist, device, local_ms: float, local_units: int, local_ok: bool) -> Tuple[float, int, bool]:
    """(max over ranks of the device time, total units over ranks, all ranks converged).
    `dist` is `torch.distributed` (initialised) or None for a single process."""
    if dist is None:
        return float(local_ms), int(local_units), bool(local_ok)
    import torch
    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([int(local_units), 0 if local_ok else 1], dtype=torch.int64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t[0]), int(c[0]), int(c[1]) == 0


def throughput(total_units: int, steps: int, max_ms: float) -> float:
    """Whole-job units per second: all ranks' units per step x steps / slowest rank's time."""
    return float(total_units) * steps / (max_ms * 1e-3)


def gather_slices(dist, device, local, total: int, rank: int, world: int) -> Optional["object"]:
    """Bookkeeping helper: all-gather per-rank result slices (first axis sharded by `shard_range`) into
    one tensor on every rank.  Not on the hot path."""
    import torch
    if dist is None:
        return local
    sizes = [shard_range(total, r, world) for r in range(world)]
    biggest = max(hi - lo for lo, hi in sizes)
    pad = torch.zeros((biggest,) + tuple(local.shape[1:]), dtype=local.dtype, device=device)
    pad[: local.shape[0]] = local
    outs = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(outs, pad)
    return torch.cat([o[: hi - lo] for o, (lo, hi) in zip(outs, sizes)], dim=0)
