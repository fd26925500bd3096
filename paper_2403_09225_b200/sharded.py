"""Event-sharded evaluation over several ranks (Eqs. 4-7): host-side plumbing only.

Each rank owns a handle over its shard of data and MC events.  One evaluation is
    pwa_raw_sums (this rank's additive raw sums, 4 + 4P doubles)  ->  all-reduce(sum)  ->  pwa_combine (Eqs. 4, 6, 7)
so that every rank ends with the same NLL, gradient and Hv.  The sum must be taken over the RAW sums, before the
logarithm and the division by G.  `dist` is torch.distributed (NCCL on GPUs; the CPU tests drive the same functions
with gloo and the raw vector filled by the test).
"""
from __future__ import annotations

RAW_HEADER = 4  # raw[0] = sum_data w ln I, raw[1] = W, raw[2] = G, raw[3] = N_mc, then gd | gG | hd | hG


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous shard [lo, hi) of n events for `rank`: sizes differ by at most one, every event in exactly one shard."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def allreduce_raw(raw, dist=None):
    """Sums the raw vector over all ranks in place (no-op for a single process)."""
    if dist is not None and dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(raw, op=dist.ReduceOp.SUM)
    return raw


def sharded_nll_grad_hvp(pwa, handle, theta, v, raw, nll, grad, hv, dist=None) -> None:
    """One evaluation over all ranks' shards; all tensors live on this rank's device."""
    pwa.pwa_raw_sums(handle, theta, v, raw)
    allreduce_raw(raw, dist)
    pwa.pwa_combine(handle, raw, v, nll, grad, hv)
