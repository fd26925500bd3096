"""Event-sharded evaluation over several ranks (Eqs. 4-7): host-side plumbing only.

Each rank owns a handle over its shard of data and MC events.  One evaluation is
    pwa_raw_sums (this rank's additive raw sums, 4 + 4P doubles)  ->  all-reduce(sum)  ->  pwa_combine (Eqs. 4, 6, 7)
so that every rank ends with the same NLL, gradient and Hv.  The sum must be taken over the RAW sums, before the
logarithm and the division by G.  `dist` is torch.distributed (NCCL on GPUs; the CPU tests drive the same functions
with gloo and the raw vector filled by the test).
"""
from __future__ import annotations

RAW_HEADER = 4  # raw[0] = sum_data w ln I, raw[1] = W, raw[2] = G, raw[3] = N_mc, then gd | gG | hd | hG


def shard_range(n: int, rank: int, world: int, align: int = 32) -> tuple[int, int]:
    """Contiguous shard [lo, hi) of n events for `rank`; every event in exactly one shard.  Interior cuts fall on
    multiples of `align` events (default 32 = one tile of the sweep kernel): a zero-copy window (pwa_create with
    borrow = 1) that starts on an odd event is not 16-byte aligned per plane and would be served by the slow generic
    kernel.  Shard sizes differ by less than 2 `align` (one tile, plus the ragged last tile)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    if align < 1:
        raise ValueError("align must be >= 1")
    units = -(-n // align)  # whole tiles, the last one possibly ragged
    base, rem = divmod(units, world)
    lo_u = rank * base + min(rank, rem)
    hi_u = lo_u + base + (1 if rank < rem else 0)
    return min(lo_u * align, n), min(hi_u * align, n)


def allreduce_raw(raw, dist=None, deterministic: bool = False):
    """Sums the raw vector over all ranks in place (no-op for a single process).
    deterministic = True: all-gather + a sum in rank order on every rank, so that the result is the same bits on every
    rank whatever reduction algorithm the backend picks.  A CUDA tensor under the gloo backend (the
    one-GPU tests) is staged through the host."""
    if not (dist is not None and dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1):
        return raw
    import torch
    buf = raw.cpu() if (raw.is_cuda and dist.get_backend() == "gloo") else raw
    if deterministic:
        parts = [torch.empty_like(buf) for _ in range(dist.get_world_size())]
        dist.all_gather(parts, buf)
        total = parts[0].clone()
        for p in parts[1:]:
            total += p
        buf.copy_(total)
    else:
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)
    if buf is not raw:
        raw.copy_(buf)
    return raw


def sharded_nll_grad_hvp(pwa, handle, theta, v, raw, nll, grad, hv, dist=None, deterministic: bool = False) -> None:
    """One evaluation over all ranks' shards; all tensors live on this rank's device.  The library enqueues on the
    handle's stream (the legacy default stream unless one was given to pwa_create) and torch.distributed on torch's
    current stream: with a handle on its own stream, make that stream current (torch.cuda.stream) around this call."""
    pwa.pwa_raw_sums(handle, theta, v, raw)
    allreduce_raw(raw, dist, deterministic)
    pwa.pwa_combine(handle, raw, v, nll, grad, hv)
