"""World-size-2 test of the event-sharded evaluation (Eqs. 4-7) on CPU with gloo.

The host-side plumbing under test is paper_2403_09225_b200/sharded.py: shard_range (every event in exactly one
shard), the layout of the raw vector, the all-reduce over the RAW sums (before ln and 1/G) and the redundant
combination on every rank.  No GPU is available to these tests, so each rank fills its raw vector with the CPU
oracle's raw sums of its shard (the stand-in for pwa_raw_sums) and combines with the oracle's Eqs. 4/6/7 (the
stand-in for pwa_combine); the CUDA raw sums themselves are compared with the oracle's, block by block, in
tests/test_gpu_parity.py::test_shard_additivity_through_raw_sums.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from helpers import random_model, random_theta, rel_l2

R, H, C, N_DATA, N_MC = 5, 2, 2, 1_001, 4_003  # odd sizes: the two shards differ in length


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _pack(sd, sm, gd, gG, hd, hG):
    return np.concatenate([[sd[0], sd[1], sm[0], sm[1]], gd, gG, hd, hG]).astype(np.float64)


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_2403_09225_b200 import sharded
        om = random_model(oracle, 11, R, H, C, N_DATA, N_MC, weighted=True)
        th, v = random_theta(12, R), np.random.RandomState(13).normal(size=4 * R)
        d0, d1 = sharded.shard_range(N_DATA, rank, world)
        m0, m1 = sharded.shard_range(N_MC, rank, world)
        sd, gd, hd = oracle.raw_sums(om, "data", th, v, "d", first=d0, count=d1 - d0)
        sm, gG, hG = oracle.raw_sums(om, "mc", th, v, "d", first=m0, count=m1 - m0)
        raw = torch.from_numpy(_pack(sd, sm, gd, gG, hd, hG))
        assert raw.numel() == sharded.RAW_HEADER + 4 * om.n_par
        det = raw.clone()
        sharded.allreduce_raw(raw, dist)
        sharded.allreduce_raw(det, dist, deterministic=True)   # all-gather + rank-order sum
        assert np.allclose(det.numpy(), raw.numpy(), rtol=1e-15, atol=0.0)
        r = det.numpy()
        P = om.n_par
        blk = lambda k: r[4 + k * P: 4 + (k + 1) * P]
        nll, grad, hv = oracle.combine(r[0:2], r[2:4], blk(0), blk(1), blk(2), blk(3), v, "d")
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), nll=float(nll), grad=np.asarray(grad, np.float64),
                 hv=np.asarray(hv, np.float64), n_mc=r[3], shard=np.array([d0, d1, m0, m1]))
    finally:
        dist.destroy_process_group()


def test_shard_range_partitions_every_event():
    from paper_2403_09225_b200.sharded import shard_range
    for n in (0, 1, 7, 1_000, 1_001, 5_500_000):
        for world in (1, 2, 3, 8):
            cuts = [shard_range(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) < 2 * 32
            assert all(lo % 32 == 0 or lo == n for lo, _ in cuts)  # zero-copy windows stay 16-byte aligned per plane
            exact = [shard_range(n, r, world, align=1) for r in range(world)]
            assert max(hi - lo for lo, hi in exact) - min(hi - lo for lo, hi in exact) <= 1
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def test_two_rank_sharded_evaluation_matches_the_unsharded_oracle(oracle_mod, tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    om = random_model(oracle_mod, 11, R, H, C, N_DATA, N_MC, weighted=True)
    th, v = random_theta(12, R), np.random.RandomState(13).normal(size=4 * R)
    f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
    outs = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    # every rank ends with the same bits (the combination is redundant, theta stays replicated)
    assert outs[0]["nll"] == outs[1]["nll"]
    assert outs[0]["grad"].tobytes() == outs[1]["grad"].tobytes() and outs[0]["hv"].tobytes() == outs[1]["hv"].tobytes()
    # shards are disjoint and cover both samples
    s0, s1 = outs[0]["shard"], outs[1]["shard"]
    assert s0[0] == 0 and s0[1] == s1[0] and s1[1] == N_DATA and s0[2] == 0 and s0[3] == s1[2] and s1[3] == N_MC
    assert outs[0]["n_mc"] == N_MC
    # and the result is the unsharded one
    assert abs(float(outs[0]["nll"]) - float(f0)) <= 1e-12 * max(1.0, abs(float(f0)))
    assert rel_l2(outs[0]["grad"], g0) < 1e-12 and rel_l2(outs[0]["hv"], h0) < 1e-12


def test_summing_after_the_logarithm_would_be_wrong(oracle_mod):
    """The reduction must act on the raw sums: averaging per-shard NLLs is not the NLL (log of a sum)."""
    from paper_2403_09225_b200.sharded import shard_range
    om = random_model(oracle_mod, 11, R, H, C, N_DATA, N_MC, weighted=True)
    th = random_theta(12, R)
    f0 = float(oracle_mod.nll(om, th, "d"))
    per_shard = 0.0
    for rank in range(2):
        d0, d1 = shard_range(N_DATA, rank, 2)
        m0, m1 = shard_range(N_MC, rank, 2)
        sd, gd, _ = oracle_mod.raw_sums(om, "data", th, None, "d", first=d0, count=d1 - d0)
        sm, gG, _ = oracle_mod.raw_sums(om, "mc", th, None, "d", first=m0, count=m1 - m0)
        per_shard += float(oracle_mod.combine(sd, sm, gd, gG, prec="d")[0])
    assert abs(per_shard - f0) > 1e-6 * abs(f0)
