"""The REAL kernels under a process group (Eqs. 4-7): world size 2, backend gloo,
both ranks on cuda:0 (the one GPU of this pool; the ranks' kernels never wait on one another - the exchange is a
host-side gloo collective).  Each rank creates a ZERO-COPY window handle over its sharded.shard_range of one seeded
workload, runs the CUDA pwa_raw_sums, sharded.allreduce_raw on the CUDA tensor, and the CUDA pwa_combine.  Both ranks
must end with the same bits, and those must equal the unsharded 80-bit oracle within the north_star tolerances."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from helpers import rel_l2

pytestmark = pytest.mark.gpu
N_MC, N_DATA = 40_014, 5_002  # ragged (the last shard ends off a tile boundary) but even: planes of a borrowed store must be 16-byte aligned


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str, deterministic: bool):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import paper_2403_09225_b200 as pwa
        import workloads
        from paper_2403_09225_b200 import sharded
        pwa.load()
        dev = torch.device("cuda", 0)
        cfg = workloads.CONFIGS[3].scaled(N_MC, N_DATA)
        w = workloads.make_workload(cfg, dev, chunk=1 << 14, imax_events=N_MC)   # same seeded arrays on both ranks
        d0, d1 = sharded.shard_range(cfg.n_data, rank, world)
        m0, m1 = sharded.shard_range(cfg.n_mc, rank, world)
        h = pwa.pwa_create(w.res_chan, w.data_mass, w.data_amp, w.data_weight, w.mc_mass, w.mc_amp, borrow=True,
                           data_first=d0, n_data=d1 - d0, mc_first=m0, n_mc=m1 - m0)
        variant = pwa.pwa_kernel_variant(h)
        P = cfg.n_par
        th = torch.tensor(workloads.random_start(cfg, 1).numpy(), device=dev)
        v = torch.tensor(workloads.direction(cfg, 2).numpy(), device=dev)
        raw = torch.zeros(sharded.RAW_HEADER + 4 * P, dtype=torch.float64, device=dev)
        nll = torch.zeros(1, dtype=torch.float64, device=dev)
        g = torch.zeros(P, dtype=torch.float64, device=dev)
        hv = torch.zeros(P, dtype=torch.float64, device=dev)
        sharded.sharded_nll_grad_hvp(pwa, h, th, v, raw, nll, g, hv, dist, deterministic=deterministic)
        torch.cuda.synchronize()
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), nll=nll.cpu().numpy(), grad=g.cpu().numpy(), hv=hv.cpu().numpy(),
                 n_mc=raw[3].item(), shard=np.array([d0, d1, m0, m1]), variant=np.array(variant))
        pwa.pwa_destroy(h)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("deterministic", [False, True])
def test_two_ranks_cuda_raw_sums_allreduce_combine(oracle_mod, tmp_path, deterministic):
    import workloads
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path), deterministic), nprocs=world, join=True)
    outs = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    for o in outs:
        assert str(o["variant"]).startswith("lanes"), str(o["variant"])   # aligned cuts: the fast kernel on both shards
    assert outs[0]["nll"].tobytes() == outs[1]["nll"].tobytes()
    assert outs[0]["grad"].tobytes() == outs[1]["grad"].tobytes() and outs[0]["hv"].tobytes() == outs[1]["hv"].tobytes()
    s0, s1 = outs[0]["shard"], outs[1]["shard"]
    assert s0[0] == 0 and s0[1] == s1[0] and s1[1] == N_DATA and s0[2] == 0 and s0[3] == s1[2] and s1[3] == N_MC
    assert outs[0]["n_mc"] == N_MC
    cfg = workloads.CONFIGS[3].scaled(N_MC, N_DATA)
    w = workloads.make_workload(cfg, torch.device("cuda", 0), chunk=1 << 14, imax_events=N_MC)
    om = oracle_mod.model_from_workload(w)
    th, v = workloads.random_start(cfg, 1).numpy(), workloads.direction(cfg, 2).numpy()
    f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
    assert abs(float(outs[0]["nll"][0]) - float(f0)) <= 1e-10 * max(1.0, abs(float(f0)))
    assert rel_l2(outs[0]["grad"], g0) < 1e-8 and rel_l2(outs[0]["hv"], h0) < 1e-8
