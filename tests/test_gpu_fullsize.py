"""GPU parity at BASELINE.json's FULL config-3 size, in the launch configuration bench.py times (device-generated
workload, borrowed buffers, persistent lanes kernel), through the C ABI.

The 80-bit oracle needs minutes for 5.5 M events x 30 resonances; what it can do in seconds:
  * the oracle's double build (Neumaier-compensated sums, OpenMP) evaluates the WHOLE workload in about a second on
    the box's cores -> NLL, every gradient and every HVP component compared at the north_star tolerances;
  * that double build is tied to the 80-bit reference on sampled windows of the same arrays;
  * sampled windows of the full store (first events, a tile-straddling middle piece, the ragged end) evaluated by
    the CUDA path on zero-copy views against the 80-bit oracle on host copies of those windows;
  * a property that holds at any size: the raw sums of two zero-copy shards of the full store add up to the raw
    sums of the whole (Eqs. 4-7), and repeat runs are bit-identical.
"""
import numpy as np
import pytest
import torch

from helpers import rel_l2

pytestmark = pytest.mark.gpu

NLL_TOL = 1e-10
VEC_TOL = 1e-8


@pytest.fixture(scope="module")
def full(oracle_mod):
    import paper_2403_09225_b200 as pwa
    import workloads
    from paper_2403_09225_b200.build import build
    build()
    pwa.load()
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    cfg = workloads.CONFIGS[3]
    w = workloads.make_workload(cfg, torch.device("cuda", 0))
    gm = pwa.Model(w, device=0, borrow=True)
    assert pwa.pwa_kernel_variant(gm.h).startswith("lanes"), pwa.pwa_kernel_variant(gm.h)
    om = oracle_mod.model_from_workload(w)  # host copies (5.4 GB)
    yield pwa, workloads, cfg, w, gm, om
    gm.close()


def _nll_err(a, b):
    return abs(float(a) - float(b)) / max(abs(float(b)), 1.0)


def test_whole_workload_against_the_oracle_double_build(oracle_mod, full):
    pwa, workloads, cfg, w, gm, om = full
    assert cfg.n_mc == 5_000_000 and cfg.n_data == 500_000 and cfg.n_res == 30
    nt = oracle_mod.max_threads()
    for k, th in enumerate((workloads.theta_true(cfg).numpy(), workloads.random_start(cfg, 0).numpy())):
        v = workloads.direction(cfg, k).numpy()
        f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "d", threads=nt)
        f, g, hv = gm.nll_grad_hvp(th, v)
        assert _nll_err(f, f0) < NLL_TOL, (k, f, float(f0))
        assert rel_l2(g, g0) < VEC_TOL, k
        assert rel_l2(hv, h0) < VEC_TOL, k
        assert pwa.pwa_status_flags(gm.h) == 0
        # separate entry points take the other two kernel modes through the same store
        assert _nll_err(gm.nll(th), f0) < NLL_TOL
        f1, g1 = gm.nll_grad(th)
        assert _nll_err(f1, f0) < NLL_TOL and rel_l2(g1, g0) < VEC_TOL


def _window_model(oracle_mod, w, m0, m1, d0, d1):
    to_np = lambda t: t.detach().cpu().numpy()
    wt = None if w.data_weight is None else to_np(w.data_weight[d0:d1].contiguous())
    return oracle_mod.Model(to_np(w.res_chan),
                            oracle_mod.Sample(to_np(w.data_mass[:, d0:d1].contiguous()), to_np(w.data_amp[:, :, d0:d1].contiguous()), wt),
                            oracle_mod.Sample(to_np(w.mc_mass[:, m0:m1].contiguous()), to_np(w.mc_amp[:, :, m0:m1].contiguous()), None))


# (first MC event, MC count, first data event, data count): the beginning, a piece that straddles tiles and ends
# off a tile boundary, and the ragged end of both samples; firsts are even (16-byte aligned mass planes)
WINDOWS = [(0, 4_097, 0, 1_025), (2_499_998, 6_001, 249_990, 1_537), (4_995_904, 4_096, 499_488, 512)]


@pytest.mark.parametrize("m0,nm,d0,nd", WINDOWS)
def test_sampled_windows_against_the_80bit_oracle(oracle_mod, full, m0, nm, d0, nd):
    pwa, workloads, cfg, w, gm, om = full
    assert m0 + nm <= cfg.n_mc and d0 + nd <= cfg.n_data
    th, v = workloads.random_start(cfg, 1).numpy(), workloads.direction(cfg, 3).numpy()
    wm = _window_model(oracle_mod, w, m0, m0 + nm, d0, d0 + nd)
    f0, g0, h0 = oracle_mod.nll_grad_hvp(wm, th, v, "ld")
    fd, gd, hd = oracle_mod.nll_grad_hvp(wm, th, v, "d")
    assert _nll_err(fd, f0) < 1e-13 and rel_l2(gd, g0) < 1e-12 and rel_l2(hd, h0) < 1e-12  # double build == 80-bit
    h = pwa.pwa_create(w.res_chan, w.data_mass, w.data_amp, w.data_weight, w.mc_mass, w.mc_amp, borrow=True,
                       data_first=d0, n_data=nd, mc_first=m0, n_mc=nm)
    try:
        dev = torch.device("cuda", 0)
        nll = torch.zeros(1, dtype=torch.float64, device=dev)
        g = torch.zeros(cfg.n_par, dtype=torch.float64, device=dev)
        hv = torch.zeros(cfg.n_par, dtype=torch.float64, device=dev)
        pwa.pwa_nll_grad_hvp(h, torch.tensor(th, device=dev), torch.tensor(v, device=dev), nll, g, hv)
        torch.cuda.synchronize()
        assert pwa.pwa_kernel_variant(h).startswith("lanes")
        assert _nll_err(nll.item(), f0) < NLL_TOL
        assert rel_l2(g.cpu().numpy(), g0) < VEC_TOL and rel_l2(hv.cpu().numpy(), h0) < VEC_TOL
    finally:
        pwa.pwa_destroy(h)


def test_zero_copy_shards_add_up_and_runs_repeat(full):
    pwa, workloads, cfg, w, gm, om = full
    dev = torch.device("cuda", 0)
    th = torch.tensor(workloads.random_start(cfg, 2).numpy(), device=dev)
    v = torch.tensor(workloads.direction(cfg, 4).numpy(), device=dev)
    whole = gm.raw_sums(th, v).clone()
    again = gm.raw_sums(th, v)
    assert whole.cpu().numpy().tobytes() == again.cpu().numpy().tobytes()
    cut_m, cut_d = 2_718_282, 314_160
    total = torch.zeros_like(whole)
    for (m0, nm, d0, nd) in ((0, cut_m, 0, cut_d), (cut_m, cfg.n_mc - cut_m, cut_d, cfg.n_data - cut_d)):
        h = pwa.pwa_create(w.res_chan, w.data_mass, w.data_amp, w.data_weight, w.mc_mass, w.mc_amp, borrow=True,
                           data_first=d0, n_data=nd, mc_first=m0, n_mc=nm)
        raw = torch.zeros_like(whole)
        pwa.pwa_raw_sums(h, th, v, raw)
        torch.cuda.synchronize()
        total += raw
        pwa.pwa_destroy(h)
    a, b = total.cpu().numpy(), whole.cpu().numpy()
    assert a[3] == cfg.n_mc and b[3] == cfg.n_mc
    assert abs(a[0] - b[0]) <= 1e-12 * abs(b[0]) and abs(a[2] - b[2]) <= 1e-12 * abs(b[2])
    P = cfg.n_par
    for k in range(4):
        assert rel_l2(a[4 + k * P: 4 + (k + 1) * P], b[4 + k * P: 4 + (k + 1) * P]) < 1e-11, k
