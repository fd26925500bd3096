"""GPU parity at BASELINE.json's FULL config-4 size ("Big": R = 100, H = 4, 10 M MC + 1 M data events, 70.7 GB of event
store), through the C ABI ("config 4 on chunks copied back from the device"; hard part 7), in both launch
configurations `bench.py --config 4` can time: the planes adopted zero-copy (`--store borrow`, tensor copies) and the
library-owned tiled copy (`--store copy`, the default: one bulk copy per stage), which must give the same bits.

  * the WHOLE workload: the oracle's double build evaluates it chunk by chunk on host copies of <= 2 GB
    (oracle.raw_sums per chunk; shard additivity of the raw sums is pin P6), the chunk sums are added in 80-bit and
    combined by oracle.combine -> NLL, every gradient and every HVP component at the north_star tolerances;
  * sampled zero-copy windows (the first events, a tile-straddling middle piece, the ragged end; in this store any two
    planes of a resonance lie 160 MB apart and the last plane 64 GB from the first, far beyond 2^32 bytes) against
    the 80-bit oracle on host copies;
  * the oracle's throughput on this configuration is printed (it goes into profiles/).
"""
import time

import numpy as np
import pytest
import torch

from helpers import rel_l2

pytestmark = pytest.mark.gpu

NLL_TOL = 1e-10
VEC_TOL = 1e-8
CHUNK = 300_000  # events per host copy: 300 k x 6.4 KB = 1.9 GB


@pytest.fixture(scope="module")
def big(oracle_mod):
    import paper_2403_09225_b200 as pwa
    import workloads
    from paper_2403_09225_b200.build import build
    build()
    pwa.load()
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    free, total = torch.cuda.mem_get_info(0)
    if total < 100e9:
        pytest.skip("config 4 needs a 180 GB device")
    cfg = workloads.CONFIGS[4]
    w = workloads.make_workload(cfg, torch.device("cuda", 0))
    gm = pwa.Model(w, device=0, borrow=True)
    yield pwa, workloads, cfg, w, gm
    gm.close()


def _chunk_model(oracle_mod, w, which, a, b):
    """Host copy of events [a, b) of one sample as an oracle Model (the other sample is a one-event stub)."""
    to_np = lambda t: t.detach().cpu().numpy()
    if which == "mc":
        smp = oracle_mod.Sample(to_np(w.mc_mass[:, a:b].contiguous()), to_np(w.mc_amp[:, :, a:b].contiguous()), None)
        stub = oracle_mod.Sample(to_np(w.data_mass[:, :1].contiguous()), to_np(w.data_amp[:, :, :1].contiguous()), None)
        return oracle_mod.Model(to_np(w.res_chan), stub, smp)
    wt = None if w.data_weight is None else to_np(w.data_weight[a:b].contiguous())
    smp = oracle_mod.Sample(to_np(w.data_mass[:, a:b].contiguous()), to_np(w.data_amp[:, :, a:b].contiguous()), wt)
    stub = oracle_mod.Sample(to_np(w.mc_mass[:, :1].contiguous()), to_np(w.mc_amp[:, :, :1].contiguous()), None)
    return oracle_mod.Model(to_np(w.res_chan), smp, stub)


def test_whole_config4_against_the_oracle_chunk_by_chunk(oracle_mod, big, capsys):
    pwa, workloads, cfg, w, gm = big
    assert cfg.n_mc == 10_000_000 and cfg.n_data == 1_000_000 and cfg.n_res == 100 and cfg.n_hel == 4
    assert pwa.pwa_kernel_variant(gm.h).startswith("lanes"), pwa.pwa_kernel_variant(gm.h)
    assert pwa.pwa_bytes_per_eval(gm.h) == 11_000_000 * 6424
    nt = oracle_mod.max_threads()
    th, v = workloads.random_start(cfg, 0).numpy(), workloads.direction(cfg, 0).numpy()
    P = cfg.n_par
    ld = np.longdouble
    tot = {k: [np.zeros(2, ld), np.zeros(P, ld), np.zeros(P, ld)] for k in ("mc", "data")}
    t_oracle, n_done = 0.0, 0
    for which, n in (("mc", cfg.n_mc), ("data", cfg.n_data)):
        for a in range(0, n, CHUNK):
            b = min(n, a + CHUNK)
            cm = _chunk_model(oracle_mod, w, which, a, b)
            t0 = time.perf_counter()
            sc, g, h = oracle_mod.raw_sums(cm, which, th, v, "d", threads=nt)
            t_oracle += time.perf_counter() - t0
            n_done += b - a
            tot[which][0] += sc
            tot[which][1] += g
            tot[which][2] += h
            del cm
    f0, g0, h0 = oracle_mod.combine(tot["data"][0], tot["mc"][0], tot["data"][1], tot["mc"][1], tot["data"][2],
                                    tot["mc"][2], v, "ld")
    f, g, hv = gm.nll_grad_hvp(th, v)
    with capsys.disabled():
        print(f"\nconfig 4 whole workload: oracle (double build, {nt} threads) {n_done / t_oracle:.3e} events/s "
              f"({t_oracle:.1f} s for {n_done} events); nll gpu {f:.12e} oracle {float(f0):.12e} "
              f"rel {abs(f - float(f0)) / abs(float(f0)):.2e}; grad {rel_l2(g, g0):.2e}; hvp {rel_l2(hv, h0):.2e}")
    assert abs(f - float(f0)) / max(abs(float(f0)), 1.0) < NLL_TOL
    assert rel_l2(g, g0) < VEC_TOL and rel_l2(hv, h0) < VEC_TOL
    assert pwa.pwa_status_flags(gm.h) == 0
    f1, g1 = gm.nll_grad(th)
    assert abs(f1 - float(f0)) / max(abs(float(f0)), 1.0) < NLL_TOL and rel_l2(g1, g0) < VEC_TOL
    f2, g2, hv2 = gm.nll_grad_hvp(th, v)
    assert f2 == f and g2.tobytes() == g.tobytes() and hv2.tobytes() == hv.tobytes()  # repeat runs: same bits
    # the library-owned tiled copy of the same 70.7 GB (what bench.py --config 4 times by default): same bits
    torch.cuda.empty_cache()
    tm = pwa.Model(w, device=0, borrow=False)
    try:
        assert "tile=8t," in pwa.pwa_kernel_variant(tm.h), pwa.pwa_kernel_variant(tm.h)
        f3, g3, hv3 = tm.nll_grad_hvp(th, v)
        assert f3 == f and g3.tobytes() == g.tobytes() and hv3.tobytes() == hv.tobytes()
        f4, g4 = tm.nll_grad(th)
        assert f4 == f1 and g4.tobytes() == g1.tobytes()
        assert pwa.pwa_status_flags(tm.h) == 0
    finally:
        tm.close()


WINDOWS = [(0, 1_031, 0, 517), (4_999_990, 2_051, 499_994, 1_027), (9_998_976, 1_024, 999_744, 256)]


@pytest.mark.parametrize("m0,nm,d0,nd", WINDOWS)
def test_config4_windows_against_the_80bit_oracle(oracle_mod, big, m0, nm, d0, nd):
    pwa, workloads, cfg, w, gm = big
    assert m0 + nm <= cfg.n_mc and d0 + nd <= cfg.n_data
    th, v = workloads.random_start(cfg, 1).numpy(), workloads.direction(cfg, 3).numpy()
    to_np = lambda t: t.detach().cpu().numpy()
    wm = oracle_mod.Model(to_np(w.res_chan),
                          oracle_mod.Sample(to_np(w.data_mass[:, d0:d0 + nd].contiguous()), to_np(w.data_amp[:, :, d0:d0 + nd].contiguous()), None),
                          oracle_mod.Sample(to_np(w.mc_mass[:, m0:m0 + nm].contiguous()), to_np(w.mc_amp[:, :, m0:m0 + nm].contiguous()), None))
    f0, g0, h0 = oracle_mod.nll_grad_hvp(wm, th, v, "ld", threads=oracle_mod.max_threads())
    for borrow in (True, False):  # zero-copy window of the planes; the library's tiled copy of the window
        h = pwa.pwa_create(w.res_chan, w.data_mass, w.data_amp, w.data_weight, w.mc_mass, w.mc_amp, borrow=borrow,
                           data_first=d0, n_data=nd, mc_first=m0, n_mc=nm)
        try:
            dev = torch.device("cuda", 0)
            nll = torch.zeros(1, dtype=torch.float64, device=dev)
            g = torch.zeros(cfg.n_par, dtype=torch.float64, device=dev)
            hv = torch.zeros(cfg.n_par, dtype=torch.float64, device=dev)
            pwa.pwa_nll_grad_hvp(h, torch.tensor(th, device=dev), torch.tensor(v, device=dev), nll, g, hv)
            torch.cuda.synchronize()
            # the variants bench.py --config 4 runs (--store borrow / the default --store copy)
            if borrow:
                assert pwa.pwa_kernel_variant(h) == pwa.pwa_kernel_variant(gm.h)
            else:
                assert "tile=8t," in pwa.pwa_kernel_variant(h)
            assert abs(nll.item() - float(f0)) / max(abs(float(f0)), 1.0) < NLL_TOL
            assert rel_l2(g.cpu().numpy(), g0) < VEC_TOL and rel_l2(hv.cpu().numpy(), h0) < VEC_TOL
        finally:
            pwa.pwa_destroy(h)
