"""Edge shapes through the C ABI against the oracle: the smallest and largest models each kernel family serves, event
counts below one tile, one event, the shape-selection boundaries (capacity 4 / 6 / 8 / 10 / 12 / 16 / 20 / 24 / 32 / 48 / 64 /
96 / 128, more than 128
resonances and more than 4 helicities on the generic kernel), weighted and unweighted data."""
import numpy as np
import pytest
import torch

from helpers import random_theta, rel_l2

pytestmark = pytest.mark.gpu

# (R, H, C, n_data, n_mc, weighted)
SHAPES = [(1, 1, 1, 1, 1, False), (1, 1, 1, 33, 65, True), (2, 4, 1, 7, 100, True), (4, 3, 2, 31, 32, False),
          (5, 2, 2, 257, 1000, True), (12, 1, 3, 100, 999, False), (13, 2, 3, 100, 999, True), (16, 4, 2, 64, 640, False),
          (17, 3, 1, 65, 700, True), (32, 2, 3, 129, 1025, True), (33, 2, 2, 90, 800, False), (33, 4, 3, 90, 515, True),
          (64, 1, 3, 50, 600, False), (65, 3, 2, 40, 400, True), (128, 4, 3, 33, 300, False), (129, 2, 3, 33, 300, True),
          (6, 5, 2, 50, 500, True), (3, 8, 1, 20, 333, False),
          # the two-events-per-lane fused kernel (13 <= R <= 32, H <= 2): H = 1, one event, fewer tiles than blocks and warps
          (20, 1, 2, 70, 900, True), (30, 2, 3, 1, 1, False), (25, 2, 1, 33, 65, True), (32, 1, 3, 31, 4777, False),
          # the capacity boundaries of the finer shape grid (6, 8, 20, 24 slots on 32-event tiles; 48, 96 on 8-event tiles)
          (6, 2, 1, 100, 1001, True), (7, 3, 2, 65, 700, False), (8, 4, 2, 9, 333, True), (9, 2, 3, 40, 401, False),
          (17, 2, 3, 100, 999, True), (20, 4, 3, 33, 515, False), (21, 3, 2, 70, 640, True), (24, 2, 3, 129, 1025, False),
          (34, 2, 3, 50, 600, True), (48, 4, 2, 17, 300, False), (49, 1, 3, 64, 512, True), (96, 2, 3, 33, 257, False),
          (97, 3, 2, 20, 200, True)]


@pytest.fixture(scope="module")
def pwa():
    import paper_2403_09225_b200 as p
    from paper_2403_09225_b200.build import build
    build()
    p.load()
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    return p


@pytest.mark.parametrize("R,H,C,nd,nm,weighted", SHAPES)
def test_shape(pwa, oracle_mod, R, H, C, nd, nm, weighted):
    rs = np.random.RandomState(1000 * R + 10 * H + C)
    res_chan = (np.arange(R) % C).astype(np.int32)

    def sample(n, w):
        return rs.uniform(0.3, 3.0, size=(C, n)), rs.normal(size=(R, H, n, 2)), (rs.uniform(0.5, 1.5, size=n) if w else None)

    dm, da, dw = sample(nd, weighted)
    mm, ma, _ = sample(nm, False)
    om = oracle_mod.Model(res_chan, oracle_mod.Sample(dm, da, dw), oracle_mod.Sample(mm, ma, None))
    t = lambda x: None if x is None else torch.from_numpy(np.ascontiguousarray(x))
    h = pwa.pwa_create(t(res_chan), t(dm), t(da), t(dw), t(mm), t(ma))
    try:
        name = pwa.pwa_kernel_variant(h)
        assert name.startswith("lanes") == (R <= 128 and H <= 4), name
        dev = torch.device("cuda", 0)
        th = random_theta(7 + R, R)
        v = rs.normal(size=4 * R)
        P = 4 * R
        nll = torch.zeros(1, dtype=torch.float64, device=dev)
        g = torch.zeros(P, dtype=torch.float64, device=dev)
        hv = torch.zeros(P, dtype=torch.float64, device=dev)
        thd, vd = torch.tensor(th, device=dev), torch.tensor(v, device=dev)
        f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
        err = lambda f: abs(f - float(f0)) / max(abs(float(f0)), 1.0)
        pwa.pwa_nll_grad_hvp(h, thd, vd, nll, g, hv)
        assert err(nll.item()) < 1e-10, name
        assert rel_l2(g.cpu().numpy(), g0) < 1e-8 and rel_l2(hv.cpu().numpy(), h0) < 1e-8, name
        pwa.pwa_nll(h, thd, nll)
        assert err(nll.item()) < 1e-10
        g.zero_(); hv.zero_()
        pwa.pwa_nll_grad_for_hvp(h, thd, nll, g)
        pwa.pwa_hvp_cached(h, vd, hv)
        assert err(nll.item()) < 1e-10
        assert rel_l2(g.cpu().numpy(), g0) < 1e-8 and rel_l2(hv.cpu().numpy(), h0) < 1e-8, name
        fr = torch.zeros(R, dtype=torch.float64, device=dev)
        pwa.pwa_fit_fractions(h, thd, fr)
        from oracle.fractions import fit_fractions
        assert np.max(np.abs(fr.cpu().numpy() - fit_fractions(om, th)) / fit_fractions(om, th)) < 1e-10
        assert pwa.pwa_status_flags(h) == 0
    finally:
        pwa.pwa_destroy(h)
