"""The library-owned TILED event store (copy-mode handles of shapes that need 8-event tiles: more than 32 resonances
with a stage of 32 events that does not fit twice in shared memory, e.g. BASELINE.json's config 4, R = 100, H = 4).
Same kernels, same event -> thread map and the same order of additions as the tensor-copy path over borrowed planes, so
every result must be the same BITS; the oracle parity of these shapes is in test_gpu_parity.py / test_gpu_shapes.py,
whose handles are copy-mode handles."""
import numpy as np
import pytest
import torch

from helpers import random_theta, rel_l2

pytestmark = pytest.mark.gpu

# (R, H, C, n_data, n_mc, weighted); even event counts (borrowed planes need an even stride for the tensor copies), ragged
# against the 8-event tile; the last case spans several staging chunks of the host upload
SHAPES = [(100, 4, 3, 518, 2_050, False), (100, 4, 3, 2, 10, True), (64, 4, 2, 334, 1_002, True), (40, 4, 1, 64, 640, False),
          (128, 3, 3, 258, 1_500, True), (100, 4, 3, 1_004, 45_002, True)]


@pytest.fixture(scope="module")
def pwa():
    import paper_2403_09225_b200 as p
    from paper_2403_09225_b200.build import build
    build()
    p.load()
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    return p


def _all_results(pwa, h, th, v, R):
    dev = th.device
    P = 4 * R
    z = lambda n: torch.zeros(n, dtype=torch.float64, device=dev)
    out = {}
    nll, g, hv = z(1), z(P), z(P)
    pwa.pwa_nll_grad_hvp(h, th, v, nll, g, hv)
    out["fused"] = (nll.item(), g.cpu().numpy().copy(), hv.cpu().numpy().copy())
    pwa.pwa_nll(h, th, nll)
    out["nll"] = nll.item()
    pwa.pwa_nll_grad(h, th, nll, g)
    out["grad"] = (nll.item(), g.cpu().numpy().copy())
    pwa.pwa_nll_grad_for_hvp(h, th, nll, g)
    pwa.pwa_hvp_cached(h, v, hv)
    out["split"] = (nll.item(), g.cpu().numpy().copy(), hv.cpu().numpy().copy())
    raw = z(4 + 4 * P)
    pwa.pwa_raw_sums(h, th, v, raw)
    out["raw"] = raw.cpu().numpy().copy()
    fr = z(R)
    pwa.pwa_fit_fractions(h, th, fr)
    out["frac"] = fr.cpu().numpy().copy()
    assert pwa.pwa_status_flags(h) == 0
    return out


def _same(a, b):
    if isinstance(a, tuple):
        return all(_same(x, y) for x, y in zip(a, b))
    return np.array_equal(np.asarray(a), np.asarray(b))


@pytest.mark.parametrize("R,H,C,nd,nm,weighted", SHAPES)
def test_tiled_store_gives_the_bits_of_the_borrowed_planes(pwa, R, H, C, nd, nm, weighted):
    rs = np.random.RandomState(31 * R + H + nd)
    dev = torch.device("cuda", 0)
    res_chan = torch.from_numpy((np.arange(R) % C).astype(np.int32))
    host = [torch.from_numpy(rs.uniform(0.3, 3.0, size=(C, nd))), torch.from_numpy(rs.normal(size=(R, H, nd, 2))),
            torch.from_numpy(rs.uniform(0.5, 1.5, size=nd)) if weighted else None,
            torch.from_numpy(rs.uniform(0.3, 3.0, size=(C, nm))), torch.from_numpy(rs.normal(size=(R, H, nm, 2)))]
    on_dev = [None if t is None else t.to(dev) for t in host]
    th = torch.tensor(random_theta(3 + R, R), device=dev)
    v = torch.tensor(rs.normal(size=4 * R), device=dev)
    results, names = {}, {}
    for kind, bufs, borrow in (("borrowed", on_dev, True), ("copy of device planes", on_dev, False), ("copy of host planes", host, False)):
        h = pwa.pwa_create(res_chan, *bufs, borrow=borrow)
        try:
            names[kind] = pwa.pwa_kernel_variant(h)
            results[kind] = _all_results(pwa, h, th, v, R)
        finally:
            pwa.pwa_destroy(h)
    assert "tile=8," in names["borrowed"], names
    assert "tile=8t," in names["copy of device planes"] and "tile=8t," in names["copy of host planes"], names
    ref = results["borrowed"]
    for kind in ("copy of device planes", "copy of host planes"):
        for key, val in results[kind].items():
            assert _same(val, ref[key]), (kind, key)


def test_tiled_store_can_be_switched_off(pwa, monkeypatch):
    R, H, C, nd, nm = 100, 4, 3, 100, 500
    rs = np.random.RandomState(5)
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x))
    args = (t((np.arange(R) % C).astype(np.int32)), t(rs.uniform(0.3, 3.0, size=(C, nd))), t(rs.normal(size=(R, H, nd, 2))), None,
            t(rs.uniform(0.3, 3.0, size=(C, nm))), t(rs.normal(size=(R, H, nm, 2))))
    monkeypatch.setenv("PWA_TILED", "0")
    h = pwa.pwa_create(*args)
    try:
        assert "tile=8," in pwa.pwa_kernel_variant(h)
    finally:
        pwa.pwa_destroy(h)
    monkeypatch.delenv("PWA_TILED")
    h = pwa.pwa_create(*args)
    try:
        assert "tile=8t," in pwa.pwa_kernel_variant(h)
    finally:
        pwa.pwa_destroy(h)
