"""pwa_nll_grad_hvp_static (include/pwa.h): the fused evaluation without a handle and without any device allocation,
its scratch in a fixed array inside the library.  Checked against the existing path - pwa_nll_grad_hvp on a handle made
from the same buffers - within the tolerances of the parity tests (NLL 1e-10 relative, gradient and HVP 1e-8 relative
L2), on two calls in a row with different parameters (the array keeps the first call's contents), then a repeat of the
first call, which must reproduce it bit for bit.

This file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide another test.
"""
import ctypes

import numpy as np
import pytest

from helpers import random_theta, rel_l2

NLL_TOL = 1e-10
VEC_TOL = 1e-8

# (R, H, C, n_data, n_mc, weighted): BASELINE.json's config-3 shape (the handle runs the two-event tiled kernel), the
# largest model the fixed array serves, a tiny one with fewer rows of events than blocks, more than 4 helicities
SHAPES = [(30, 2, 3, 1_537, 12_345, True), (64, 4, 3, 333, 2_049, False), (2, 2, 1, 7, 100, True), (6, 5, 2, 50, 500, True)]


@pytest.fixture(scope="module")
def pwa():
    import paper_2403_09225_b200 as p
    from paper_2403_09225_b200.build import build
    build()
    p.load()
    return p


def _inputs(R, H, C, nd, nm, weighted):
    import torch
    rs = np.random.RandomState(77 * R + 7 * H + C)
    dev = torch.device("cuda", 0)
    t = lambda x: torch.from_numpy(np.ascontiguousarray(x)).to(dev)
    res_chan = (np.arange(R) % C).astype(np.int32)
    data = (t(rs.uniform(0.3, 3.0, size=(C, nd))), t(rs.normal(size=(R, H, nd, 2))),
            t(rs.uniform(0.5, 1.5, size=nd)) if weighted else None)
    mc = (t(rs.uniform(0.3, 3.0, size=(C, nm))), t(rs.normal(size=(R, H, nm, 2))))
    points = [(t(random_theta(11 + k + R, R)), t(rs.normal(size=4 * R))) for k in range(2)]
    return res_chan, data, mc, points


def _close(pwa, a, b):
    assert abs(a[0] - b[0]) / max(abs(b[0]), 1.0) < NLL_TOL, (a[0], b[0])
    assert rel_l2(a[1], b[1]) < VEC_TOL and rel_l2(a[2], b[2]) < VEC_TOL


@pytest.mark.gpu
@pytest.mark.parametrize("R,H,C,nd,nm,weighted", SHAPES)
def test_static_entry_point_matches_the_handle_path(pwa, R, H, C, nd, nm, weighted):
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    dev = torch.device("cuda", 0)
    res_chan, (dm, da, dw), (mm, ma), points = _inputs(R, H, C, nd, nm, weighted)
    P = 4 * R
    out = lambda: (torch.zeros(1, dtype=torch.float64, device=dev), torch.zeros(P, dtype=torch.float64, device=dev),
                   torch.zeros(P, dtype=torch.float64, device=dev))
    host = lambda o: (o[0].item(), o[1].cpu().numpy().copy(), o[2].cpu().numpy().copy())

    h = pwa.pwa_create(torch.from_numpy(res_chan), dm, da, dw, mm, ma, borrow=True)
    try:
        want = []
        for th, v in points:
            o = out()
            pwa.pwa_nll_grad_hvp(h, th, v, *o)
            want.append(host(o))
            assert pwa.pwa_status_flags(h) == 0
    finally:
        pwa.pwa_destroy(h)

    static = lambda th, v, o: pwa.pwa_nll_grad_hvp_static(res_chan, dm, da, dw, mm, ma, th, v, *o)
    # two calls in a row (different theta and v: the second finds the first call's sums in the array) ...
    got, outs = [], [out() for _ in points]
    for k, (th, v) in enumerate(points):
        o = outs[k]
        static(th, v, o)
        got.append(host(o))
        if k == 0:
            torch.cuda.synchronize()
            free_after_first = torch.cuda.mem_get_info(dev)[0]
    for g, w in zip(got, want):
        _close(pwa, g, w)
    # ... the second of which took no device memory
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(dev)[0] >= free_after_first
    # a repeat of the first call after another one: bit-identical
    o = out()
    static(*points[0], o)
    again = host(o)
    assert again[0] == got[0][0] and np.array_equal(again[1], got[0][1]) and np.array_equal(again[2], got[0][2])

    # outputs not wanted may be NULL: the lighter sweeps (value only; value and gradient) agree to rounding
    th, v = points[1]
    nll = torch.zeros(1, dtype=torch.float64, device=dev)
    pwa.pwa_nll_grad_hvp_static(res_chan, dm, da, dw, mm, ma, th, None, nll, None, None)
    assert abs(nll.item() - want[1][0]) / max(abs(want[1][0]), 1.0) < NLL_TOL
    nll2, g2, _ = out()
    pwa.pwa_nll_grad_hvp_static(res_chan, dm, da, dw, mm, ma, th, v, nll2, g2, None)
    assert abs(nll2.item() - want[1][0]) / max(abs(want[1][0]), 1.0) < NLL_TOL
    assert rel_l2(g2.cpu().numpy(), want[1][1]) < VEC_TOL


@pytest.mark.gpu
def test_static_entry_point_on_a_side_stream(pwa):
    import torch
    dev = torch.device("cuda", 0)
    R, H, C = 10, 3, 2
    res_chan, (dm, da, dw), (mm, ma), points = _inputs(R, H, C, 3_001, 20_011, False)
    th, v = points[0]
    torch.cuda.synchronize()
    s = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(s):
        o = [torch.zeros(1, dtype=torch.float64, device=dev)] + [torch.zeros(4 * R, dtype=torch.float64, device=dev) for _ in range(2)]
        pwa.pwa_nll_grad_hvp_static(res_chan, dm, da, dw, mm, ma, th, v, *o, stream=s.cuda_stream)
        pwa.pwa_nll_grad_hvp_static(res_chan, dm, da, dw, mm, ma, th, v, *o, stream=s.cuda_stream)
    s.synchronize()
    h = pwa.pwa_create(torch.from_numpy(res_chan), dm, da, dw, mm, ma, borrow=True)
    try:
        w = [torch.zeros(1, dtype=torch.float64, device=dev)] + [torch.zeros(4 * R, dtype=torch.float64, device=dev) for _ in range(2)]
        pwa.pwa_nll_grad_hvp(h, th, v, *w)
        torch.cuda.synchronize()
    finally:
        pwa.pwa_destroy(h)
    _close(pwa, (o[0].item(), o[1].cpu().numpy(), o[2].cpu().numpy()), (w[0].item(), w[1].cpu().numpy(), w[2].cpu().numpy()))


def _host_desc(pwa, R, **over):
    keep = {"ch": np.zeros(R, dtype=np.int32), "mass": np.ones((1, 8)), "amp": np.ones((R, 1, 8, 2))}
    d = pwa.pwa_model_desc()
    d.n_res, d.n_hel, d.n_chan = R, 1, 1
    d.res_chan = keep["ch"].ctypes.data
    for s in (d.data, d.mc):
        s.n_events, s.stride, s.mass, s.amp, s.weight = 8, 0, keep["mass"].ctypes.data, keep["amp"].ctypes.data, None
    d.mem, d.borrow, d.device, d.stream = pwa.PWA_MEM_DEVICE, 1, 0, None
    for k, v in over.items():
        setattr(d, k, v)
    return d, keep


def test_sizes_beyond_the_fixed_array_are_rejected_with_a_clear_error(pwa):
    """Argument checks come before any CUDA call: they need no device."""
    lib = pwa.load()
    assert pwa.PWA_STATIC_MAX_RES == 64
    x = np.zeros(8)
    ptr = ctypes.c_void_p(x.ctypes.data)
    d, keep = _host_desc(pwa, pwa.PWA_STATIC_MAX_RES + 1)
    assert lib.pwa_nll_grad_hvp_static(ctypes.byref(d), ptr, ptr, ptr, ptr, ptr) == pwa.PWA_ERR_INVALID_ARG
    msg = pwa.pwa_last_error(None)
    assert "PWA_STATIC_MAX_RES" in msg and "65" in msg, msg
    for bad in (dict(n_hel=9), dict(n_chan=0), dict(mem=pwa.PWA_MEM_HOST), dict(n_res=0)):
        d, keep = _host_desc(pwa, 4, **bad)
        assert lib.pwa_nll_grad_hvp_static(ctypes.byref(d), ptr, ptr, ptr, ptr, ptr) == pwa.PWA_ERR_INVALID_ARG, bad
        assert "pwa_nll_grad_hvp_static" in pwa.pwa_last_error(None)
    d, keep = _host_desc(pwa, 4)
    assert lib.pwa_nll_grad_hvp_static(ctypes.byref(d), ptr, ptr, None, None, None) == pwa.PWA_ERR_INVALID_ARG  # no output
    assert lib.pwa_nll_grad_hvp_static(ctypes.byref(d), ptr, None, ptr, ptr, ptr) == pwa.PWA_ERR_INVALID_ARG   # hv without v
