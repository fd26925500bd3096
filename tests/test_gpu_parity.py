"""GPU parity: the CUDA path (through the C ABI of include/pwa.h) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json's north_star: NLL 1e-10 relative,
gradient and HVP 1e-8 relative L2 (denominators: DESIGN.md S12); repeat runs bit-identical.

Sizes: BASELINE.json config shapes scaled to what the 80-bit oracle finishes in seconds, always with a
ragged tail (event counts that are not multiples of 32 or of any tile size).
"""
import numpy as np
import pytest
import torch

from helpers import rel_l2

pytestmark = pytest.mark.gpu

NLL_TOL = 1e-10
VEC_TOL = 1e-8

# (config index, n_mc, n_data): config shapes of BASELINE.json at oracle-sized event counts
CASES = [(1, 50_000, 10_000), (2, 20_011, 3_001), (3, 12_345, 1_537), (4, 2_049, 517), (6, 30_001, 1_999)]


@pytest.fixture(scope="module")
def pwa():
    import paper_2403_09225_b200 as p
    from paper_2403_09225_b200.build import build
    build()
    p.load()
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    return p


_CACHE = {}


def _case(pwa, oracle_mod, idx, n_mc, n_data):
    key = (idx, n_mc, n_data)
    if key not in _CACHE:
        import workloads
        cfg = workloads.CONFIGS[idx].scaled(n_mc, n_data)
        w = workloads.make_workload(cfg, "cpu", chunk=1 << 13)
        om = oracle_mod.model_from_workload(w)
        gm = pwa.Model(w)
        _CACHE[key] = (cfg, w, om, gm)
    return _CACHE[key]


def _thetas(cfg):
    import workloads
    return [workloads.theta_true(cfg).numpy()] + [workloads.random_start(cfg, k).numpy() for k in range(3)]


def _nll_err(a, b):
    return abs(float(a) - float(b)) / max(abs(float(b)), 1.0)


@pytest.mark.parametrize("idx,n_mc,n_data", CASES)
def test_fused_sweep_matches_oracle(pwa, oracle_mod, idx, n_mc, n_data):
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    for k, th in enumerate(_thetas(cfg)):
        v = workloads.direction(cfg, k).numpy()
        f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
        f, g, hv = gm.nll_grad_hvp(th, v)
        assert _nll_err(f, f0) < NLL_TOL, (idx, k, f, float(f0))
        assert rel_l2(g, g0) < VEC_TOL, (idx, k)
        assert rel_l2(hv, h0) < VEC_TOL, (idx, k)
        assert pwa.pwa_status_flags(gm.h) == 0


@pytest.mark.parametrize("idx,n_mc,n_data", CASES[:4])
def test_separate_calls_match_oracle(pwa, oracle_mod, idx, n_mc, n_data):
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    th = _thetas(cfg)[1]
    v = workloads.direction(cfg, 5).numpy()
    f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
    assert _nll_err(gm.nll(th), f0) < NLL_TOL
    f, g = gm.nll_grad(th)
    assert _nll_err(f, f0) < NLL_TOL and rel_l2(g, g0) < VEC_TOL
    assert rel_l2(gm.hvp(th, v), h0) < VEC_TOL


@pytest.mark.parametrize("idx,n_mc,n_data", CASES[:3])
def test_repeat_runs_are_bit_identical(pwa, oracle_mod, idx, n_mc, n_data):
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    th, v = _thetas(cfg)[0], workloads.direction(cfg, 0).numpy()
    a = gm.nll_grad_hvp(th, v)
    for _ in range(3):
        b = gm.nll_grad_hvp(th, v)
        assert np.float64(a[0]).tobytes() == np.float64(b[0]).tobytes()
        assert a[1].tobytes() == b[1].tobytes() and a[2].tobytes() == b[2].tobytes()
    # a second handle on the same arrays gives the same bits too
    gm2 = pwa.Model(w)
    c = gm2.nll_grad_hvp(th, v)
    assert a[1].tobytes() == c[1].tobytes() and a[2].tobytes() == c[2].tobytes()
    gm2.close()


def test_invariance_directions_on_device(pwa, oracle_mod):
    """Global phase: H 1_phi = 0, g.1_phi = 0; common scale: g.u = 0, (H u)_a = -g_a (P2)."""
    cfg, w, om, gm = _case(pwa, oracle_mod, *CASES[1])
    th = _thetas(cfg)[2]
    P = cfg.n_par
    ones_phi = np.zeros(P); ones_phi[1::4] = 1.0
    u = np.zeros(P); u[0::4] = th[0::4]
    f, g, h1 = gm.nll_grad_hvp(th, ones_phi)
    scale = np.linalg.norm(gm.hvp(th, np.ones(P)))
    assert np.linalg.norm(h1) < 1e-9 * scale
    assert abs(g @ ones_phi) < 1e-9 * np.linalg.norm(g) * np.sqrt(P)
    assert abs(g @ u) < 1e-9 * np.linalg.norm(g) * np.linalg.norm(u)
    hu = gm.hvp(th, u)
    assert np.linalg.norm(hu[0::4] + g[0::4]) < 1e-8 * max(np.linalg.norm(g[0::4]), 1e-300) + 1e-9 * scale
    # the oracle agrees on those special directions as well
    _, _, h0 = oracle_mod.nll_grad_hvp(om, th, u, "ld")
    assert rel_l2(hu, h0) < VEC_TOL


def test_shard_additivity_through_raw_sums(pwa, oracle_mod):
    """PAPER.md:80-96 (Eqs. 4-7): raw sums of two disjoint shards add to the raw sums of the whole."""
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, *CASES[2])
    th, v = _thetas(cfg)[1], workloads.direction(cfg, 1).numpy()
    nm, nd = cfg.n_mc, cfg.n_data
    cut_m, cut_d = 5_003, 700
    parts = []
    for (m0, m1, d0, d1) in ((0, cut_m, 0, cut_d), (cut_m, nm, cut_d, nd)):
        h = pwa.pwa_create(w.res_chan, w.data_mass[:, d0:d1].contiguous(), w.data_amp[:, :, d0:d1].contiguous(),
                           None if w.data_weight is None else w.data_weight[d0:d1].contiguous(),
                           w.mc_mass[:, m0:m1].contiguous(), w.mc_amp[:, :, m0:m1].contiguous())
        raw = torch.zeros(pwa.pwa_raw_size(h), dtype=torch.float64, device="cuda")
        pwa.pwa_raw_sums(h, torch.tensor(th, device="cuda"), torch.tensor(v, device="cuda"), raw)
        parts.append(raw.clone())
        torch.cuda.synchronize()
        pwa.pwa_destroy(h)
    total = parts[0] + parts[1]
    whole = gm.raw_sums(th, v)
    assert float(total[3]) == nm and float(whole[3]) == nm
    assert rel_l2(total.cpu().numpy(), whole.cpu().numpy()) < 1e-13
    nll = torch.zeros(1, dtype=torch.float64, device="cuda")
    g = torch.zeros(cfg.n_par, dtype=torch.float64, device="cuda")
    hv = torch.zeros(cfg.n_par, dtype=torch.float64, device="cuda")
    pwa.pwa_combine(gm.h, total, torch.tensor(v, device="cuda"), nll, g, hv)
    f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
    assert _nll_err(nll.item(), f0) < NLL_TOL
    assert rel_l2(g.cpu().numpy(), g0) < VEC_TOL and rel_l2(hv.cpu().numpy(), h0) < VEC_TOL
    # and the raw vector itself matches the oracle's raw sums block by block
    sd, gd, hd = oracle_mod.raw_sums(om, "data", th, v, "ld")
    sm, gG, hG = oracle_mod.raw_sums(om, "mc", th, v, "ld")
    P = cfg.n_par
    wh = whole.cpu().numpy()
    assert _nll_err(wh[0], sd[0]) < NLL_TOL and _nll_err(wh[1], sd[1]) < 1e-13 and _nll_err(wh[2], sm[0]) < 1e-12
    for k, ref in enumerate((gd, gG, hd, hG)):
        assert rel_l2(wh[4 + k * P: 4 + (k + 1) * P], ref) < VEC_TOL, k


def test_host_entry_point(pwa, oracle_mod):
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, *CASES[1])
    th, v = _thetas(cfg)[0], workloads.direction(cfg, 2).numpy()
    nll = np.zeros(1); g = np.zeros(cfg.n_par); hv = np.zeros(cfg.n_par)
    pwa.pwa_nll_grad_hvp_host(gm.h, np.ascontiguousarray(th), np.ascontiguousarray(v), nll, g, hv)
    f1, g1, h1 = gm.nll_grad_hvp(th, v)
    assert nll[0] == f1 and g.tobytes() == g1.tobytes() and hv.tobytes() == h1.tobytes()
    g2 = np.zeros(cfg.n_par)
    pwa.pwa_nll_grad_hvp_host(gm.h, np.ascontiguousarray(th), None, nll, g2, None)
    f0, g0, _ = oracle_mod.nll_grad_hvp(om, th, None, "ld")
    assert _nll_err(nll[0], f0) < NLL_TOL and rel_l2(g2, g0) < VEC_TOL


def test_zero_mass_resonance_on_a_ragged_tail(pwa, oracle_mod):
    """M_r = 0 makes |D|^2 = m^4: finite on every event, but the zero-filled lanes beyond the ragged end of the last
    tile would see 1/0 without the kernel's denominator floor (pwa_sweep_lanes.cuh, resonance_constants)."""
    import workloads
    for case in (CASES[1], CASES[2]):
        cfg, w, om, gm = _case(pwa, oracle_mod, *case)
        assert cfg.n_mc % 32 != 0 and cfg.n_data % 32 != 0
        th = _thetas(cfg)[1].copy()
        th[2], th[3] = 0.0, 0.0       # resonance 0: M = 0, Gamma = 0
        th[6] = 0.0                   # resonance 1: M = 0, Gamma > 0
        v = workloads.direction(cfg, 7).numpy()
        f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
        f, g, hv = gm.nll_grad_hvp(th, v)
        assert np.isfinite(f) and np.all(np.isfinite(g)) and np.all(np.isfinite(hv))
        assert _nll_err(f, f0) < NLL_TOL and rel_l2(g, g0) < VEC_TOL and rel_l2(hv, h0) < VEC_TOL
        assert pwa.pwa_status_flags(gm.h) == 0


@pytest.mark.parametrize("case,combo", [(CASES[2], 10), (CASES[2], 11), (CASES[1], 10), (CASES[0], 11), (CASES[4], 10),
                                        (CASES[2], 5), (CASES[2], 6), (CASES[2], 12), (CASES[1], 3), (CASES[1], 1), (CASES[0], 0),
                                        (CASES[1], 2), (CASES[1], 13), (CASES[4], 13),
                                        (CASES[2], 14), (CASES[2], 15), (CASES[1], 14), (CASES[0], 15), (CASES[3], 15),
                                        (CASES[4], 16), (CASES[4], 17), (CASES[4], 20), (CASES[0], 16), (CASES[1], 18), (CASES[1], 21),
                                        (CASES[2], 19), (CASES[2], 22), (CASES[2], 23), (CASES[2], 24), (CASES[2], 25), (CASES[1], 23)])
def test_every_kernel_shape_matches_oracle(pwa, oracle_mod, case, combo, monkeypatch):
    """The handle normally picks one shape per (n_res, n_hel); PWA_COMBO forces another entry of kLanesCombos
    (csrc/pwa_internal.h) so that every instantiated shape - 8-event swizzled tiles over planes and over the tiled store,
    both producer kinds, every slice count - is compared with the oracle on ragged inputs, not only the ones the default
    choice reaches."""
    import workloads
    cfg, w, om, _ = _case(pwa, oracle_mod, *case)
    monkeypatch.setenv("PWA_COMBO", str(combo))
    gm = pwa.Model(w)
    monkeypatch.delenv("PWA_COMBO")
    try:
        name = pwa.pwa_kernel_variant(gm.h)
        assert name.startswith("lanes"), name
        if combo in (10, 11, 22, 24):
            assert "tile=8," in name, name
        if combo in (14, 15, 23, 25):  # the library-owned tiled store (this handle owns a copy of the events)
            assert "tile=8t," in name, name
        th = _thetas(cfg)[2]
        v = workloads.direction(cfg, 9).numpy()
        f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
        f, g, hv = gm.nll_grad_hvp(th, v)
        assert _nll_err(f, f0) < NLL_TOL, (name, f, float(f0))
        assert rel_l2(g, g0) < VEC_TOL and rel_l2(hv, h0) < VEC_TOL, name
        assert _nll_err(gm.nll(th), f0) < NLL_TOL
        f1, g1 = gm.nll_grad(th)
        assert _nll_err(f1, f0) < NLL_TOL and rel_l2(g1, g0) < VEC_TOL
        f2, g2, hv2 = gm.nll_grad_hvp(th, v)
        assert g.tobytes() == g2.tobytes() and hv.tobytes() == hv2.tobytes()
    finally:
        gm.close()


@pytest.mark.parametrize("case", [CASES[1], CASES[2], CASES[3]])
@pytest.mark.parametrize("stages,nprod", [(0, 1), (0, 2), (0, 3), (2, 4), (3, 4), (4, 4), (5, 4), (6, 4), (7, 4)])
def test_ring_depth_and_producer_count_do_not_change_a_bit(pwa, oracle_mod, case, stages, nprod, monkeypatch):
    """The ring of stages is filled by up to four producer threads; their count must divide the stage
    count so that a stage is always refilled by the same thread, and the stage count must be a multiple of the tiles
    that different warps consume at the same time.  Whatever PWA_STAGES / PWA_NPROD ask for - rings shorter than the
    producer count, odd depths (a depth the shape cannot run with is ignored) - the results are the default
    configuration's, bit for bit, in every mode (the arithmetic does not depend on who copied a tile)."""
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, *case)
    th, v = _thetas(cfg)[1], workloads.direction(cfg, 2).numpy()
    want = (gm.nll_grad_hvp(th, v), gm.nll(th), gm.nll_grad(th), gm.nll_grad_for_hvp(th), gm.hvp_cached(v))
    if stages:
        monkeypatch.setenv("PWA_STAGES", str(stages))
    monkeypatch.setenv("PWA_NPROD", str(nprod))
    other = pwa.Model(w)
    monkeypatch.delenv("PWA_NPROD")
    if stages:
        monkeypatch.delenv("PWA_STAGES")
    try:
        name = pwa.pwa_kernel_variant(other.h)
        assert name.startswith("lanes"), name
        got = (other.nll_grad_hvp(th, v), other.nll(th), other.nll_grad(th), other.nll_grad_for_hvp(th), other.hvp_cached(v))
        flat = lambda r: np.concatenate([np.atleast_1d(np.asarray(x, dtype=np.float64)).ravel() for x in (r if isinstance(r, tuple) else (r,))])
        # a ring of fewer than four stages has no two-events-per-lane kernel (config-3 shape): the one-event kernel of the
        # same shape sums in another order - equal to rounding there, the same bits everywhere else
        other_kernel = case == CASES[2] and stages in (2, 3)
        for a, b in zip(got, want):
            if other_kernel:
                assert rel_l2(flat(a), flat(b)) < 1e-11, name
            else:
                assert flat(a).tobytes() == flat(b).tobytes(), name
    finally:
        other.close()


def test_one_event_fused_kernel_of_the_config3_shape(pwa, oracle_mod, monkeypatch):
    """The fused calls of the 4 x 8-slice shape run the two-events-per-lane kernel (csrc/pwa_sweep_pair.cuh); PWA_PAIR=0
    keeps the one-event kernel of the same shape reachable - both against the oracle, and against each other (the two
    sum in a different order: equal to rounding, not bit for bit)."""
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, *CASES[2])
    th, v = _thetas(cfg)[3], workloads.direction(cfg, 11).numpy()
    f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
    l0 = pwa.pwa_kernel_launches(gm.h)
    f2, g2, h2 = gm.nll_grad_hvp(th, v)
    assert pwa.pwa_kernel_launches(gm.h) - l0 == 2
    monkeypatch.setenv("PWA_PAIR", "0")
    f1, g1, h1 = gm.nll_grad_hvp(th, v)
    monkeypatch.delenv("PWA_PAIR")
    for f, g, hv in ((f1, g1, h1), (f2, g2, h2)):
        assert _nll_err(f, f0) < NLL_TOL and rel_l2(g, g0) < VEC_TOL and rel_l2(hv, h0) < VEC_TOL
    assert rel_l2(g1, g2) < 1e-12 and rel_l2(h1, h2) < 1e-12 and (g1.tobytes() != g2.tobytes() or h1.tobytes() != h2.tobytes())


def test_many_repeats_bit_identical_under_load(pwa, oracle_mod):
    """A race in the TMA ring, the shared-memory exchange rows or the ticketed reduction would show up as a changed
    bit in some repeat (compute-sanitizer is not available on the GPU pool).  150 back-to-back evaluations in all
    three kernel modes on a config-3-shaped sample large enough to wrap the ring many times."""
    import workloads
    cfg = workloads.CONFIGS[3].scaled(300_007, 30_011)
    w = workloads.make_workload(cfg, torch.device("cuda", 0))
    gm = pwa.Model(w, borrow=True)
    try:
        dev = torch.device("cuda", 0)
        th = torch.tensor(workloads.random_start(cfg, 1).numpy(), device=dev)
        v = torch.tensor(workloads.direction(cfg, 2).numpy(), device=dev)
        P = cfg.n_par
        outs = torch.zeros(150, 2 + 3 * P, dtype=torch.float64, device=dev)
        for k in range(150):
            row = outs[k]
            pwa.pwa_nll_grad_hvp(gm.h, th, v, row[0:1], row[2:2 + P], row[2 + P:2 + 2 * P])
            if k % 3 == 0:
                pwa.pwa_nll(gm.h, th, row[1:2])
            else:
                pwa.pwa_nll_grad(gm.h, th, row[1:2], row[2 + 2 * P:2 + 3 * P])
        torch.cuda.synchronize()
        o = outs.cpu().numpy()
        assert np.all(np.isfinite(o))
        for k in range(1, 150):
            assert o[k, 0].tobytes() == o[0, 0].tobytes() and o[k, 2:2 + 2 * P].tobytes() == o[0, 2:2 + 2 * P].tobytes(), k
            assert o[k, 1].tobytes() == o[0, 1].tobytes() or k % 3 != 0
        # the three modes agree on the NLL to rounding (different instruction mixes, same sums)
        assert abs(o[0, 1] - o[0, 0]) <= 1e-12 * abs(o[0, 0]) and abs(o[1, 1] - o[0, 0]) <= 1e-12 * abs(o[0, 0])
        gr = [k for k in range(150) if k % 3 != 0]
        for k in gr[1:]:
            assert o[k, 2 + 2 * P:].tobytes() == o[gr[0], 2 + 2 * P:].tobytes(), k
    finally:
        gm.close()


@pytest.mark.parametrize("idx,n_mc,n_data", CASES)
def test_fit_fractions_match_oracle(pwa, oracle_mod, idx, n_mc, n_data):
    """pwa_fit_fractions (S20) against oracle/fractions.py, element by element, 1e-10 relative."""
    from oracle.fractions import fit_fractions
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    for th in _thetas(cfg)[:2]:
        f0 = fit_fractions(om, th)
        f = gm.fit_fractions(th)
        assert f.shape == f0.shape and np.all(np.isfinite(f))
        assert np.max(np.abs(f - f0) / f0) < 1e-10, idx
        assert gm.fit_fractions(th).tobytes() == f.tobytes()  # repeat runs bit-identical


@pytest.mark.parametrize("idx,n_mc,n_data", CASES)
def test_split_evaluation_matches_oracle(pwa, oracle_mod, idx, n_mc, n_data):
    """pwa_nll_grad_for_hvp + pwa_hvp_cached (the Newton-CG split of include/pwa.h) against the oracle: NLL and
    gradient from the keeping call, then several HVPs at the kept theta with other calls in between."""
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    for k, th in enumerate(_thetas(cfg)[:2]):
        f0, g0, _ = oracle_mod.nll_grad_hvp(om, th, None, "ld")
        f, g = gm.nll_grad_for_hvp(th)
        assert _nll_err(f, f0) < NLL_TOL and rel_l2(g, g0) < VEC_TOL
        other = _thetas(cfg)[3]
        for j in range(3):
            v = workloads.direction(cfg, 10 + j).numpy()
            h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")[2]
            hv = gm.hvp_cached(v)
            assert rel_l2(hv, h0) < VEC_TOL, (idx, k, j)
            assert rel_l2(hv, gm.hvp(th, v)) < 1e-12           # same sums, other association
            gm.nll(other); gm.nll_grad(other)                    # what is kept survives other evaluations
            assert gm.hvp_cached(v).tobytes() == hv.tobytes()
        assert pwa.pwa_status_flags(gm.h) == 0


def test_hvp_cached_needs_a_keeping_call(pwa, oracle_mod):
    import workloads
    cfg, w, om, _ = _case(pwa, oracle_mod, *CASES[0])
    gm = pwa.Model(w)
    try:
        with pytest.raises(pwa.PwaError) as e:
            gm.hvp_cached(workloads.direction(cfg, 0).numpy())
        assert e.value.status == 1
    finally:
        gm.close()


@pytest.mark.parametrize("idx,n_mc,n_data", [CASES[1], CASES[2]])
def test_unconstrained_parameter_domain(pwa, oracle_mod, idx, n_mc, n_data):
    """Reading S7: the evaluation calls take unconstrained reals.  One coupling exactly zero among non-zero
    ones (its d/da entry stays finite and non-zero: e^{i phi} B S), a negative modulus, a negative width (the pole moves
    to the other half plane), phases of order 1e3 (sincos argument reduction) - every entry point against the oracle."""
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    base = workloads.random_start(cfg, 2).numpy()
    v = workloads.direction(cfg, 6).numpy()
    variants = {}
    t = base.copy(); t[4 * 1] = 0.0; variants["a_1 = 0"] = t
    t = base.copy(); t[4 * 0] = -t[4 * 0]; t[4 * 2] = -0.37; variants["a < 0"] = t
    t = base.copy(); t[4 * 1 + 3] = -t[4 * 1 + 3]; variants["Gamma_1 < 0"] = t
    t = base.copy(); t[1::4] += 1000.0 * np.where(np.arange(cfg.n_res) % 2 == 0, 1.0, -1.0); variants["|phi| ~ 1e3"] = t
    t = base.copy(); t[4 * 1] = 0.0; t[4 * 0] = -1.2; t[4 * 2 + 3] = -0.11; t[1::4] -= 777.0; variants["all at once"] = t
    for name, th in variants.items():
        f0, g0, h0 = oracle_mod.nll_grad_hvp(om, th, v, "ld")
        f, g, hv = gm.nll_grad_hvp(th, v)
        assert _nll_err(f, f0) < NLL_TOL, (name, f, float(f0))
        assert rel_l2(g, g0) < VEC_TOL and rel_l2(hv, h0) < VEC_TOL, name
        assert pwa.pwa_status_flags(gm.h) == 0, name
        assert _nll_err(gm.nll(th), f0) < NLL_TOL, name
        f1, g1 = gm.nll_grad_for_hvp(th)
        assert _nll_err(f1, f0) < NLL_TOL and rel_l2(g1, g0) < VEC_TOL, name
        assert rel_l2(gm.hvp_cached(v), h0) < VEC_TOL, name
        if name == "a_1 = 0":
            assert g[4] != 0.0 and np.isfinite(g[4])
            assert abs(g[4] - float(g0[4])) <= 1e-8 * abs(float(g0[4]))


def test_handle_used_from_another_host_thread(pwa, oracle_mod):
    """PAPER.md:98 runs one host thread per GPU.  Every C-ABI entry binds the calling thread to the handle's device for
    the duration of the call and restores the caller's current device (csrc/pwa_internal.h: DeviceGuard), so a handle
    created in one thread gives the same bits when it is called from a fresh thread (whose CUDA context state is the
    default one), and the caller's current device is left as it was.  (This pool has one GPU per box: the case of a
    thread whose current device is ANOTHER ordinal cannot be run here.)"""
    import threading
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, *CASES[1])
    th = _thetas(cfg)[1]
    v = workloads.direction(cfg, 3).numpy()
    want = gm.nll_grad_hvp(th, v)
    out = {}

    def work():
        before = torch.cuda.current_device()
        out["res"] = gm.nll_grad_hvp(th, v)
        out["fit"] = gm.fit(th, None)[1].status
        out["dev"] = (before, torch.cuda.current_device())

    t = threading.Thread(target=work)
    t.start()
    t.join()
    assert out["res"][0] == want[0] and out["res"][1].tobytes() == want[1].tobytes() and out["res"][2].tobytes() == want[2].tobytes()
    assert out["dev"][0] == out["dev"][1] and out["fit"] in (0, 5)
