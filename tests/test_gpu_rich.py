"""The richer model on the GPU (pwa_create_rich; readings S21, S22) against its oracle
(oracle/pwa_oracle_rich.c, pinned in tests/test_oracle_rich.py), through the C ABI, at the north_star tolerances.

  * shared resonances, all constant-width: the FAST kernels (lanes sweep, split evaluation) with expansion / contraction;
  * mixed lineshape kinds (constant width, mass-dependent width, Flatte across the K K threshold): the general-lineshape
    kernel; every entry point; raw-sum additivity of two shards; bit-identical repeats;
  * the fit in the [waves | resonances] layout: box on the right entries, the oracle's verdict on the returned point.
"""
import numpy as np
import pytest
import torch

from helpers import rel_l2

pytestmark = pytest.mark.gpu
M_PI, M_K = 0.13957, 0.49368


@pytest.fixture(scope="module")
def env(oracle_mod):
    import paper_2403_09225_b200 as pwa
    from oracle import rich
    from paper_2403_09225_b200.build import build
    build()
    pwa.load()
    rich.build()
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    return pwa, rich


def _samples(oracle, seed, W, H, C, n_data, n_mc, weighted):
    rs = np.random.RandomState(seed)

    def sample(n, w):
        return oracle.Sample(rs.uniform(0.3, 3.0, size=(C, n)), rs.normal(size=(W, H, n, 2)),
                             rs.uniform(0.5, 1.5, size=n) if w else None)

    return sample(n_data, weighted), sample(n_mc, False)


def _theta(seed, W, L):
    rs = np.random.RandomState(seed)
    th = np.empty(2 * W + 2 * L)
    th[0:2 * W:2] = rs.uniform(0.5, 1.5, W)
    th[1:2 * W:2] = rs.uniform(-np.pi, np.pi, W)
    th[2 * W::2] = rs.uniform(1.1, 2.6, L)
    th[2 * W + 1::2] = rs.uniform(0.08, 0.4, L)
    return th


def _build(env, oracle, wave_res, ls_chan, kind, shape, H, C, n_data, n_mc, weighted, seed):
    pwa, rich = env
    W = len(wave_res)
    data, mc = _samples(oracle, seed, W, H, C, n_data, n_mc, weighted)
    rm = rich.RichModel(wave_res, ls_chan, kind, shape, data, mc)
    t = lambda a: None if a is None else torch.from_numpy(a)

    class Wl:
        res_chan = None
        data_mass, data_amp, data_weight = t(data.mass), t(data.amp), t(data.weight)
        mc_mass, mc_amp = t(mc.mass), t(mc.amp)

    gm = pwa.Model(Wl, rich={"wave_res": wave_res, "ls_chan": ls_chan, "ls_kind": kind, "ls_shape": shape})
    return rm, gm


def _shared_const(env, oracle):
    """24 waves on 9 constant-width resonances over 3 channels, 2 helicities (the config-3 kernel shape), weighted."""
    _, rich = env
    W, L = 24, 9
    wave_res = np.array([(3 * m + m // 5) % L for m in range(W)], dtype=np.int32)
    return _build(env, oracle, wave_res, np.arange(L, dtype=np.int32) % 3, np.zeros(L, dtype=np.int32),
                  np.zeros((L, rich.N_SP)), 2, 3, 3_001, 20_011, True, 71)


def _mixed(env, oracle):
    """11 waves on 5 resonances: 2 constant-width, 2 mass-dependent (L = 0 and L = 2, pi pi), 1 Flatte (pi pi / K K)."""
    _, rich = env
    wave_res = np.array([0, 1, 2, 3, 4, 0, 1, 2, 4, 1, 3], dtype=np.int32)
    kind = np.array([0, 1, 2, 0, 1], dtype=np.int32)
    shape = np.zeros((5, rich.N_SP))
    shape[1, :3] = (M_PI, M_PI, 2.0)
    shape[2, :5] = (M_PI, M_PI, M_K, M_K, 4.21)
    shape[4, :3] = (M_PI, M_PI, 0.0)
    return _build(env, oracle, wave_res, np.array([0, 1, 0, 1, 1], dtype=np.int32), kind, shape, 3, 2, 2_003, 12_007, True, 72)


@pytest.mark.parametrize("which", ["shared_const", "mixed"])
def test_every_entry_point_matches_the_rich_oracle(oracle_mod, env, which):
    pwa, rich = env
    rm, gm = (_shared_const if which == "shared_const" else _mixed)(env, oracle_mod)
    variant = pwa.pwa_kernel_variant(gm.h)
    assert variant.startswith("lanes") and variant.endswith("+shared") if which == "shared_const" else variant.startswith("rich")
    assert gm.P == rm.n_par == 2 * rm.n_wave + 2 * rm.n_ls
    for seed in (1, 2):
        th = _theta(seed, rm.n_wave, rm.n_ls)
        v = np.random.RandomState(10 + seed).normal(size=rm.n_par)
        f0, g0, h0 = rich.nll_grad_hvp(rm, th, v, "ld")
        f, g, hv = gm.nll_grad_hvp(th, v)
        assert abs(f - float(f0)) <= 1e-10 * max(1.0, abs(float(f0)))
        assert rel_l2(g, g0) < 1e-8 and rel_l2(hv, h0) < 1e-8
        assert pwa.pwa_status_flags(gm.h) == 0
        assert abs(gm.nll(th) - float(f0)) <= 1e-10 * max(1.0, abs(float(f0)))
        f1, g1 = gm.nll_grad(th)
        assert abs(f1 - float(f0)) <= 1e-10 * max(1.0, abs(float(f0))) and rel_l2(g1, g0) < 1e-8
        assert rel_l2(gm.hvp(th, v), h0) < 1e-8
        f2, g2 = gm.nll_grad_for_hvp(th)
        assert abs(f2 - float(f0)) <= 1e-10 * max(1.0, abs(float(f0))) and rel_l2(g2, g0) < 1e-8
        assert rel_l2(gm.hvp_cached(v), h0) < 1e-8
        f3, g3, hv3 = gm.nll_grad_hvp(th, v)
        assert f3 == f and g3.tobytes() == g.tobytes() and hv3.tobytes() == hv.tobytes()
    # batches and the Hessian go through single passes on such handles: still the same numbers
    thetas = np.stack([_theta(s, rm.n_wave, rm.n_ls) for s in (3, 4, 5)])
    got = gm.nll_batch(thetas)
    for k in range(3):
        f0 = float(rich.nll(rm, thetas[k], "ld"))
        assert abs(got[k] - f0) <= 1e-10 * max(1.0, abs(f0))
    gm.close()


def test_rich_raw_sums_are_additive_and_user_sized(oracle_mod, env):
    pwa, rich = env
    rm, gm = _mixed(env, oracle_mod)
    th, v = _theta(6, rm.n_wave, rm.n_ls), np.random.RandomState(3).normal(size=rm.n_par)
    raw = gm.raw_sums(th, v).cpu().numpy()
    P = rm.n_par
    assert raw.shape == (4 + 4 * P,) and pwa.pwa_raw_size(gm.h) == 4 + 4 * P
    sd, gd, hd = rich.raw_sums(rm, "data", th, v, "ld")
    sm, gG, hG = rich.raw_sums(rm, "mc", th, v, "ld")
    assert abs(raw[0] - float(sd[0])) <= 1e-10 * abs(float(sd[0])) and abs(raw[2] - float(sm[0])) <= 1e-10 * abs(float(sm[0]))
    assert raw[1] == pytest.approx(float(sd[1]), rel=1e-13) and raw[3] == rm.mc.n
    for k, ref in enumerate((gd, gG, hd, hG)):
        assert rel_l2(raw[4 + k * P: 4 + (k + 1) * P], ref) < 1e-8, k
    gm.close()


def test_fit_of_a_shared_resonance_model(oracle_mod, env):
    """Data drawn by accept-reject from the model itself; the fit starts at the generating parameters, converges,
    keeps M and Gamma (the LAST 2L entries in this layout) inside the S19 box, and the rich oracle confirms the point."""
    pwa, rich = env
    o = oracle_mod
    W, L, H = 6, 3, 2
    wave_res = np.array([0, 1, 2, 0, 1, 2], dtype=np.int32)
    rs = np.random.RandomState(5)
    th_true = _theta(8, W, L)
    n_mc, n_cand = 30_000, 120_000
    cand = o.Sample(rs.uniform(0.3, 3.0, size=(1, n_cand)), rs.normal(size=(W, H, n_cand, 2)), None)
    mc = o.Sample(rs.uniform(0.3, 3.0, size=(1, n_mc)), rs.normal(size=(W, H, n_mc, 2)), None)
    shape = np.zeros((L, rich.N_SP))
    gen = rich.RichModel(wave_res, np.zeros(L, dtype=np.int32), np.zeros(L, dtype=np.int32), shape, cand, mc)
    inten = rich.intensity(gen, "data", th_true, "d")
    keep = rs.uniform(size=n_cand) * inten.max() < inten
    data = o.Sample(cand.mass[:, keep], cand.amp[:, :, keep], None)
    assert data.n > 2_000
    rm = rich.RichModel(wave_res, np.zeros(L, dtype=np.int32), np.zeros(L, dtype=np.int32), shape, data, mc)
    t = torch.from_numpy

    class Wl:
        res_chan = None
        data_mass, data_amp, data_weight = t(data.mass), t(data.amp), None
        mc_mass, mc_amp = t(mc.mass), t(mc.amp)

    gm = pwa.Model(Wl, rich={"wave_res": wave_res, "ls_chan": np.zeros(L, dtype=np.int32)})
    th, res = gm.fit(th_true)
    assert res.status == 0 and res.stop_reason in (1, 2, 3), (res.status, res.stop_reason, res.grad_inf_norm)
    f0, g0, _ = rich.nll_grad_hvp(rm, th, None, "d", threads=o.max_threads())
    assert abs(float(f0) - res.nll) <= 1e-10 * max(1.0, abs(float(f0)))
    assert res.nll < float(rich.nll(rm, th_true, "d", threads=o.max_threads()))
    opts = pwa.pwa_fit_opts_default()
    M, G = th[2 * W::2], th[2 * W + 1::2]
    assert np.all(M >= opts.mass_min) and np.all(M <= opts.mass_max) and np.all(G >= opts.gamma_min) and np.all(G <= opts.gamma_max)
    g0 = np.asarray(g0, dtype=np.float64)
    free = np.ones(len(th), dtype=bool)
    free[2 * W::2] = ~(((M <= opts.mass_min) & (g0[2 * W::2] > 0)) | ((M >= opts.mass_max) & (g0[2 * W::2] < 0)))
    free[2 * W + 1::2] = ~(((G <= opts.gamma_min) & (g0[2 * W + 1::2] > 0)) | ((G >= opts.gamma_max) & (g0[2 * W + 1::2] < 0)))
    assert float(np.max(np.abs(g0[free]))) <= max(10 * res.grad_inf_norm, 1e-3)
    # a box that bites on a shared width: the bound sits on the resonance entry, not on a coupling
    o2 = pwa.pwa_fit_opts_default()
    o2.gamma_max = 0.8 * float(G.min())
    th2, res2 = gm.fit(th_true, o2)
    assert np.all(th2[2 * W + 1::2] <= o2.gamma_max) and res2.n_active >= 1 and res2.nll > res.nll
    assert np.any(th2[0:2 * W:2] > o2.gamma_max)   # couplings are not boxed
    gm.close()


def test_fit_runs_on_the_general_lineshape_kernel(oracle_mod, env):
    """A few Newton-CG iterations on the mixed-kind model (k_sweep_rich serves value, gradient and HVP of the driver):
    the NLL goes down, the reported value is the rich oracle's NLL at the returned point, the box holds."""
    pwa, rich = env
    rm, gm = _mixed(env, oracle_mod)
    th0 = _theta(11, rm.n_wave, rm.n_ls)
    o = pwa.pwa_fit_opts_default()
    o.max_outer = 6
    th, res = gm.fit(th0, o)
    f_start = float(rich.nll(rm, th0, "d", threads=oracle_mod.max_threads()))
    f_end = float(rich.nll(rm, th, "d", threads=oracle_mod.max_threads()))
    assert res.outer_iters == 6 and res.stop_reason == 4 and res.n_hvp >= 6
    assert res.nll < f_start and abs(res.nll - f_end) <= 1e-10 * max(1.0, abs(f_end))
    W = rm.n_wave
    assert np.all(th[2 * W::2] >= o.mass_min) and np.all(th[2 * W + 1::2] >= o.gamma_min)
    gm.close()


@pytest.mark.parametrize("which", ["shared_const", "mixed"])
def test_resonance_fractions_match_the_oracle(oracle_mod, env, which):
    """pwa_fit_fractions on a pwa_create_rich handle: one coherent fraction per RESONANCE (Table 1 of the paper lists
    one per resonance), every lineshape kind, against oracle/fractions.py::fit_fractions_rich."""
    from oracle.fractions import fit_fractions_rich
    pwa, rich = env
    rm, gm = (_shared_const if which == "shared_const" else _mixed)(env, oracle_mod)
    th = _theta(4, rm.n_wave, rm.n_ls)
    want = fit_fractions_rich(rm, th)
    got = gm.fit_fractions(th)
    assert got.shape == (rm.n_ls,)
    assert np.max(np.abs(got - want)) <= 1e-10 * np.max(np.abs(want))
    gm.close()
