"""Pins for the richer-model oracle (oracle/pwa_oracle_rich.c, oracle/rich.py; readings S21, S22).  CPU only.

R1  one wave per resonance, constant width: the rich oracle IS the base oracle (pwa_oracle.c, pinned by closed forms
    in test_oracle_pins.py) after the permutation between the two parameter layouts: NLL, gradient, HVP.
R2  Richardson central finite differences in 80-bit arithmetic: gradient from the NLL, HVP from the gradient, for every
    lineshape kind and with several waves sharing one resonance (the chain rule through shared M, Gamma).
R3  per-event equivalence: an event's intensity with a kind-1 / kind-2 resonance equals the BASE oracle's intensity of
    that event with a constant-width propagator at event-wise (M', Gamma'), where M'^2 - i M' Gamma' reproduces D; the
    break-up momenta and phase-space factors behind (M', Gamma') are computed HERE from the textbook two-body
    formulas (numpy, Kallen function), not by the oracle.  Covers Flatte below and above the second threshold.
R4  invariance under a global phase and a common rescaling; Hessian symmetry; H 1_phi = 0.
R5  waves of one resonance with identical projections add coherently: the NLL depends on Lambda_1 + Lambda_2 only.
R6  shared resonance = base model at the expanded parameter vector, gradient and HVP contracted (E^T g, E^T H E v):
    the identity the CUDA path uses to serve shared resonances.
"""
import numpy as np
import pytest

from helpers import rel_l2

LD = np.longdouble
M_PI, M_K = 0.13957, 0.49368


def _richardson(f, x, d, h):
    x = np.asarray(x, dtype=LD)
    d = np.asarray(d, dtype=LD)
    D1 = (f(x + h * d) - f(x - h * d)) / (2 * h)
    D2 = (f(x + 2 * h * d) - f(x - 2 * h * d)) / (4 * h)
    return (4 * D1 - D2) / 3


@pytest.fixture(scope="module")
def rich(oracle_mod):
    from oracle import rich as r
    r.build()
    return r


def _samples(oracle, seed, W, H, C, n_data, n_mc, weighted=True, lo=0.3, hi=3.0):
    rs = np.random.RandomState(seed)

    def sample(n, w):
        return oracle.Sample(rs.uniform(lo, hi, size=(C, n)), rs.normal(size=(W, H, n, 2)),
                             rs.uniform(0.5, 1.5, size=n) if w else None)

    return sample(n_data, weighted), sample(n_mc, False)


def _theta(seed, W, L):
    rs = np.random.RandomState(seed)
    th = np.empty(2 * W + 2 * L)
    th[0:2 * W:2] = rs.uniform(0.5, 1.5, W)
    th[1:2 * W:2] = rs.uniform(-np.pi, np.pi, W)
    th[2 * W::2] = rs.uniform(1.1, 2.6, L)       # above the K K threshold (kind 1 needs q(M) real)
    th[2 * W + 1::2] = rs.uniform(0.08, 0.4, L)
    return th


def _mixed_model(oracle, rich, seed=21, weighted=True):
    """5 waves on 3 resonances: resonance 0 (constant width) has 2 waves, resonance 1 (mass-dependent width, L = 2, pi pi)
    has 2 waves, resonance 2 (Flatte, pi pi / K K, g2/g1 = 4.21) has 1; two mass channels."""
    wave_res = [0, 1, 0, 2, 1]
    data, mc = _samples(oracle, seed, 5, 2, 2, 40, 160, weighted)
    shape = np.zeros((3, rich.N_SP))
    shape[1, :3] = (M_PI, M_PI, 2.0)
    shape[2, :5] = (M_PI, M_PI, M_K, M_K, 4.21)
    return rich.RichModel(wave_res, [0, 1, 1], [0, 1, 2], shape, data, mc)


# ----------------------------------------------------------------------------------------------- R1
def test_r1_one_wave_per_constant_width_resonance_is_the_base_model(oracle_mod, rich):
    o = oracle_mod
    W = 4
    data, mc = _samples(o, 3, W, 3, 2, 60, 200)
    res_chan = np.array([0, 1, 1, 0], dtype=np.int32)
    base = o.Model(res_chan, data, mc)
    rm = rich.RichModel(np.arange(W), res_chan, np.zeros(W), np.zeros((W, rich.N_SP)), data, mc)
    th_r = _theta(4, W, W)
    perm = np.empty(4 * W, dtype=int)          # base index 4r+k -> rich index
    for r in range(W):
        perm[4 * r:4 * r + 4] = (2 * r, 2 * r + 1, 2 * W + 2 * r, 2 * W + 2 * r + 1)
    v_r = np.random.RandomState(5).normal(size=4 * W)
    f0, g0, h0 = o.nll_grad_hvp(base, th_r[perm], v_r[perm], "ld")
    f1, g1, h1 = rich.nll_grad_hvp(rm, th_r, v_r, "ld")
    assert abs(float(f1 - f0)) <= 1e-15 * abs(float(f0))
    assert rel_l2(np.asarray(g1)[perm], g0) < 1e-15 and rel_l2(np.asarray(h1)[perm], h0) < 1e-15


# ----------------------------------------------------------------------------------------------- R2
@pytest.mark.parametrize("weighted", [False, True])
def test_r2_gradient_and_hvp_match_finite_differences(oracle_mod, rich, weighted):
    rm = _mixed_model(oracle_mod, rich, weighted=weighted)
    th = _theta(7, rm.n_wave, rm.n_ls).astype(LD)
    P = rm.n_par
    _, grad, _ = rich.nll_grad_hvp(rm, th, None, "ld")
    h = LD(1e-5)
    fd = np.array([_richardson(lambda x: rich.nll(rm, x, "ld"), th, np.eye(P, dtype=LD)[k], h) for k in range(P)], dtype=LD)
    assert rel_l2(grad, fd) < 1e-11
    assert float(np.max(np.abs(grad - fd))) < 1e-10 * float(np.max(np.abs(fd)))
    for seed in (1, 2):
        v = np.random.RandomState(seed).normal(size=P).astype(LD)
        _, _, hv = rich.nll_grad_hvp(rm, th, v, "ld")
        fdh = _richardson(lambda x: rich.nll_grad_hvp(rm, x, None, "ld")[1], th, v, h)
        assert rel_l2(hv, fdh) < 1e-11
    # every single Hessian column of the shared lineshape parameters (where the chain rule is not diagonal)
    for k in range(2 * rm.n_wave, P):
        e = np.eye(P, dtype=LD)[k]
        _, _, hv = rich.nll_grad_hvp(rm, th, e, "ld")
        fdh = _richardson(lambda x: rich.nll_grad_hvp(rm, x, None, "ld")[1], th, e, h)
        assert rel_l2(hv, fdh) < 1e-10, k


# ----------------------------------------------------------------------------------------------- R3
def _q2(s, m1, m2):
    """Kallen: q^2 = lambda(s, m1^2, m2^2) / (4 s)."""
    lam = s * s + m1 ** 4 + m2 ** 4 - 2 * s * m1 * m1 - 2 * s * m2 * m2 - 2 * m1 * m1 * m2 * m2
    return lam / (4 * s)


@pytest.mark.parametrize("kind", [1, 2])
def test_r3_event_wise_equivalence_with_a_constant_width_propagator(oracle_mod, rich, kind):
    o = oracle_mod
    data, mc = _samples(o, 31, 2, 2, 1, 1, 300, weighted=False, lo=0.3, hi=2.5)
    shape = np.zeros((2, rich.N_SP))
    if kind == 1:
        shape[1, :3] = (M_PI, M_K, 1.0)       # unequal daughters, P wave; threshold 0.633: cut the sample above it
        mc = o.Sample(np.maximum(mc.mass, 0.7), mc.amp, None)
    else:
        shape[1, :5] = (M_PI, M_PI, M_K, M_K, 4.21)
    rm = rich.RichModel([0, 1], [0, 0], [0, kind], shape, data, mc)
    th = np.array([1.1, 0.4, 0.8, -1.3, 1.9, 0.21, 1.02, 0.17])   # a0 phi0 a1 phi1 | M0 G0 | M1 G1
    got = rich.intensity(rm, "mc", th, "ld")
    m = mc.mass[0]
    M1, G1 = th[6], th[7]
    assert np.any(m < 2 * M_K) and np.any(m > 2 * M_K)            # both sides of the K K threshold
    if kind == 1:
        qm, q0 = np.sqrt(_q2(m * m, M_PI, M_K)), np.sqrt(_q2(M1 * M1, M_PI, M_K))
        D = M1 * M1 - m * m - 1j * M1 * (G1 * (qm / q0) ** 3 * M1 / m)
    else:
        rho1 = 2 * np.sqrt(_q2(m * m, M_PI, M_PI).astype(complex)) / m
        rho2 = 2 * np.sqrt(_q2(m * m, M_K, M_K).astype(complex)) / m     # principal root: +i|.| below threshold
        D = M1 * M1 - m * m - 1j * G1 * (rho1 + 4.21 * rho2)
    # constant-width propagator with the same denominator at THIS event: M'^2 = Re D + m^2, M' Gamma' = -Im D
    Mp = np.sqrt(D.real + m * m)
    Gp = -D.imag / Mp
    base_th = np.array([th[0], th[1], th[4], th[5], th[2], th[3], 0.0, 0.0])
    for j in range(mc.n):
        one = o.Sample(mc.mass[:, j:j + 1], mc.amp[:, :, j:j + 1], None)
        bm = o.Model(np.array([0, 0], dtype=np.int32), one, one)
        base_th[6], base_th[7] = Mp[j], Gp[j]
        want = o.intensity(bm, "mc", base_th, prec="ld")[0]
        assert abs(got[j] - want) <= 1e-12 * abs(want), (j, m[j], got[j], want)


# ----------------------------------------------------------------------------------------------- R4
def test_r4_gauge_invariances_and_hessian_symmetry(oracle_mod, rich):
    rm = _mixed_model(oracle_mod, rich)
    W, P = rm.n_wave, rm.n_par
    th = _theta(9, W, rm.n_ls).astype(LD)
    f0, g, _ = rich.nll_grad_hvp(rm, th, None, "ld")
    t2 = th.copy(); t2[0:2 * W:2] *= LD(1.7); t2[1:2 * W:2] += LD(0.9)
    assert abs(float(rich.nll(rm, t2, "ld") - f0)) <= 1e-14 * abs(float(f0))
    assert abs(float(np.sum(th[0:2 * W:2] * g[0:2 * W:2]))) <= 1e-13 * float(np.max(np.abs(g)))
    assert abs(float(np.sum(g[1:2 * W:2]))) <= 1e-13 * float(np.max(np.abs(g)))
    ones_phi = np.zeros(P, dtype=LD); ones_phi[1:2 * W:2] = 1
    _, _, h1 = rich.nll_grad_hvp(rm, th, ones_phi, "ld")
    rs = np.random.RandomState(2)
    v1, v2 = rs.normal(size=P).astype(LD), rs.normal(size=P).astype(LD)
    _, _, hv1 = rich.nll_grad_hvp(rm, th, v1, "ld")
    _, _, hv2 = rich.nll_grad_hvp(rm, th, v2, "ld")
    assert float(np.max(np.abs(h1))) <= 1e-12 * float(np.max(np.abs(hv1)))
    assert abs(float(v2 @ hv1 - v1 @ hv2)) <= 1e-13 * abs(float(v2 @ hv1))


# ----------------------------------------------------------------------------------------------- R5
def test_r5_identical_waves_of_one_resonance_add_coherently(oracle_mod, rich):
    o = oracle_mod
    data, mc = _samples(o, 41, 3, 2, 1, 30, 90)
    for s in (data, mc):
        s.amp[1] = s.amp[0]                                        # waves 0 and 1: same projections, same resonance
    shape = np.zeros((2, rich.N_SP)); shape[0, :3] = (M_PI, M_PI, 1.0)
    rm = rich.RichModel([0, 0, 1], [0, 0], [1, 0], shape, data, mc)
    th = _theta(3, 3, 2)
    c = th[0] * np.exp(1j * th[1]) + th[2] * np.exp(1j * th[3])
    merged = th.copy()
    merged[0], merged[1] = abs(c), np.angle(c)
    merged[2] = 0.0
    assert abs(float(rich.nll(rm, th, "ld") - rich.nll(rm, merged, "ld"))) <= 1e-13 * abs(float(rich.nll(rm, th, "ld")))


# ----------------------------------------------------------------------------------------------- R6
def test_r6_shared_resonance_is_the_base_model_expanded_and_contracted(oracle_mod, rich):
    o = oracle_mod
    W, L = 5, 2
    wave_res = np.array([0, 1, 1, 0, 1])
    res_chan = np.array([1, 0], dtype=np.int32)
    data, mc = _samples(o, 51, W, 2, 2, 50, 170)
    rm = rich.RichModel(wave_res, res_chan, np.zeros(L), np.zeros((L, rich.N_SP)), data, mc)
    base = o.Model(res_chan[wave_res], data, mc)
    th, v = _theta(6, W, L), np.random.RandomState(8).normal(size=2 * W + 2 * L)
    E = np.zeros((4 * W, 2 * W + 2 * L))                        # base (expanded) parameters = E theta
    for m in range(W):
        E[4 * m, 2 * m] = E[4 * m + 1, 2 * m + 1] = 1
        E[4 * m + 2, 2 * W + 2 * wave_res[m]] = E[4 * m + 3, 2 * W + 2 * wave_res[m] + 1] = 1
    f0, g0, h0 = o.nll_grad_hvp(base, E @ th, E @ v, "ld")
    f1, g1, h1 = rich.nll_grad_hvp(rm, th, v, "ld")
    assert abs(float(f1 - f0)) <= 1e-15 * abs(float(f0))
    assert rel_l2(g1, E.T @ np.asarray(g0, dtype=LD)) < 1e-14
    assert rel_l2(h1, E.T @ np.asarray(h0, dtype=LD)) < 1e-14


# ----------------------------------------------------------------------------------------------- fractions
def test_resonance_fractions_reduce_to_the_known_cases(oracle_mod, rich):
    """fit_fractions_rich (one coherent fraction per resonance): one wave per constant-width resonance gives the base
    per-resonance fractions (oracle/fractions.py, pinned by closed forms in test_oracle_fractions.py); two waves of ONE
    resonance with identical projections give |c_1 + c_2|^2 B-weighted, i.e. the fraction of the merged wave; a model
    with a single resonance has fraction 1 whatever its waves; global phase and common scale drop out."""
    from oracle.fractions import fit_fractions, fit_fractions_rich
    o = oracle_mod
    W = 4
    data, mc = _samples(o, 61, W, 2, 2, 10, 400)
    res_chan = np.array([0, 1, 1, 0], dtype=np.int32)
    rm = rich.RichModel(np.arange(W), res_chan, np.zeros(W), np.zeros((W, rich.N_SP)), data, mc)
    th = _theta(5, W, W)
    base_th = np.empty(4 * W)
    base_th[0::4], base_th[1::4], base_th[2::4], base_th[3::4] = th[0:2 * W:2], th[1:2 * W:2], th[2 * W::2], th[2 * W + 1::2]
    want = fit_fractions(o.Model(res_chan, data, mc), base_th)
    assert np.max(np.abs(fit_fractions_rich(rm, th) - want)) <= 1e-14
    # waves 0 and 1 identical, both in resonance 0 (Flatte), wave 2 in resonance 1
    data, mc = _samples(o, 62, 3, 2, 1, 10, 300)
    mc.amp[1] = mc.amp[0]
    shape = np.zeros((2, rich.N_SP)); shape[0, :5] = (M_PI, M_PI, M_K, M_K, 4.21)
    rm2 = rich.RichModel([0, 0, 1], [0, 0], [2, 0], shape, data, mc)
    th2 = _theta(6, 3, 2)
    c = th2[0] * np.exp(1j * th2[1]) + th2[2] * np.exp(1j * th2[3])
    merged = th2.copy(); merged[0], merged[1], merged[2] = abs(c), np.angle(c), 0.0
    f2, fm = fit_fractions_rich(rm2, th2), fit_fractions_rich(rm2, merged)
    assert np.max(np.abs(f2 - fm)) <= 1e-13
    gauge = th2.copy(); gauge[0:6:2] *= 2.5; gauge[1:6:2] -= 0.7
    assert np.max(np.abs(fit_fractions_rich(rm2, gauge) - f2)) <= 1e-13
    one = rich.RichModel([0, 0, 0], [0], [1], np.array([[M_PI, M_PI, 1.0, 0, 0, 0]]), data, mc)
    assert abs(fit_fractions_rich(one, _theta(7, 3, 1))[0] - 1.0) <= 1e-14
