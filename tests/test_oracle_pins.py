"""Pins for the CPU oracle: things the paper and the mathematics fix, none of which call the oracle's
own formulas a second time (SURVEY.md §8(c) "What pins the oracle").  CPU only.

P1  Richardson central finite differences in 80-bit arithmetic (gradient from the NLL, HVP from the gradient)
P2  invariance of the NLL under a global phase and a common rescaling of all couplings, and what these
    imply for the gradient and the HVP; symmetry of the Hessian
P3  closed forms of the |BW|^2 and BW_1 conj(BW_2) integrals (constant F) for the MC normalisation
P4  the MC term as a Hermitian form c^H Q c through a library matmul
P5  special cases (one resonance; two identical resonances)
P6  weight linearity, permutation of events, shard additivity (Eqs. 4-7)
P7  sign / statistics: data drawn from the model prefer theta_true to random parameter sets
"""
import numpy as np
import pytest

from helpers import random_model, random_theta, rel_l2

LD = np.longdouble


# ----------------------------------------------------------------------------------------------- P1
def _richardson(f, x, d, h):
    """4th-order central difference of f along d: (4 D_h - D_2h)/3, all in long double."""
    x = np.asarray(x, dtype=LD)
    d = np.asarray(d, dtype=LD)
    D1 = (f(x + h * d) - f(x - h * d)) / (2 * h)
    D2 = (f(x + 2 * h * d) - f(x - 2 * h * d)) / (4 * h)
    return (4 * D1 - D2) / 3


@pytest.mark.parametrize("weighted", [False, True])
def test_p1_gradient_matches_finite_differences_of_nll(oracle_mod, weighted):
    o = oracle_mod
    R = 3
    m = random_model(o, 11, R, H=2, C=2, n_data=40, n_mc=150, weighted=weighted)
    th = random_theta(5, R).astype(LD)
    _, grad, _ = o.nll_grad_hvp(m, th, None, "ld")
    h = LD(1e-5)
    fd = np.array([_richardson(lambda x: o.nll(m, x, "ld"), th, np.eye(4 * R, dtype=LD)[k], h)
                   for k in range(4 * R)], dtype=LD)
    assert rel_l2(grad, fd) < 1e-12
    assert float(np.max(np.abs(grad - fd))) < 1e-11 * float(np.max(np.abs(fd)))


@pytest.mark.parametrize("weighted", [False, True])
def test_p1_hvp_matches_finite_differences_of_gradient(oracle_mod, weighted):
    o = oracle_mod
    R = 3
    m = random_model(o, 12, R, H=3, C=2, n_data=30, n_mc=120, weighted=weighted)
    th = random_theta(6, R).astype(LD)
    v = np.random.RandomState(3).normal(size=4 * R).astype(LD)
    _, _, hv = o.nll_grad_hvp(m, th, v, "ld")
    fd = _richardson(lambda x: o.nll_grad_hvp(m, x, None, "ld")[1], th, v, LD(1e-5))
    assert rel_l2(hv, fd) < 1e-12
    # per-sample pieces too (data and MC raw sums are differentiated separately)
    for which in ("data", "mc"):
        _, _, hs = o.raw_sums(m, which, th, v, "ld")
        sign = -1 if which == "data" else 1   # data raw sums carry d^2(-ln I), i.e. minus the sum of ln I
        if which == "mc":
            fd_s = _richardson(lambda x: o.raw_sums(m, which, x, None, "ld")[1], th, v, LD(1e-5))
        else:
            fd_s = -_richardson(lambda x: o.raw_sums(m, which, x, None, "ld")[1], th, v, LD(1e-5))
        assert rel_l2(hs, fd_s) < 1e-12, (which, sign)


def test_p1_data_gradient_sum_is_derivative_of_log_sum(oracle_mod):
    o = oracle_mod
    R = 2
    m = random_model(o, 13, R, H=2, C=1, n_data=25, n_mc=10, weighted=True)
    th = random_theta(7, R).astype(LD)
    _, gd, _ = o.raw_sums(m, "data", th, None, "ld")
    fd = np.array([_richardson(lambda x: o.raw_sums(m, "data", x, None, "ld")[0][0], th,
                               np.eye(4 * R, dtype=LD)[k], LD(1e-5)) for k in range(4 * R)], dtype=LD)
    assert rel_l2(gd, fd) < 1e-12


# ----------------------------------------------------------------------------------------------- P2
def test_p2_global_phase_and_scale_invariance(oracle_mod):
    o = oracle_mod
    R = 4
    m = random_model(o, 21, R, H=2, C=2, n_data=200, n_mc=700, weighted=True)
    th = random_theta(8, R)
    v = np.random.RandomState(4).normal(size=4 * R)
    nll0, g, hv = o.nll_grad_hvp(m, th, v, "ld")
    t2 = th.reshape(R, 4).copy()
    t2[:, 0] *= 1.7
    t2[:, 1] += 0.9
    nll1 = o.nll(m, t2.reshape(-1), "ld")
    assert abs(float(nll1 - nll0)) < 1e-13 * abs(float(nll0))

    g = np.asarray(g, dtype=np.float64).reshape(R, 4)
    a = th.reshape(R, 4)[:, 0]
    gscale = float(np.abs(g).max())
    assert abs(float((a * g[:, 0]).sum())) < 1e-12 * gscale       # grad . c = 0  (north_star)
    assert abs(float(g[:, 1].sum())) < 1e-12 * gscale             # grad . 1_phi = 0

    one_phi = np.zeros((R, 4)); one_phi[:, 1] = 1.0
    u = np.zeros((R, 4)); u[:, 0] = a
    _, _, h_phi = o.nll_grad_hvp(m, th, one_phi.reshape(-1), "ld")
    _, _, h_u = o.nll_grad_hvp(m, th, u.reshape(-1), "ld")
    hscale = float(np.abs(np.asarray(hv, dtype=np.float64)).max())
    assert float(np.abs(np.asarray(h_phi, dtype=np.float64)).max()) < 1e-12 * hscale   # H 1_phi = 0
    # differentiate grad . u = 0: H u = -g on the a-entries, 0 elsewhere
    expect = np.zeros((R, 4)); expect[:, 0] = -g[:, 0]
    assert float(np.abs(np.asarray(h_u, dtype=np.float64) - expect.reshape(-1)).max()) < 1e-12 * hscale


def test_p2_hessian_is_symmetric(oracle_mod):
    o = oracle_mod
    R = 3
    m = random_model(o, 22, R, H=2, C=3, n_data=80, n_mc=300, weighted=False)
    th = random_theta(9, R)
    rs = np.random.RandomState(5)
    v1, v2 = rs.normal(size=4 * R), rs.normal(size=4 * R)
    _, _, h1 = o.nll_grad_hvp(m, th, v1, "ld")
    _, _, h2 = o.nll_grad_hvp(m, th, v2, "ld")
    a, b = float((v2 * h1).sum()), float((v1 * h2).sum())
    assert abs(a - b) < 1e-12 * max(abs(a), abs(b))


# ----------------------------------------------------------------------------------------------- P3
def _prim_inv(q, m):
    """Primitive of 1/(q^2 - m^2) in m for complex q off the real axis (principal log is continuous)."""
    return np.log((q + m) / (q - m)) / (2 * q)


def test_p3_closed_form_bw_integrals_uniform_in_m(oracle_mod):
    """MC term for constant F on a midpoint grid in m:  G (hi-lo)/N = sum_h int |sum_r c_r f_rh BW_r|^2 dm.
    int BW_1 conj(BW_2) dm by partial fractions of 1/((q1^2-m^2)(conj(q2)^2-m^2)), q_r^2 = M_r^2 - i M_r Gamma_r."""
    o = oracle_mod
    lo, hi, N = 0.3, 3.0, 200_000
    grid = lo + (np.arange(N) + 0.5) * (hi - lo) / N
    R, H = 2, 2
    th = np.array([0.8, 0.6, 1.3, 0.07, 1.4, -2.1, 1.9, 0.25])
    f = np.array([[1.0 + 0.0j, 0.3 - 0.5j], [1.3 * np.exp(0.7j), -0.4 + 0.9j]])      # f[r][h]
    amp = np.empty((R, H, N, 2))
    amp[..., 0] = f.real[:, :, None]
    amp[..., 1] = f.imag[:, :, None]
    mc = o.Sample(grid.reshape(1, N), amp, None)
    m = o.Model(np.zeros(R, np.int32), o.Sample(grid[:3].reshape(1, 3), amp[:, :, :3], None), mc)
    scal, _, _ = o.raw_sums(m, "mc", th, None, "ld")
    got = float(scal[0]) * (hi - lo) / N

    a, phi, M, G = th.reshape(R, 4).T
    c = a * np.exp(1j * phi)
    q2 = M * M - 1j * M * G                           # D_r = q_r^2 - m^2
    q = np.sqrt(q2)
    X = np.empty((R, R), complex)                     # X[r][s] = int BW_r conj(BW_s) dm
    for r in range(R):
        for s in range(R):
            p2 = np.conj(q2[s]); p = np.sqrt(p2)
            X[r, s] = ((_prim_inv(q[r], hi) - _prim_inv(q[r], lo)) - (_prim_inv(p, hi) - _prim_inv(p, lo))) / (p2 - q2[r])
    want = 0.0
    for h in range(H):
        ce = c * f[:, h]
        want += np.real(np.einsum("r,rs,s->", ce, X, np.conj(ce)))
    assert abs(got - want) < 2e-12 * abs(want)
    # and the single-resonance special case quoted in north_star: int |BW|^2 dm = Im(int BW dm)/(M Gamma)
    J = np.imag(_prim_inv(q[0], hi) - _prim_inv(q[0], lo)) / (M[0] * G[0])
    assert abs(np.real(X[0, 0]) - J) < 1e-13 * J


def test_p3_closed_form_bw_integral_uniform_in_s(oracle_mod):
    """Grid uniform in s = m^2: int ds / ((M^2-s)^2 + M^2 Gamma^2) = [atan((s-M^2)/(M Gamma))]/(M Gamma)."""
    o = oracle_mod
    lo, hi, N = 0.3, 3.0, 200_000
    s = lo * lo + (np.arange(N) + 0.5) * (hi * hi - lo * lo) / N
    amp = np.zeros((1, 1, N, 2)); amp[..., 0] = 1.0
    mc = o.Sample(np.sqrt(s).reshape(1, N), amp, None)
    m = o.Model(np.zeros(1, np.int32), o.Sample(mc.mass[:, :2], amp[:, :, :2], None), mc)
    a, M, G = 1.7, 1.3, 0.07
    scal, _, _ = o.raw_sums(m, "mc", np.array([a, 0.4, M, G]), None, "ld")
    got = float(scal[0]) * (hi * hi - lo * lo) / N
    want = a * a * (np.arctan((hi * hi - M * M) / (M * G)) - np.arctan((lo * lo - M * M) / (M * G))) / (M * G)
    assert abs(got - want) < 2e-12 * want


def test_p3_full_nll_closed_form_pins_the_additive_constant(oracle_mod):
    """The WHOLE NLL of Eq. 3 (readings S2, S3) in closed form, additive constant included:
    R = 1, H = 1, F = 1, MC masses on a midpoint grid uniform in s = m^2 over [lo^2, hi^2], five weighted data events
    at chosen masses:
        NLL = - sum_i w_i ln( a^2 / ((M^2 - m_i^2)^2 + M^2 Gamma^2) ) + W ln( a^2 J / (hi^2 - lo^2) ),
        J = [atan((s - M^2)/(M Gamma))] over [lo^2, hi^2] / (M Gamma),    W = sum_i w_i,
    evaluated here with numpy only.  Every other pin is blind to a theta-independent shift of the NLL (they differentiate
    it or compare two NLLs that share W and N_mc); a dropped 1/N_mc inside the logarithm, or a logarithm of another
    base, changes this value by W ln N_mc (= 65) or by a factor ln 10 and fails here."""
    o = oracle_mod
    lo, hi, N = 0.3, 3.0, 400_000
    s = lo * lo + (np.arange(N) + 0.5) * (hi * hi - lo * lo) / N
    amp = np.zeros((1, 1, N, 2)); amp[..., 0] = 1.0
    mc = o.Sample(np.sqrt(s).reshape(1, N), amp, None)
    md = np.array([0.45, 1.1, 1.31, 1.9, 2.7])
    w = np.array([0.5, 1.5, 1.0, 0.75, 1.25])
    ad = np.zeros((1, 1, md.size, 2)); ad[..., 0] = 1.0
    m = o.Model(np.zeros(1, np.int32), o.Sample(md.reshape(1, -1), ad, w), mc)
    a, phi, M, G = 1.7, 0.4, 1.3, 0.07
    J = (np.arctan((hi * hi - M * M) / (M * G)) - np.arctan((lo * lo - M * M) / (M * G))) / (M * G)
    want = -np.sum(w * np.log(a * a / ((M * M - md * md) ** 2 + (M * G) ** 2))) + w.sum() * np.log(a * a * J / (hi * hi - lo * lo))
    for prec in ("ld", "d"):
        got = float(o.nll(m, np.array([a, phi, M, G]), prec))
        assert abs(got - want) < 1e-11 * abs(want), (prec, got, want)
    # the constant really is visible to this test: the two plausible mistakes named above move the value far outside
    assert abs(w.sum() * np.log(N)) > 1e3 * 1e-11 * abs(want) and abs(want) * (1 - 1 / np.log(10)) > 1.0


# ----------------------------------------------------------------------------------------------- P4
def test_p4_mc_term_is_a_hermitian_form_in_the_couplings(oracle_mod):
    o = oracle_mod
    R, H, C, N = 5, 3, 2, 400
    m = random_model(o, 41, R, H, C, n_data=5, n_mc=N, weighted=False)
    th = random_theta(10, R)
    a, phi, M, G = th.reshape(R, 4).T
    c = a * np.exp(1j * phi)
    mass = m.mc.mass[m.res_chan]                                        # [R][N]
    B = 1.0 / ((M * M)[:, None] - mass ** 2 - 1j * (M * G)[:, None])    # definition of BW (configs[0])
    Fc = m.mc.amp[..., 0] + 1j * m.mc.amp[..., 1]                       # [R][H][N]
    Y = (B[:, None, :] * Fc).reshape(R, H * N)
    Q = Y.conj() @ Y.T                                                  # library matmul: Q[r][s] = sum conj(Y_r) Y_s
    Qc = Q @ c
    scal, gG, _ = o.raw_sums(m, "mc", th, None, "ld")
    Gval = np.real(np.conj(c) @ Qc)
    assert abs(float(scal[0]) - Gval) < 1e-13 * Gval
    gG = np.asarray(gG, dtype=np.float64).reshape(R, 4)
    dG_da = 2 * np.real(np.exp(-1j * phi) * Qc)
    dG_dphi = 2 * np.imag(np.conj(c) * Qc)
    assert np.abs(gG[:, 0] - dG_da).max() < 1e-12 * np.abs(dG_da).max()
    assert np.abs(gG[:, 1] - dG_dphi).max() < 1e-12 * np.abs(dG_dphi).max()
    # the (a, phi) block of the MC Hessian-vector product also follows from Q (G is quadratic in c)
    rs = np.random.RandomState(6)
    v = np.zeros((R, 4)); v[:, 0] = rs.normal(size=R); v[:, 1] = rs.normal(size=R)
    _, _, hG = o.raw_sums(m, "mc", th, v.reshape(-1), "ld")
    hG = np.asarray(hG, dtype=np.float64).reshape(R, 4)
    e = np.exp(1j * phi)
    cdot = e * v[:, 0] + 1j * c * v[:, 1]
    Qcd = Q @ cdot
    h_a = 2 * np.real(np.conj(e) * Qcd) + 2 * np.real(np.conj(1j * e * v[:, 1]) * Qc)
    h_phi = 2 * np.real(np.conj(1j * c) * Qcd) + 2 * np.real(np.conj(1j * cdot) * Qc)
    assert np.abs(hG[:, 0] - h_a).max() < 1e-12 * np.abs(h_a).max()
    assert np.abs(hG[:, 1] - h_phi).max() < 1e-12 * np.abs(h_phi).max()


# ----------------------------------------------------------------------------------------------- P5
def test_p5_single_resonance_has_no_coupling_gradient(oracle_mod):
    o = oracle_mod
    m = random_model(o, 51, 1, H=2, C=1, n_data=60, n_mc=200, weighted=True)
    th = np.array([1.3, 0.4, 1.5, 0.2])
    _, g, _ = o.nll_grad_hvp(m, th, None, "ld")
    g = np.asarray(g, dtype=np.float64)
    assert abs(g[0]) < 1e-12 * np.abs(g[2:]).max() and abs(g[1]) < 1e-12 * np.abs(g[2:]).max()
    assert np.abs(g[2:]).max() > 1e-3


def test_p5_identical_resonances_add_coherently(oracle_mod):
    o = oracle_mod
    base = random_model(o, 52, 2, H=2, C=1, n_data=50, n_mc=150, weighted=False)
    for s in (base.data, base.mc):
        s.amp[1] = s.amp[0]
    M, G = 1.4, 0.15
    c1, c2 = 0.7 * np.exp(0.3j), 1.1 * np.exp(-1.9j)
    d1, d2 = 0.2 * np.exp(2.5j), c1 + c2 - 0.2 * np.exp(2.5j)
    th1 = np.array([abs(c1), np.angle(c1), M, G, abs(c2), np.angle(c2), M, G])
    th2 = np.array([abs(d1), np.angle(d1), M, G, abs(d2), np.angle(d2), M, G])
    n1, n2 = float(o.nll(base, th1, "ld")), float(o.nll(base, th2, "ld"))
    assert abs(n1 - n2) < 1e-12 * abs(n1)


# ----------------------------------------------------------------------------------------------- P6
def test_p6_weight_two_equals_two_copies(oracle_mod):
    o = oracle_mod
    R = 3
    m = random_model(o, 61, R, H=2, C=2, n_data=30, n_mc=100, weighted=True)
    w = m.data.weight.copy(); w[4] = 2.0
    a = o.Model(m.res_chan, o.Sample(m.data.mass, m.data.amp, w), m.mc)
    idx = list(range(30)) + [4]
    w1 = w[idx].copy(); w1[4] = 1.0; w1[-1] = 1.0
    b = o.Model(m.res_chan, o.Sample(m.data.mass[:, idx], m.data.amp[:, :, idx], w1), m.mc)
    th = random_theta(11, R)
    v = np.random.RandomState(7).normal(size=4 * R)
    ra, rb = o.nll_grad_hvp(a, th, v, "ld"), o.nll_grad_hvp(b, th, v, "ld")
    assert abs(float(ra[0] - rb[0])) < 1e-15 * abs(float(ra[0])) + 1e-15
    assert rel_l2(ra[1], rb[1]) < 1e-15 and rel_l2(ra[2], rb[2]) < 1e-15


def test_p6_permutation_and_unit_weights(oracle_mod):
    o = oracle_mod
    R = 3
    m = random_model(o, 62, R, H=2, C=2, n_data=40, n_mc=90, weighted=False)
    perm = np.random.RandomState(8).permutation(90)
    b = o.Model(m.res_chan, o.Sample(m.data.mass, m.data.amp, np.ones(40)),
                o.Sample(m.mc.mass[:, perm], m.mc.amp[:, :, perm], None))
    th = random_theta(12, R)
    v = np.random.RandomState(9).normal(size=4 * R)
    ra, rb = o.nll_grad_hvp(m, th, v, "ld"), o.nll_grad_hvp(b, th, v, "ld")
    assert abs(float(ra[0] - rb[0])) < 1e-16 * abs(float(ra[0])) * 90
    assert rel_l2(ra[1], rb[1]) < 1e-15 and rel_l2(ra[2], rb[2]) < 1e-15


@pytest.mark.parametrize("prec", ["ld", "d"])
def test_p6_shard_additivity(oracle_mod, prec):
    """Eqs. 4-7: raw sums of the shards, added, then combined, equal the whole."""
    o = oracle_mod
    R = 3
    m = random_model(o, 63, R, H=2, C=2, n_data=101, n_mc=333, weighted=True)
    th = random_theta(13, R)
    v = np.random.RandomState(10).normal(size=4 * R)
    whole = o.nll_grad_hvp(m, th, v, prec)
    parts = {"data": [(0, 37), (37, 64)], "mc": [(0, 100), (100, 200), (300, 33)]}
    tot = {}
    for which, shards in parts.items():
        acc = None
        for first, count in shards:
            r = o.raw_sums(m, which, th, v, prec, first=first, count=count)
            acc = r if acc is None else tuple(x + y for x, y in zip(acc, r))
        tot[which] = acc
    got = o.combine(tot["data"][0], tot["mc"][0], tot["data"][1], tot["mc"][1], tot["data"][2], tot["mc"][2], v, prec)
    tol = 1e-15 if prec == "ld" else 1e-13
    assert abs(float(got[0] - whole[0])) < tol * abs(float(whole[0]))
    assert rel_l2(got[1], whole[1]) < tol and rel_l2(got[2], whole[2]) < tol


def test_double_build_and_threads_agree_with_long_double(oracle_mod):
    o = oracle_mod
    R = 4
    m = random_model(o, 64, R, H=3, C=2, n_data=500, n_mc=2000, weighted=True)
    th = random_theta(14, R)
    v = np.random.RandomState(11).normal(size=4 * R)
    ref = o.nll_grad_hvp(m, th, v, "ld")
    for threads in (1, 3):
        got = o.nll_grad_hvp(m, th, v, "d", threads=threads)
        assert abs(float(got[0]) - float(ref[0])) < 1e-13 * abs(float(ref[0]))
        assert rel_l2(got[1], ref[1]) < 1e-13 and rel_l2(got[2], ref[2]) < 1e-13
    # per-event entry points are consistent with the sums
    I = o.intensity(m, "mc", th)
    assert abs(I.sum() - float(o.raw_sums(m, "mc", th, None, "ld")[0][0])) < 1e-12 * I.sum()
    Ii, Idot, g, hv = o.event(m, "mc", 7, th, v)
    assert abs(float(Ii) - I[7]) < 1e-15 * I[7]
    assert abs(float(Idot) - float((np.asarray(g, dtype=np.float64) * v).sum())) < 1e-12 * abs(float(Idot))


# ----------------------------------------------------------------------------------------------- P7
def test_p7_data_from_the_model_prefer_theta_true():
    import oracle as o
    import workloads as wl
    cfg = wl.CONFIGS[1].scaled(20_000, 2_000)
    w = wl.make_workload(cfg)
    m = o.model_from_workload(w)
    n_true = float(o.nll(m, w.theta_true.numpy(), "d", threads=4))
    others = [float(o.nll(m, wl.random_start(cfg, k).numpy(), "d", threads=4)) for k in range(6)]
    assert all(n_true < x - 10.0 for x in others), (n_true, others)
