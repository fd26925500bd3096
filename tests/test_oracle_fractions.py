"""Pins for oracle/fractions.py (the fit fractions of Table 1's kind, S20): closed forms and invariances
chosen so that a wrong denominator, a missing helicity sum, a dropped propagator or a coherent/incoherent mix-up fails."""
import numpy as np
import pytest

from helpers import random_model, random_theta


def test_single_resonance_has_fraction_one(oracle_mod):
    from oracle.fractions import fit_fractions
    om = random_model(oracle_mod, 21, R=1, H=3, C=1, n_data=10, n_mc=500, weighted=False)
    f = fit_fractions(om, random_theta(22, 1))
    assert f.shape == (1,) and abs(f[0] - 1.0) < 1e-15


def test_identical_lineshapes_and_amplitudes_give_the_coupling_ratio(oracle_mod):
    """Two resonances with the same (M, Gamma), the same channel and F_1h = F_2h: A = (c_1 + c_2) B F, so
    F_r = |c_r|^2 / |c_1 + c_2|^2 exactly, whatever the events are (closed form with full interference)."""
    from oracle.fractions import fit_fractions
    rs = np.random.RandomState(23)
    n = 400
    mass = rs.uniform(0.3, 3.0, size=(1, n))
    one = rs.normal(size=(1, 2, n, 2))
    amp = np.concatenate([one, one], axis=0)
    om = oracle_mod.Model(np.zeros(2, np.int32), oracle_mod.Sample(mass[:, :5], amp[:, :, :5], None),
                          oracle_mod.Sample(mass, amp, None))
    th = np.array([0.7, 0.4, 1.3, 0.2, 1.9, -2.1, 1.3, 0.2])
    c = th[0::4] * np.exp(1j * th[1::4])
    f = fit_fractions(om, th)
    assert np.allclose(f, np.abs(c) ** 2 / abs(c.sum()) ** 2, rtol=1e-14, atol=0)
    # destructive interference: the fractions add up to more than one here
    assert f.sum() > 1.0


def test_non_interfering_resonances_add_up_to_one(oracle_mod):
    """Resonance r couples to helicity component h = r only: no interference term survives, sum_r F_r = 1, and
    F_r is the ratio of the incoherent pieces computed by hand."""
    from oracle.fractions import fit_fractions
    rs = np.random.RandomState(24)
    R = H = 3
    n = 600
    mass = rs.uniform(0.3, 3.0, size=(2, n))
    amp = np.zeros((R, H, n, 2))
    for r in range(R):
        amp[r, r] = rs.normal(size=(n, 2))
    res_chan = np.array([0, 1, 0], np.int32)
    om = oracle_mod.Model(res_chan, oracle_mod.Sample(mass[:, :5], amp[:, :, :5], None), oracle_mod.Sample(mass, amp, None))
    th = random_theta(25, R)
    f = fit_fractions(om, th)
    assert abs(f.sum() - 1.0) < 1e-14
    own = np.empty(R)
    for r in range(R):
        a, phi, M, G = th[4 * r: 4 * r + 4]
        m = mass[res_chan[r]]
        bw2 = 1.0 / ((M * M - m * m) ** 2 + (M * G) ** 2)          # |B|^2, textbook Breit-Wigner
        own[r] = a * a * np.sum(bw2 * (amp[r, r, :, 0] ** 2 + amp[r, r, :, 1] ** 2))
    assert np.allclose(f, own / own.sum(), rtol=1e-13, atol=0)


def test_invariances_and_consistency_with_the_likelihood_oracle(oracle_mod):
    from oracle.fractions import fit_fractions
    om = random_model(oracle_mod, 26, R=4, H=2, C=2, n_data=50, n_mc=800, weighted=False)
    th = random_theta(27, 4)
    f = fit_fractions(om, th)
    assert np.all(f > 0)
    th2 = th.copy(); th2[1::4] += 0.83; th2[0::4] *= 2.5       # global phase and common scale: unchanged
    assert np.allclose(fit_fractions(om, th2), f, rtol=1e-14, atol=0)
    # the denominator is the normalisation sum G of Eq. 3 as the C oracle computes it
    G = float(oracle_mod.raw_sums(om, "mc", th, None, "ld")[0][0])
    for r in range(4):
        solo = th.copy()
        solo[0::4] = 0.0
        solo[4 * r] = th[4 * r]                                  # only resonance r switched on
        Gr = float(oracle_mod.raw_sums(om, "mc", solo, None, "ld")[0][0])
        assert abs(f[r] - Gr / G) <= 1e-13 * f[r]
    # doubling one coupling quadruples its own numerator
    th3 = th.copy(); th3[0] *= 2.0
    G3 = float(oracle_mod.raw_sums(om, "mc", th3, None, "ld")[0][0])
    assert abs(fit_fractions(om, th3)[0] - 4.0 * f[0] * G / G3) <= 1e-13
