"""Pins for the reference fit (oracle/fit.py), which follows SURVEY §8(c-F) on the oracle's NLL / gradient / HVP.

The fit is an iteration, so it is pinned by what does not depend on its trajectory:
  - SciPy's Newton-CG (the optimiser the paper names) fed with the same oracle callbacks reaches
    the same minimum from the same start (an independent implementation of the same method);
  - at the returned point the gradient vanishes and the Hessian is positive along random directions;
  - the NLL never increases along the trace (Armijo), and the S19 box holds at every accepted point.
"""
import numpy as np
import pytest

from helpers import random_model, random_theta


@pytest.fixture(scope="module")
def toy(oracle_mod):
    import workloads
    cfg = workloads.CONFIGS[1].scaled(6_000, 1_200)
    w = workloads.make_workload(cfg, "cpu", chunk=1 << 12, imax_events=6_000)
    return cfg, oracle_mod.model_from_workload(w), workloads.theta_true(cfg).numpy()


def test_fit_from_theta_true_converges_and_matches_scipy(oracle_mod, toy):
    from scipy.optimize import minimize
    from oracle.fit import fit_newton_cg
    cfg, om, th0 = toy
    res = fit_newton_cg(om, th0, prec="d", threads=oracle_mod.max_threads())
    assert res.converged and res.stop_reason in (1, 2, 3)
    assert res.grad_inf_norm < 1e-2
    f0 = float(oracle_mod.nll(om, th0, "d"))
    assert res.nll < f0                       # data drawn at theta_true: the fit still gains O(P/2)
    assert f0 - res.nll < 10 * cfg.n_par      # ... and not more than a statistical fluctuation's worth
    vals = [f for (_, f, _) in res.trace]
    assert all(b <= a + 1e-9 * abs(a) for a, b in zip(vals, vals[1:]))

    fun = lambda t: float(oracle_mod.nll(om, t, "d"))
    jac = lambda t: np.asarray(oracle_mod.nll_grad_hvp(om, t, None, "d")[1], dtype=np.float64)
    hessp = lambda t, p: np.asarray(oracle_mod.nll_grad_hvp(om, t, p, "d")[2], dtype=np.float64)
    sp = minimize(fun, th0, jac=jac, hessp=hessp, method="Newton-CG", options={"xtol": 1e-10, "maxiter": 400})
    assert abs(sp.fun - res.nll) <= 1e-7 * max(1.0, abs(sp.fun)), (sp.fun, res.nll)


def test_minimum_is_stationary_with_positive_curvature(oracle_mod, toy):
    from oracle.fit import fit_newton_cg
    cfg, om, th0 = toy
    res = fit_newton_cg(om, th0, prec="d", threads=oracle_mod.max_threads())
    th = np.asarray(res.theta, dtype=np.float64)
    rs = np.random.RandomState(5)
    # gauge directions (global phase, common scale) are flat: project them out of the probe
    u = np.zeros_like(th); u[0::4] = th[0::4]
    ph = np.zeros_like(th); ph[1::4] = 1.0
    for _ in range(4):
        v = rs.normal(size=th.shape)
        for gdir in (u, ph):
            v -= gdir * (v @ gdir) / (gdir @ gdir)
        _, g, hv = oracle_mod.nll_grad_hvp(om, th, v, "ld")
        assert float(np.max(np.abs(g))) < 1e-2
        assert float(np.dot(v, np.asarray(hv, dtype=np.float64))) > 0.0


def test_box_is_respected_and_bad_start_is_reported(oracle_mod):
    from oracle.fit import FitOpts, fit_newton_cg
    om = random_model(oracle_mod, 3, R=2, H=2, C=1, n_data=300, n_mc=1500, weighted=False)
    th0 = random_theta(4, 2)
    o = FitOpts(max_outer=30)
    res = fit_newton_cg(om, th0, o, prec="d")
    th = np.asarray(res.theta, dtype=np.float64)
    assert np.all(th[3::4] >= o.gamma_min) and np.all(th[3::4] <= o.gamma_max)
    assert np.all(th[2::4] >= o.mass_min) and np.all(th[2::4] <= o.mass_max)
    assert res.nll <= float(oracle_mod.nll(om, th0, "d"))
    assert res.stop_reason in (1, 2, 3, 4, 6)


def test_active_bound_minimum_matches_scipy_lbfgsb(oracle_mod, toy):
    """The projected Newton-CG of DESIGN.md S15'/S19 against SciPy's L-BFGS-B (an independent bound-constrained
    optimiser) on a box that cuts the unconstrained minimum off: same NLL, KKT conditions at the returned point."""
    from scipy.optimize import minimize
    from oracle.fit import FitOpts, bounds, fit_newton_cg, projected_gradient
    cfg, om, th0 = toy
    free_fit = fit_newton_cg(om, th0, prec="d", threads=oracle_mod.max_threads())
    g_hat = np.asarray(free_fit.theta, dtype=np.float64)[3::4]
    # upper width bound below the smallest fitted width, lower mass bound above the smallest fitted mass
    o = FitOpts(gamma_max=0.8 * float(g_hat.min()), mass_min=float(np.asarray(free_fit.theta, dtype=np.float64)[2::4].min()) + 0.02)
    res = fit_newton_cg(om, th0, o, prec="d", threads=oracle_mod.max_threads())
    assert res.converged and res.n_active >= 2 and res.nll > free_fit.nll
    th = np.asarray(res.theta, dtype=np.float64)
    lo, hi = bounds(len(th), o)
    assert np.all(th >= lo) and np.all(th <= hi)
    _, g, _ = oracle_mod.nll_grad_hvp(om, th, None, "d")
    g = np.asarray(g, dtype=np.float64)
    gP, free = projected_gradient(th, g, lo, hi)
    assert float(np.max(np.abs(gP))) < 1e-2                 # stationary on the free variables
    assert np.all(g[~free & (th <= lo)] > 0) and np.all(g[~free & (th >= hi)] < 0)  # multipliers have the right sign
    vals = [f for (_, f, _) in res.trace]
    assert all(b <= a + 1e-9 * abs(a) for a, b in zip(vals, vals[1:]))

    fun = lambda t: float(oracle_mod.nll(om, t, "d"))
    jac = lambda t: np.asarray(oracle_mod.nll_grad_hvp(om, t, None, "d")[1], dtype=np.float64)
    sp = minimize(fun, np.clip(th0, lo, hi), jac=jac, method="L-BFGS-B", bounds=list(zip(lo, hi)),
                  options={"maxiter": 2000, "ftol": 1e-15, "gtol": 1e-8})
    assert abs(sp.fun - res.nll) <= 1e-7 * max(1.0, abs(sp.fun)), (sp.fun, res.nll)


def test_start_outside_the_box_is_projected(oracle_mod):
    from oracle.fit import FitOpts, fit_newton_cg
    om = random_model(oracle_mod, 3, R=2, H=2, C=1, n_data=300, n_mc=1500, weighted=False)
    th0 = random_theta(4, 2)
    th0[3] = 5.0      # Gamma_0 above gamma_max
    th0[6] = 0.01     # M_1 below mass_min
    o = FitOpts(max_outer=0)
    res = fit_newton_cg(om, th0, o, prec="d")
    th = np.asarray(res.theta, dtype=np.float64)
    assert th[3] == o.gamma_max and th[6] == o.mass_min and res.stop_reason == 4
    assert res.nll == float(oracle_mod.nll(om, th, "d"))
