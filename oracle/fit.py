"""Reference fit: projected, truncated line-search Newton-CG on top of the CPU oracle's NLL / gradient / HVP.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rule as oracle/__init__.py).  It follows DESIGN.md reading S15' / S19
step by step, in that order and notation.  The paper only names SciPy's Newton-CG, mentions
undefined "constraint conditions" and the configuration asks for "<= 50 CG iterations per outer step,
Armijo line search" (BASELINE.json configs[4]).  The box of S19 (Gamma_r in [gamma_min, gamma_max], M_r in
[mass_min, mass_max]; a_r, phi_r free) is treated the textbook way for bound constraints (Bertsekas, projected
Newton; Nocedal & Wright, Numerical Optimization, ch. 16.7 gradient projection + Alg. 7.1 for the inner CG):
variables that sit on a bound with the gradient pushing outward are frozen for the inner solve, and trial points are
projected onto the box instead of being rejected.  Plain numpy, one HVP per CG iteration, no shortcuts:

  0. theta <- clip(theta0, lo, hi).
  1. f, g at theta.  Active set A = {k : (theta_k <= lo_k and g_k > 0) or (theta_k >= hi_k and g_k < 0)};
     projected gradient gP = g with the entries of A set to 0.  Stop (1) if |gP|_inf <= gtol.
  2. eps = min(0.5, sqrt(|gP|_2)) |gP|_2 ;  z = 0, r = gP, d = -gP.
  3. for j < max_cg:  q = H d with the entries of A set to 0;  gamma = d.q.
       if gamma <= 1e-14 d.d:  p = -gP if j == 0 else z;  leave.
       alpha = r.r / gamma;  z += alpha d;  r_new = r + alpha q;  if |r_new|_2 <= eps:  p = z;  leave.
       beta = r_new.r_new / r.r;  d = -r_new + beta d;  r = r_new.            exhausted:  p = z.
  4. Projected Armijo: t = 1; trial = clip(theta + t p), s = trial - theta; while f(trial) is not finite or
       f(trial) > f + c1 g.s :  t *= rho.  After max_backtrack shrinks: if p was not -gP, restart this step once with
       p = -gP, t = 1; otherwise give up (6).
  5. theta <- trial.  Stop if |s|_inf <= xtol (2) or |f_new - f| <= ftol max(1, |f|) (3), or max_outer (4).
  converged  <=>  stopped on test 1, 2 or 3  and  |gP|_inf <= gconv  (gP of the final point).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import nll as _nll
from . import nll_grad_hvp as _nll_grad_hvp


@dataclass
class FitOpts:
    max_outer: int = 500
    max_cg: int = 50
    gtol: float = 1e-5
    xtol: float = 1e-8
    ftol: float = 1e-12
    armijo_c1: float = 1e-4
    backtrack: float = 0.5
    max_backtrack: int = 40
    gamma_min: float = 5e-3
    gamma_max: float = 2.0
    mass_min: float = 0.1
    mass_max: float = 4.0
    gconv: float = 1.0


@dataclass
class FitResult:
    theta: np.ndarray
    nll: float
    grad_inf_norm: float
    outer_iters: int = 0
    cg_iters: int = 0
    n_nll: int = 0
    n_grad: int = 0
    n_hvp: int = 0
    stop_reason: int = 0
    converged: bool = False
    n_active: int = 0
    trace: list = field(default_factory=list)


def bounds(n_par: int, o: FitOpts, dt=np.float64):
    """lo[k], hi[k] of reading S19: only M (k % 4 == 2) and Gamma (k % 4 == 3) are boxed; a pair of zeros = no box."""
    lo = np.full(n_par, -np.inf, dtype=dt)
    hi = np.full(n_par, np.inf, dtype=dt)
    if not (o.mass_min == 0.0 and o.mass_max == 0.0):
        lo[2::4], hi[2::4] = o.mass_min, o.mass_max
    if not (o.gamma_min == 0.0 and o.gamma_max == 0.0):
        lo[3::4], hi[3::4] = o.gamma_min, o.gamma_max
    return lo, hi


def projected_gradient(theta, g, lo, hi):
    """g with the entries of the active set (on a bound, gradient pushing outward) set to zero; the mask of free entries."""
    active = ((theta <= lo) & (g > 0)) | ((theta >= hi) & (g < 0))
    free = ~active
    return np.where(free, g, 0), free


def fit_newton_cg(model, theta0, opts: FitOpts | None = None, prec: str = "d", threads: int = 1) -> FitResult:
    o = opts or FitOpts()
    dt = np.longdouble if prec == "ld" else np.float64
    lo, hi = bounds(len(theta0), o, dt)
    theta = np.clip(np.array(theta0, dtype=dt), lo, hi)  # step 0
    res = FitResult(theta=theta, nll=np.nan, grad_inf_norm=np.nan)

    def value_grad(th):
        f, g, _ = _nll_grad_hvp(model, th, None, prec, threads=threads)
        res.n_grad += 1
        return dt(f), np.asarray(g, dtype=dt)

    def hvp(th, d):
        _, _, q = _nll_grad_hvp(model, th, d, prec, threads=threads)
        res.n_hvp += 1
        return np.asarray(q, dtype=dt)

    f, g = value_grad(theta)
    stop = 0
    outer = 0
    while True:
        # step 1
        gP, free = projected_gradient(theta, g, lo, hi)
        ginf = float(np.max(np.abs(gP)))
        res.trace.append((outer, float(f), ginf))
        if not (np.isfinite(float(f)) and np.isfinite(float(np.max(np.abs(g))))):
            stop = -1
            break
        if ginf <= o.gtol:
            stop = 1
            break
        if outer >= o.max_outer:
            stop = 4
            break
        outer += 1
        res.outer_iters = outer
        # step 2
        gnorm = float(np.sqrt(np.dot(gP, gP)))
        eps = min(0.5, np.sqrt(gnorm)) * gnorm
        z = np.zeros_like(gP)
        r = gP.copy()
        d = -gP
        p = None
        # step 3
        for j in range(o.max_cg):
            q = np.where(free, hvp(theta, d), 0)
            res.cg_iters += 1
            gamma = np.dot(d, q)
            if not (gamma > 1e-14 * np.dot(d, d)):
                p = -gP if j == 0 else z.copy()
                break
            rr = np.dot(r, r)
            alpha = rr / gamma
            z = z + alpha * d
            r_new = r + alpha * q
            if float(np.sqrt(np.dot(r_new, r_new))) <= eps:
                p = z.copy()
                break
            beta = np.dot(r_new, r_new) / rr
            d = -r_new + beta * d
            r = r_new
        if p is None:
            p = z.copy()
        # step 4
        accepted = False
        f_new = f
        is_sd = bool(np.array_equal(p, -gP))
        while True:
            t = dt(1.0)
            for _ in range(o.max_backtrack + 1):
                trial = np.clip(theta + t * p, lo, hi)
                s = trial - theta
                f_new = dt(_nll(model, trial, prec, threads=threads))
                res.n_nll += 1
                if np.isfinite(float(f_new)) and f_new <= f + o.armijo_c1 * np.dot(g, s):
                    accepted = True
                    break
                t = t * o.backtrack
            if accepted or is_sd:
                break
            p, is_sd = -gP, True  # one restart along the projected steepest descent
        if not accepted:
            stop = 6
            break
        # step 5
        step_inf = float(np.max(np.abs(s)))
        theta = trial
        f_old = f
        f, g = value_grad(theta)
        if step_inf <= o.xtol:
            stop = 2
        elif abs(float(f_new - f_old)) <= o.ftol * max(1.0, abs(float(f_old))):
            stop = 3
        if stop:
            gP, free = projected_gradient(theta, g, lo, hi)
            res.trace.append((outer, float(f), float(np.max(np.abs(gP)))))
            break
    gP, free = projected_gradient(theta, g, lo, hi)
    res.theta = theta
    res.nll = float(f)
    res.grad_inf_norm = float(np.max(np.abs(gP)))
    res.n_active = int(np.sum(~free))
    res.stop_reason = stop
    res.converged = stop in (1, 2, 3) and res.grad_inf_norm <= o.gconv
    return res
