"""Reference fit: truncated line-search Newton-CG on top of the CPU oracle's NLL / gradient / HVP.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rule as oracle/__init__.py).  It follows SURVEY.md §8(c-F)
(S15, S19) step by step, in that order and notation; the paper only names SciPy's Newton-CG
 and the configuration asks for "<= 50 CG iterations per outer step, Armijo line search"
(BASELINE.json configs[4]).  Plain numpy, one HVP per CG iteration, no shortcuts:

  1. f, g at theta.  Stop (gtol) if |g|_inf <= gtol.
  2. eps = min(0.5, sqrt(|g|_2)) |g|_2 ;  z = 0, r = g, d = -g.
  3. for j < max_cg:  q = H d;  gamma = d.q.
       if gamma <= 1e-14 d.d:  p = -g if j == 0 else z;  leave.
       alpha = r.r / gamma;  z += alpha d;  r_new = r + alpha q;  if |r_new|_2 <= eps:  p = z;  leave.
       beta = r_new.r_new / r.r;  d = -r_new + beta d;  r = r_new.            exhausted:  p = z.
  4. Armijo: t = 1; while theta + t p leaves the box (S19), or f(theta + t p) is not finite, or
       f(theta + t p) > f + c1 t g.p :  t *= rho;  give up after max_backtrack shrinks.
  5. theta += t p.  Stop if t |p|_inf <= xtol (2) or |f_new - f| <= ftol max(1, |f|) (3), or max_outer (4).
  converged  <=>  stopped on test 1, 2 or 3  and  |g|_inf <= gconv.
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
    trace: list = field(default_factory=list)


def _feasible(theta: np.ndarray, o: FitOpts) -> bool:
    M, G = theta[2::4], theta[3::4]
    ok = True
    if not (o.gamma_min == 0.0 and o.gamma_max == 0.0):
        ok = ok and bool(np.all(G >= o.gamma_min) and np.all(G <= o.gamma_max))
    if not (o.mass_min == 0.0 and o.mass_max == 0.0):
        ok = ok and bool(np.all(M >= o.mass_min) and np.all(M <= o.mass_max))
    return ok


def fit_newton_cg(model, theta0, opts: FitOpts | None = None, prec: str = "d", threads: int = 1) -> FitResult:
    o = opts or FitOpts()
    dt = np.longdouble if prec == "ld" else np.float64
    theta = np.array(theta0, dtype=dt)
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
        ginf = float(np.max(np.abs(g)))
        res.trace.append((outer, float(f), ginf))
        if not (np.isfinite(float(f)) and np.isfinite(ginf)):
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
        gnorm = float(np.sqrt(np.dot(g, g)))
        eps = min(0.5, np.sqrt(gnorm)) * gnorm
        z = np.zeros_like(g)
        r = g.copy()
        d = -g
        p = None
        # step 3
        for j in range(o.max_cg):
            q = hvp(theta, d)
            res.cg_iters += 1
            gamma = np.dot(d, q)
            if gamma <= 1e-14 * np.dot(d, d):
                p = -g if j == 0 else z.copy()
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
        gp = np.dot(g, p)
        t = dt(1.0)
        accepted = False
        f_new = f
        for _ in range(o.max_backtrack + 1):
            trial = theta + t * p
            if _feasible(trial, o):
                f_new = dt(_nll(model, trial, prec, threads=threads))
                res.n_nll += 1
                if np.isfinite(float(f_new)) and f_new <= f + o.armijo_c1 * t * gp:
                    accepted = True
                    break
            t = t * o.backtrack
        if not accepted:
            stop = 6
            break
        # step 5
        theta = theta + t * p
        step_inf = float(t * np.max(np.abs(p)))
        f_old = f
        f, g = value_grad(theta)
        if step_inf <= o.xtol:
            stop = 2
        elif abs(float(f_new - f_old)) <= o.ftol * max(1.0, abs(float(f_old))):
            stop = 3
        if stop:
            res.trace.append((outer, float(f), float(np.max(np.abs(g)))))
            break
    res.theta = theta
    res.nll = float(f)
    res.grad_inf_norm = float(np.max(np.abs(g)))
    res.stop_reason = stop
    res.converged = stop in (1, 2, 3) and res.grad_inf_norm <= o.gconv
    return res
