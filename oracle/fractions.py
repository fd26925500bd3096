"""Fit fractions of the resonances (TEST INFRASTRUCTURE, see oracle/__init__.py).

PAPER.md:102-113 (section 3, Table 1) lists a "fraction" F_i for every resonance of its model without printing the
formula; the reading taken (S20) is the standard one of partial wave analyses, evaluated on the phase-space
Monte-Carlo sample exactly like the normalisation integral of Eq. 3:

    F_r = sum_j sum_h | z_r(j) F_rh(j) |^2  /  sum_j I_j ,      z_r = c_r B_r,   I_j = sum_h | sum_r z_r F_rh |^2

(interference makes sum_r F_r differ from 1).  Plain numpy in 80-bit arithmetic, one resonance at a time, the
definition written out; no blocking, no reuse of anything under paper_2403_09225_b200/.
"""
from __future__ import annotations

import numpy as np


def fit_fractions(model, theta) -> np.ndarray:
    """model: oracle.Model; theta[4R] = (a, phi, M, Gamma) per resonance.  Returns F[R] (float64)."""
    ld, cld = np.longdouble, np.clongdouble
    th = np.asarray(theta, dtype=ld).reshape(-1, 4)
    R, H = model.n_res, model.n_hel
    assert th.shape[0] == R
    mc = model.mc
    mass = np.asarray(mc.mass, dtype=ld)                                   # [C][N]
    amp = np.asarray(mc.amp, dtype=ld)                                     # [R][H][N][2]
    n = mass.shape[1]
    A = np.zeros((H, n), dtype=cld)
    own = np.zeros(R, dtype=ld)
    for r in range(R):
        a, phi, M, G = th[r]
        m = mass[int(model.res_chan[r])]
        D = (M * M - m * m).astype(cld) - 1j * cld(M * G)                  # D = M^2 - m^2 - i M Gamma
        z = (a * (np.cos(phi) + 1j * np.sin(phi))).astype(cld) / D         # z = c B
        for h in range(H):
            F = amp[r, h, :, 0].astype(cld) + 1j * amp[r, h, :, 1].astype(cld)
            t = z * F
            A[h] += t
            own[r] += np.sum(t.real * t.real + t.imag * t.imag)
    total = np.sum(A.real * A.real + A.imag * A.imag)
    return np.asarray(own / total, dtype=np.float64)


def fit_fractions_rich(model, theta) -> np.ndarray:
    """Richer model (oracle/rich.py; S20, S21): one fraction per RESONANCE l, the coherent sum of its partial
    waves,  F_l = sum_j sum_h | sum_{m in l} z_m(j) F_mh(j) |^2 / sum_j I_j.  Written as the definition says it: the
    numerator is the MC intensity sum with every coupling outside resonance l switched off.  model: oracle.rich.RichModel;
    theta in its [waves | resonances] layout.  Returns F[L] (float64)."""
    from . import rich
    ld = np.longdouble
    th = np.asarray(theta, dtype=ld)
    W, L = model.n_wave, model.n_ls
    total = np.sum(np.asarray(rich.intensity(model, "mc", th, "ld"), dtype=ld))
    out = np.zeros(L, dtype=ld)
    for l in range(L):
        only = th.copy()
        for m in range(W):
            if int(model.wave_res[m]) != l:
                only[2 * m] = 0
        out[l] = np.sum(np.asarray(rich.intensity(model, "mc", only, "ld"), dtype=ld)) / total
    return np.asarray(out, dtype=np.float64)
