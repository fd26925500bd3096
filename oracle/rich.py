"""Python face of the richer-model oracle (oracle/pwa_oracle_rich.c): partial waves sharing resonance lineshapes,
lineshape kinds (constant width, mass-dependent width, Flatte).  DESIGN.md readings S21, S22; SURVEY.md 8(f) rank 3.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rule as oracle/__init__.py).  Shares no code with paper_2403_09225_b200.
Parameters: theta = [a_0, phi_0, ..., a_{W-1}, phi_{W-1}, M_0, Gamma_0, ..., M_{L-1}, Gamma_{L-1}].
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import Sample, _DTYPE, _p, _real, combine

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pwa_oracle_rich.c")
_LIBS = {}
N_SP = 6
KIND_CONST, KIND_MASSDEP, KIND_FLATTE = 0, 1, 2


def build(force: bool = False) -> None:
    for prec, flag in (("ld", ["-DORACLE_LD"]), ("d", [])):
        out = os.path.join(_HERE, f"libpwa_oracle_rich_{prec}.so")
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
            subprocess.run(["gcc", "-O2", "-std=c11", "-fopenmp", "-fcx-limited-range", "-fPIC", "-shared", *flag,
                            _SRC, "-o", out, "-lm"], check=True)


def _lib(prec: str):
    if prec not in _LIBS:
        build()
        _LIBS[prec] = ctypes.CDLL(os.path.join(_HERE, f"libpwa_oracle_rich_{prec}.so"))
    return _LIBS[prec]


@dataclass
class RichModel:
    wave_res: np.ndarray          # [W] int32: resonance (lineshape) of each partial wave
    res_chan: np.ndarray          # [L] int32: mass channel of each resonance
    kind: np.ndarray              # [L] int32: 0 constant width, 1 mass-dependent width, 2 Flatte
    shape: np.ndarray             # [L][6] float64: kind 1 (m1, m2, L); kind 2 (m1, m2, m3, m4, g2/g1)
    data: Sample
    mc: Sample

    def __post_init__(self):
        self.wave_res = np.ascontiguousarray(self.wave_res, dtype=np.int32)
        self.res_chan = np.ascontiguousarray(self.res_chan, dtype=np.int32)
        self.kind = np.ascontiguousarray(self.kind, dtype=np.int32)
        self.shape = np.ascontiguousarray(self.shape, dtype=np.float64)
        assert self.shape.shape == (self.n_ls, N_SP) and self.kind.shape == (self.n_ls,)
        assert self.wave_res.shape == (self.n_wave,) and 0 <= self.wave_res.min() and self.wave_res.max() < self.n_ls
        assert self.data.amp.shape[:2] == self.mc.amp.shape[:2]

    @property
    def n_wave(self) -> int:
        return self.mc.amp.shape[0]

    @property
    def n_ls(self) -> int:
        return self.res_chan.shape[0]

    @property
    def n_hel(self) -> int:
        return self.mc.amp.shape[1]

    @property
    def n_chan(self) -> int:
        return self.mc.mass.shape[0]

    @property
    def n_par(self) -> int:
        return 2 * self.n_wave + 2 * self.n_ls


def raw_sums(model: RichModel, which: str, theta, v=None, prec: str = "ld", first: int = 0,
             count: Optional[int] = None, threads: int = 1):
    s = model.data if which == "data" else model.mc
    count = s.n - first if count is None else count
    dt = _DTYPE[prec]
    th, vv = _real(theta, prec), _real(v, prec)
    assert th.shape == (model.n_par,) and (vv is None or vv.shape == th.shape)
    scal, g = np.zeros(2, dt), np.zeros(model.n_par, dt)
    h = np.zeros(model.n_par, dt) if vv is not None else None
    rc = getattr(_lib(prec), f"rich_raw_sums_{prec}")(
        ctypes.c_int(model.n_wave), ctypes.c_int(model.n_ls), ctypes.c_int(model.n_hel), ctypes.c_int(model.n_chan),
        _p(model.wave_res), _p(model.res_chan), _p(model.kind), _p(model.shape), ctypes.c_int64(s.n), _p(s.mass),
        _p(s.amp), _p(s.weight), ctypes.c_int64(first), ctypes.c_int64(count), ctypes.c_int(1 if which == "data" else 0),
        _p(th), _p(vv), _p(scal), _p(g), _p(h), ctypes.c_int(threads))
    if rc != 0:
        raise ValueError("rich_raw_sums: bad sizes")
    return scal, g, h


def nll_grad_hvp(model: RichModel, theta, v=None, prec: str = "ld", threads: int = 1):
    """NLL, gradient, HVP: raw sums of both samples, then Eqs. 4, 6, 7 (oracle.combine)."""
    sd, gd, hd = raw_sums(model, "data", theta, v, prec, threads=threads)
    sm, gG, hG = raw_sums(model, "mc", theta, v, prec, threads=threads)
    return combine(sd, sm, gd, gG, hd, hG, v, prec)


def nll(model: RichModel, theta, prec: str = "ld", threads: int = 1):
    return nll_grad_hvp(model, theta, None, prec, threads)[0]


def intensity(model: RichModel, which: str, theta, prec: str = "ld"):
    s = model.data if which == "data" else model.mc
    out = np.zeros(s.n, np.float64)
    rc = getattr(_lib(prec), f"rich_intensity_{prec}")(
        ctypes.c_int(model.n_wave), ctypes.c_int(model.n_ls), ctypes.c_int(model.n_hel), ctypes.c_int(model.n_chan),
        _p(model.wave_res), _p(model.res_chan), _p(model.kind), _p(model.shape), ctypes.c_int64(s.n), _p(s.mass),
        _p(s.amp), ctypes.c_int64(0), ctypes.c_int64(s.n), _p(_real(theta, prec)), _p(out))
    if rc != 0:
        raise ValueError("rich_intensity: bad sizes")
    return out
