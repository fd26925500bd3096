"""Python face of the CPU oracle (oracle/pwa_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg may import this package.  It shares no code with
paper_2403_09225_b200 and does not import it.

Two builds of the same C file are loaded: `ld` (REAL = long double, the parity reference) and
`d` (REAL = double with compensated sums, OpenMP; the timed CPU baseline).  Parameters, directions
and results are numpy arrays of the build's REAL type; event data is float64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pwa_oracle.c")
_LIBS = {}
_DTYPE = {"ld": np.longdouble, "d": np.float64}


def build(force: bool = False) -> None:
    """Compile both builds of the oracle with gcc (no CUDA involved)."""
    for prec, flag in (("ld", ["-DORACLE_LD"]), ("d", [])):
        out = os.path.join(_HERE, f"libpwa_oracle_{prec}.so")
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
            cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fcx-limited-range", "-fPIC", "-shared", *flag,
                   _SRC, "-o", out, "-lm"]
            subprocess.run(cmd, check=True)


def _lib(prec: str):
    if prec not in _LIBS:
        build()
        _LIBS[prec] = ctypes.CDLL(os.path.join(_HERE, f"libpwa_oracle_{prec}.so"))
    return _LIBS[prec]


def max_threads() -> int:
    return int(getattr(_lib("d"), "oracle_max_threads_d")())


@dataclass
class Sample:
    mass: np.ndarray                 # [C][N] float64
    amp: np.ndarray                  # [R][H][N][2] float64
    weight: Optional[np.ndarray]     # [N] float64 or None

    def __post_init__(self):
        self.mass = np.ascontiguousarray(self.mass, dtype=np.float64)
        self.amp = np.ascontiguousarray(self.amp, dtype=np.float64)
        if self.weight is not None:
            self.weight = np.ascontiguousarray(self.weight, dtype=np.float64)
        assert self.amp.ndim == 4 and self.amp.shape[3] == 2 and self.mass.ndim == 2
        assert self.amp.shape[2] == self.mass.shape[1]

    @property
    def n(self) -> int:
        return self.mass.shape[1]


@dataclass
class Model:
    res_chan: np.ndarray             # [R] int32
    data: Sample
    mc: Sample

    def __post_init__(self):
        self.res_chan = np.ascontiguousarray(self.res_chan, dtype=np.int32)
        assert self.data.amp.shape[:2] == self.mc.amp.shape[:2]
        assert self.res_chan.shape == (self.n_res,)
        assert self.res_chan.min() >= 0 and self.res_chan.max() < self.n_chan

    @property
    def n_res(self) -> int:
        return self.mc.amp.shape[0]

    @property
    def n_hel(self) -> int:
        return self.mc.amp.shape[1]

    @property
    def n_chan(self) -> int:
        return self.mc.mass.shape[0]

    @property
    def n_par(self) -> int:
        return 4 * self.n_res


def model_from_workload(w) -> Model:
    """Build an oracle Model from a workloads.Workload (tensors are copied to host numpy)."""
    to_np = lambda t: None if t is None else t.detach().cpu().numpy()
    return Model(to_np(w.res_chan), Sample(to_np(w.data_mass), to_np(w.data_amp), to_np(w.data_weight)),
                 Sample(to_np(w.mc_mass), to_np(w.mc_amp), None))


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _real(x, prec):
    return None if x is None else np.ascontiguousarray(np.asarray(x, dtype=_DTYPE[prec]))


def raw_sums(model: Model, which: str, theta, v=None, prec: str = "ld", first: int = 0,
             count: Optional[int] = None, threads: int = 1):
    """Raw sums of events first..first+count-1 of the data or MC sample.
    Returns (scal[2], gsum[P], hsum[P] or None); see oracle_raw_sums in pwa_oracle.c."""
    s = model.data if which == "data" else model.mc
    count = s.n - first if count is None else count
    assert 0 <= first and first + count <= s.n
    dt = _DTYPE[prec]
    th, vv = _real(theta, prec), _real(v, prec)
    assert th.shape == (model.n_par,) and (vv is None or vv.shape == th.shape)
    scal, g = np.zeros(2, dt), np.zeros(model.n_par, dt)
    h = np.zeros(model.n_par, dt) if vv is not None else None
    fn = getattr(_lib(prec), f"oracle_raw_sums_{prec}")
    rc = fn(ctypes.c_int(model.n_res), ctypes.c_int(model.n_hel), ctypes.c_int(model.n_chan), _p(model.res_chan),
            ctypes.c_int64(s.n), _p(s.mass), _p(s.amp), _p(s.weight), ctypes.c_int64(first), ctypes.c_int64(count),
            ctypes.c_int(1 if which == "data" else 0), _p(th), _p(vv), _p(scal), _p(g), _p(h),
            ctypes.c_int(threads))
    if rc != 0:
        raise ValueError("oracle_raw_sums: bad sizes")
    return scal, g, h


def combine(scal_data, scal_mc, gd, gG, hd=None, hG=None, v=None, prec: str = "ld"):
    """Eqs. 4, 6, 7 on raw sums already added over shards -> (nll, grad, hv or None)."""
    dt = _DTYPE[prec]
    sd, sm, gd, gG = _real(scal_data, prec), _real(scal_mc, prec), _real(gd, prec), _real(gG, prec)
    hd, hG, vv = _real(hd, prec), _real(hG, prec), _real(v, prec)
    P = gd.shape[0]
    nll, grad = np.zeros(1, dt), np.zeros(P, dt)
    hv = np.zeros(P, dt) if vv is not None else None
    getattr(_lib(prec), f"oracle_combine_{prec}")(ctypes.c_int(P), _p(sd), _p(sm), _p(gd), _p(gG), _p(hd), _p(hG),
                                                   _p(vv), _p(nll), _p(grad), _p(hv))
    return nll[0], grad, hv


def nll_grad_hvp(model: Model, theta, v=None, prec: str = "ld", threads: int = 1):
    """NLL, gradient and (if v is given) Hessian-vector product over the whole model."""
    sd, gd, hd = raw_sums(model, "data", theta, v, prec, threads=threads)
    sm, gG, hG = raw_sums(model, "mc", theta, v, prec, threads=threads)
    return combine(sd, sm, gd, gG, hd, hG, v, prec)


def nll(model: Model, theta, prec: str = "ld", threads: int = 1):
    return nll_grad_hvp(model, theta, None, prec, threads)[0]


def intensity(model: Model, which: str, theta, first: int = 0, count: Optional[int] = None, prec: str = "ld"):
    s = model.data if which == "data" else model.mc
    count = s.n - first if count is None else count
    out = np.zeros(count, np.float64)
    th = _real(theta, prec)
    rc = getattr(_lib(prec), f"oracle_intensity_{prec}")(
        ctypes.c_int(model.n_res), ctypes.c_int(model.n_hel), ctypes.c_int(model.n_chan), _p(model.res_chan),
        ctypes.c_int64(s.n), _p(s.mass), _p(s.amp), ctypes.c_int64(first), ctypes.c_int64(count), _p(th), _p(out))
    if rc != 0:
        raise ValueError("oracle_intensity: bad sizes")
    return out


def event(model: Model, which: str, i: int, theta, v=None, prec: str = "ld"):
    """(I_i, g_i.v, g_i[P], (H_i v)[P]) of one event."""
    s = model.data if which == "data" else model.mc
    dt = _DTYPE[prec]
    th, vv = _real(theta, prec), _real(v, prec)
    I, Idot = np.zeros(1, dt), np.zeros(1, dt)
    g, hv = np.zeros(model.n_par, dt), np.zeros(model.n_par, dt)
    rc = getattr(_lib(prec), f"oracle_event_{prec}")(
        ctypes.c_int(model.n_res), ctypes.c_int(model.n_hel), ctypes.c_int(model.n_chan), _p(model.res_chan),
        ctypes.c_int64(s.n), _p(s.mass), _p(s.amp), ctypes.c_int64(i), _p(th), _p(vv), _p(I), _p(Idot), _p(g), _p(hv))
    if rc != 0:
        raise ValueError("oracle_event: bad sizes")
    return I[0], Idot[0], g, (hv if vv is not None else None)
