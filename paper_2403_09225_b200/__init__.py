"""Thin Python binding of libpwa_b200.so (include/pwa.h): argument marshalling only.

Every step of the likelihood path runs in the library's CUDA kernels; PyTorch is used here for device
memory (tensors whose data_ptr() is handed to the C ABI) and streams.  There is no CPU fallback: if
the shared library is missing or no CUDA device is usable the calls raise.

Function names mirror the C ABI: pwa_create, pwa_nll, pwa_nll_grad, pwa_hvp, pwa_nll_grad_hvp,
pwa_raw_sums, pwa_combine, pwa_fit_newton_cg, pwa_nll_grad_hvp_host, ...
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_double, c_int32, c_int64, c_uint32, c_void_p
from typing import Optional

__all__ = ["PwaError", "lib_path", "load", "pwa_create", "pwa_create_rich", "pwa_rich_desc", "PWA_LS_CONST", "PWA_LS_MASSDEP", "PWA_LS_FLATTE", "pwa_destroy", "pwa_n_params", "pwa_raw_size", "pwa_nll",
           "pwa_nll_grad", "pwa_hvp", "pwa_nll_grad_hvp", "pwa_raw_sums", "pwa_combine", "pwa_fit_opts",
           "pwa_fit_result", "pwa_fit_opts_default", "pwa_fit_newton_cg", "pwa_nll_grad_hvp_host", "pwa_nll_grad_hvp_static", "pwa_fit_fractions",
           "pwa_nll_grad_for_hvp", "pwa_hvp_cached", "pwa_nll_batch", "pwa_hvp_cached_batch", "pwa_hessian",
           "pwa_status_flags", "pwa_profile_enable", "pwa_profile_read", "pwa_kernel_launches", "pwa_bytes_per_eval",
           "pwa_kernel_variant", "pwa_last_error", "pwa_version", "Model", "STATUS_NAMES", "EXPORTS"]

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

PWA_OK, PWA_ERR_INVALID_ARG, PWA_ERR_CUDA, PWA_ERR_OOM, PWA_ERR_NONFINITE, PWA_ERR_NOT_CONVERGED = range(6)
STATUS_NAMES = ["PWA_OK", "PWA_ERR_INVALID_ARG", "PWA_ERR_CUDA", "PWA_ERR_OOM", "PWA_ERR_NONFINITE",
                "PWA_ERR_NOT_CONVERGED"]
PWA_MEM_HOST, PWA_MEM_DEVICE = 0, 1
PWA_LS_CONST, PWA_LS_MASSDEP, PWA_LS_FLATTE = 0, 1, 2

# every symbol include/pwa.h declares
EXPORTS = ["pwa_create", "pwa_create_rich", "pwa_destroy", "pwa_n_params", "pwa_nll", "pwa_nll_grad", "pwa_hvp", "pwa_nll_grad_hvp",
           "pwa_raw_size", "pwa_raw_sums", "pwa_combine", "pwa_fit_opts_default", "pwa_fit_newton_cg",
           "pwa_nll_grad_hvp_host", "pwa_nll_grad_hvp_static", "pwa_fit_fractions", "pwa_nll_grad_for_hvp", "pwa_hvp_cached", "pwa_nll_batch", "pwa_hvp_cached_batch", "pwa_hessian",
           "pwa_status_flags", "pwa_profile_enable", "pwa_profile_read",
           "pwa_kernel_launches", "pwa_bytes_per_eval", "pwa_kernel_variant", "pwa_last_error", "pwa_version"]


class PwaError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else status}: {msg}")
        self.status = status


class pwa_sample(Structure):
    _fields_ = [("n_events", c_int64), ("stride", c_int64), ("mass", c_void_p), ("amp", c_void_p),
                ("weight", c_void_p)]


class pwa_model_desc(Structure):
    _fields_ = [("n_res", c_int32), ("n_hel", c_int32), ("n_chan", c_int32), ("res_chan", c_void_p),
                ("data", pwa_sample), ("mc", pwa_sample), ("mem", c_int32), ("borrow", c_int32),
                ("device", c_int32), ("stream", c_void_p)]


class pwa_rich_desc(Structure):
    _fields_ = [("n_lineshape", c_int32), ("wave_res", c_void_p), ("ls_chan", c_void_p), ("ls_kind", c_void_p),
                ("ls_shape", c_void_p)]


class pwa_fit_opts(Structure):
    _fields_ = [("max_outer", c_int32), ("max_cg", c_int32), ("gtol", c_double), ("xtol", c_double),
                ("ftol", c_double), ("armijo_c1", c_double), ("backtrack", c_double), ("max_backtrack", c_int32),
                ("max_seconds", c_double), ("gamma_min", c_double), ("gamma_max", c_double),
                ("mass_min", c_double), ("mass_max", c_double), ("gconv", c_double)]


class pwa_fit_result(Structure):
    _fields_ = [("nll", c_double), ("grad_inf_norm", c_double), ("outer_iters", c_int32), ("cg_iters", c_int32),
                ("n_nll", c_int32), ("n_grad", c_int32), ("n_hvp", c_int32), ("stop_reason", c_int32),
                ("status", c_int32), ("seconds", c_double), ("n_active", c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def lib_path() -> str:
    return os.path.join(_HERE, "libpwa_b200.so")


def load():
    """Loads libpwa_b200.so (built by `python -m paper_2403_09225_b200.build`).  Raises if it is missing."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = lib_path()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_2403_09225_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    vp, dp = c_void_p, c_void_p
    lib.pwa_create.argtypes = [POINTER(pwa_model_desc), POINTER(vp)]
    lib.pwa_create_rich.argtypes = [POINTER(pwa_model_desc), POINTER(pwa_rich_desc), POINTER(vp)]
    lib.pwa_destroy.argtypes = [vp]
    lib.pwa_n_params.argtypes = [vp]
    lib.pwa_raw_size.argtypes = [vp]
    lib.pwa_nll.argtypes = [vp, dp, dp]
    lib.pwa_nll_grad.argtypes = [vp, dp, dp, dp]
    lib.pwa_hvp.argtypes = [vp, dp, dp, dp]
    lib.pwa_nll_grad_hvp.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.pwa_raw_sums.argtypes = [vp, dp, dp, dp]
    lib.pwa_combine.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.pwa_fit_opts_default.argtypes = [POINTER(pwa_fit_opts)]
    lib.pwa_fit_opts_default.restype = None
    lib.pwa_fit_newton_cg.argtypes = [vp, dp, POINTER(pwa_fit_opts), POINTER(pwa_fit_result)]
    lib.pwa_nll_grad_hvp_host.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.pwa_nll_grad_hvp_static.argtypes = [POINTER(pwa_model_desc), dp, dp, dp, dp, dp]
    lib.pwa_fit_fractions.argtypes = [vp, dp, dp]
    lib.pwa_nll_grad_for_hvp.argtypes = [vp, dp, dp, dp]
    lib.pwa_hvp_cached.argtypes = [vp, dp, dp]
    lib.pwa_nll_batch.argtypes = [vp, c_int32, dp, dp]
    lib.pwa_hvp_cached_batch.argtypes = [vp, c_int32, dp, dp]
    lib.pwa_hessian.argtypes = [vp, dp, dp]
    lib.pwa_status_flags.argtypes = [vp, POINTER(c_uint32)]
    lib.pwa_profile_enable.argtypes = [vp, c_int32]
    lib.pwa_profile_read.argtypes = [vp, POINTER(c_double), POINTER(c_int64)]
    lib.pwa_kernel_launches.argtypes = [vp]
    lib.pwa_kernel_launches.restype = c_int64
    lib.pwa_bytes_per_eval.argtypes = [vp]
    lib.pwa_bytes_per_eval.restype = c_int64
    lib.pwa_kernel_variant.argtypes = [vp]
    lib.pwa_kernel_variant.restype = c_char_p
    lib.pwa_last_error.argtypes = [vp]
    lib.pwa_last_error.restype = c_char_p
    lib.pwa_version.argtypes = []
    lib.pwa_version.restype = c_char_p
    _LIB = lib
    return lib


def _check(status: int, h=None):
    if status != PWA_OK:
        raise PwaError(status, pwa_last_error(h))


def _ptr(t) -> Optional[int]:
    """Address of a torch tensor / numpy array / raw int, or None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _dev_f64(t, n, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
            and t.numel() >= n):
        raise TypeError(f"{name}: expected a contiguous CUDA float64 tensor with >= {n} elements")
    return t.data_ptr()


# ---- the C calls, one to one ------------------------------------------------------------------------------
def pwa_create(res_chan, data_mass, data_amp, data_weight, mc_mass, mc_amp, *, borrow: bool = False, device: int = 0,
               stream: int = 0, data_stride: int = 0, mc_stride: int = 0, n_data: Optional[int] = None,
               n_mc: Optional[int] = None, data_first: int = 0, mc_first: int = 0, rich: Optional[dict] = None) -> int:
    """Creates a handle from torch tensors (CPU or CUDA, float64, contiguous) in the layouts of pwa.h:
    mass [C][N], amp [R][H][N][2], weight [N] or None, res_chan [R] int32 (CPU).  Returns the handle.
    A window of a larger store (an event shard) is described without copying by `*_first` (first
    event), `n_*` (event count) and `*_stride` (events between planes of the full store).
    `rich` (pwa_create_rich, readings S21 / S22): dict with wave_res [R], ls_chan [L], and optionally ls_kind [L],
    ls_shape [L][6]; res_chan is then ignored (may be None)."""
    import torch
    lib = load()
    tensors = [data_mass, data_amp, mc_mass, mc_amp] + ([data_weight] if data_weight is not None else [])
    on_dev = {t.is_cuda for t in tensors}
    if len(on_dev) != 1:
        raise TypeError("all event buffers must live on the same side (host or device)")
    for t in tensors:
        if t.dtype != torch.float64 or not t.is_contiguous():
            raise TypeError("event buffers must be contiguous float64 tensors")
    rc = (res_chan if res_chan is not None else torch.zeros(int(mc_amp.shape[0]))).to(torch.int32).cpu().contiguous()
    R, H = int(mc_amp.shape[0]), int(mc_amp.shape[1])
    C = int(mc_mass.shape[0])
    d = pwa_model_desc()
    d.n_res, d.n_hel, d.n_chan = R, H, C
    d.res_chan = rc.data_ptr()
    if (data_first or n_data is not None) and not data_stride:
        data_stride = int(data_mass.shape[1])
    if (mc_first or n_mc is not None) and not mc_stride:
        mc_stride = int(mc_mass.shape[1])
    d.data = pwa_sample(int(data_mass.shape[1]) - data_first if n_data is None else n_data, data_stride,
                        data_mass.data_ptr() + 8 * data_first, data_amp.data_ptr() + 16 * data_first,
                        None if data_weight is None else data_weight.data_ptr() + 8 * data_first)
    d.mc = pwa_sample(int(mc_mass.shape[1]) - mc_first if n_mc is None else n_mc, mc_stride,
                      mc_mass.data_ptr() + 8 * mc_first, mc_amp.data_ptr() + 16 * mc_first, None)
    d.mem = PWA_MEM_DEVICE if on_dev.pop() else PWA_MEM_HOST
    d.borrow = 1 if borrow else 0
    d.device = device
    d.stream = stream or None
    out = c_void_p()
    if rich is None:
        _check(lib.pwa_create(byref(d), byref(out)))
        return out.value
    i32 = lambda x: torch.as_tensor(x).to(torch.int32).cpu().contiguous()
    wave_res, ls_chan = i32(rich["wave_res"]), i32(rich["ls_chan"])
    if wave_res.numel() != R:
        raise ValueError("rich['wave_res'] must have one entry per plane group (wave)")
    L = int(ls_chan.numel())
    kind = i32(rich["ls_kind"]) if rich.get("ls_kind") is not None else None
    shape = (torch.as_tensor(rich["ls_shape"], dtype=torch.float64).cpu().contiguous()
             if rich.get("ls_shape") is not None else None)
    if kind is not None and kind.numel() != L:
        raise ValueError("rich['ls_kind'] must have one entry per resonance")
    if shape is not None and tuple(shape.shape) != (L, 6):
        raise ValueError("rich['ls_shape'] must be [L][6]")
    rd = pwa_rich_desc(L, wave_res.data_ptr(), ls_chan.data_ptr(), None if kind is None else kind.data_ptr(),
                       None if shape is None else shape.data_ptr())
    _check(lib.pwa_create_rich(byref(d), byref(rd), byref(out)))
    return out.value


def pwa_create_rich(data_mass, data_amp, data_weight, mc_mass, mc_amp, rich: dict, **kw) -> int:
    """pwa_create_rich of include/pwa.h: the plane groups are partial waves, `rich` maps them onto resonances
    (wave_res, ls_chan, ls_kind, ls_shape); other keywords as pwa_create."""
    return pwa_create(None, data_mass, data_amp, data_weight, mc_mass, mc_amp, rich=rich, **kw)


def pwa_destroy(h) -> None:
    _check(load().pwa_destroy(h))


def pwa_n_params(h) -> int:
    return load().pwa_n_params(h)


def pwa_raw_size(h) -> int:
    return load().pwa_raw_size(h)


def pwa_nll(h, theta, nll) -> None:
    P = pwa_n_params(h)
    _check(load().pwa_nll(h, _dev_f64(theta, P, "theta"), _dev_f64(nll, 1, "nll")), h)


def pwa_nll_grad(h, theta, nll, grad) -> None:
    P = pwa_n_params(h)
    _check(load().pwa_nll_grad(h, _dev_f64(theta, P, "theta"), _dev_f64(nll, 1, "nll"), _dev_f64(grad, P, "grad")), h)


def pwa_hvp(h, theta, v, hv) -> None:
    P = pwa_n_params(h)
    _check(load().pwa_hvp(h, _dev_f64(theta, P, "theta"), _dev_f64(v, P, "v"), _dev_f64(hv, P, "hv")), h)


def pwa_nll_grad_hvp(h, theta, v, nll, grad, hv) -> None:
    P = pwa_n_params(h)
    _check(load().pwa_nll_grad_hvp(h, _dev_f64(theta, P, "theta"), _dev_f64(v, P, "v"), _dev_f64(nll, 1, "nll"),
                                   _dev_f64(grad, P, "grad"), _dev_f64(hv, P, "hv")), h)


def pwa_raw_sums(h, theta, v, raw) -> None:
    P = pwa_n_params(h)
    _check(load().pwa_raw_sums(h, _dev_f64(theta, P, "theta"), None if v is None else _dev_f64(v, P, "v"),
                               _dev_f64(raw, 4 + 4 * P, "raw")), h)


def pwa_combine(h, raw, v, nll, grad, hv) -> None:
    P = pwa_n_params(h)
    _check(load().pwa_combine(h, _dev_f64(raw, 4 + 4 * P, "raw"), None if v is None else _dev_f64(v, P, "v"),
                              None if nll is None else _dev_f64(nll, 1, "nll"),
                              None if grad is None else _dev_f64(grad, P, "grad"),
                              None if hv is None else _dev_f64(hv, P, "hv")), h)


def pwa_fit_opts_default() -> pwa_fit_opts:
    o = pwa_fit_opts()
    load().pwa_fit_opts_default(byref(o))
    return o


def pwa_fit_newton_cg(h, theta_inout, opts: Optional[pwa_fit_opts] = None) -> pwa_fit_result:
    """Runs the fit; returns the result struct (status PWA_ERR_NOT_CONVERGED / NONFINITE are reported in
    result.status, not raised); raises on argument or CUDA errors."""
    P = pwa_n_params(h)
    res = pwa_fit_result()
    st = load().pwa_fit_newton_cg(h, _dev_f64(theta_inout, P, "theta"), byref(opts) if opts is not None else None,
                                  byref(res))
    if st in (PWA_ERR_INVALID_ARG, PWA_ERR_CUDA, PWA_ERR_OOM):
        _check(st, h)
    return res


def pwa_nll_grad_hvp_host(h, theta_host, v_host, nll_host, grad_host, hv_host) -> None:
    """Host-buffer entry point: numpy float64 arrays (or CPU tensors); copies in, evaluates, copies out, syncs."""
    _check(load().pwa_nll_grad_hvp_host(h, _ptr(theta_host), _ptr(v_host), _ptr(nll_host), _ptr(grad_host),
                                        _ptr(hv_host)), h)


PWA_STATIC_MAX_RES = 64


def pwa_nll_grad_hvp_static(res_chan, data_mass, data_amp, data_weight, mc_mass, mc_amp, theta, v, nll, grad, hv, *,
                            device: int = 0, stream: int = 0) -> None:
    """pwa_nll_grad_hvp_static of include/pwa.h: the fused evaluation without a handle and without any device
    allocation (fixed scratch array inside the library; n_res <= PWA_STATIC_MAX_RES; calls that overlap on the GPU
    race).  Event buffers: contiguous CUDA float64 tensors in the layouts of pwa_create, read in place; res_chan [R]
    int32 on the CPU; theta, v, nll, grad, hv: CUDA float64 tensors (v, nll, grad, hv may each be None)."""
    import torch
    R, H, C = int(mc_amp.shape[0]), int(mc_amp.shape[1]), int(mc_mass.shape[0])
    for t in [data_mass, data_amp, mc_mass, mc_amp] + ([data_weight] if data_weight is not None else []):
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise TypeError("event buffers must be contiguous CUDA float64 tensors")
    rc = torch.as_tensor(res_chan).to(torch.int32).cpu().contiguous()
    if rc.numel() != R:
        raise ValueError("res_chan must have one entry per resonance")
    d = pwa_model_desc()
    d.n_res, d.n_hel, d.n_chan = R, H, C
    d.res_chan = rc.data_ptr()
    d.data = pwa_sample(int(data_mass.shape[1]), 0, data_mass.data_ptr(), data_amp.data_ptr(),
                        None if data_weight is None else data_weight.data_ptr())
    d.mc = pwa_sample(int(mc_mass.shape[1]), 0, mc_mass.data_ptr(), mc_amp.data_ptr(), None)
    d.mem, d.borrow, d.device, d.stream = PWA_MEM_DEVICE, 1, device, stream or None
    P = 4 * R
    opt = lambda t, n, name: None if t is None else _dev_f64(t, n, name)
    _check(load().pwa_nll_grad_hvp_static(byref(d), _dev_f64(theta, P, "theta"), opt(v, P, "v"), opt(nll, 1, "nll"),
                                          opt(grad, P, "grad"), opt(hv, P, "hv")))


def pwa_nll_grad_for_hvp(h, theta, nll, grad) -> None:
    P = pwa_n_params(h)
    _check(load().pwa_nll_grad_for_hvp(h, _dev_f64(theta, P, "theta"), _dev_f64(nll, 1, "nll"), _dev_f64(grad, P, "grad")), h)


def pwa_hvp_cached(h, v, hv) -> None:
    P = pwa_n_params(h)
    _check(load().pwa_hvp_cached(h, _dev_f64(v, P, "v"), _dev_f64(hv, P, "hv")), h)


def pwa_nll_batch(h, K: int, theta, nll) -> None:
    """nll[k] (device, K doubles) <- NLL(theta[k]) for the K parameter sets theta[K][P] (device), one pass per batch."""
    P = pwa_n_params(h)
    _check(load().pwa_nll_batch(h, K, _dev_f64(theta, K * P, "theta"), _dev_f64(nll, K, "nll")), h)


def pwa_hvp_cached_batch(h, K: int, v, hv) -> None:
    """hv[k] <- H(theta) v[k] for K directions v[K][P] at the theta of the last pwa_nll_grad_for_hvp call."""
    P = pwa_n_params(h)
    _check(load().pwa_hvp_cached_batch(h, K, _dev_f64(v, K * P, "v"), _dev_f64(hv, K * P, "hv")), h)


def pwa_hessian(h, theta, hess) -> None:
    """hess[P][P] (device) <- Hessian of the NLL at theta (device)."""
    P = pwa_n_params(h)
    _check(load().pwa_hessian(h, _dev_f64(theta, P, "theta"), _dev_f64(hess, P * P, "hess")), h)


def pwa_fit_fractions(h, theta, frac) -> None:
    """frac[n_res] (device) <- fit fractions over the MC sample at theta (device)."""
    P = pwa_n_params(h)
    _check(load().pwa_fit_fractions(h, _dev_f64(theta, P, "theta"), _dev_f64(frac, 1, "frac")), h)


def pwa_status_flags(h) -> int:
    f = c_uint32(0)
    _check(load().pwa_status_flags(h, byref(f)), h)
    return f.value


def pwa_profile_enable(h, on: bool) -> None:
    _check(load().pwa_profile_enable(h, 1 if on else 0), h)


def pwa_profile_read(h):
    """(summed sweep-kernel device time in ms, number of sweep launches) since the last read."""
    ms, n = c_double(0.0), c_int64(0)
    _check(load().pwa_profile_read(h, byref(ms), byref(n)), h)
    return ms.value, n.value


def pwa_kernel_launches(h) -> int:
    return load().pwa_kernel_launches(h)


def pwa_bytes_per_eval(h) -> int:
    return load().pwa_bytes_per_eval(h)


def pwa_kernel_variant(h) -> str:
    return load().pwa_kernel_variant(h).decode()


def pwa_last_error(h=None) -> str:
    return load().pwa_last_error(h).decode()


def pwa_version() -> str:
    return load().pwa_version().decode()


# ---- a small convenience wrapper (still marshalling only) ---------------------------------------------------
class Model:
    """Owns a handle and its output tensors.  `w` is a workloads.Workload (or any object with the same fields).
    With `stream` (a cudaStream_t) the handle enqueues there, and so does every torch operation of this class."""

    def __init__(self, w, device: int = 0, borrow: bool = False, stream: int = 0, rich: Optional[dict] = None):
        import contextlib
        import torch
        self.torch = torch
        self.dev = torch.device("cuda", device)
        self._keep = w if borrow else None
        self._ext = torch.cuda.ExternalStream(stream, device=self.dev) if stream else None
        self._on = (lambda: torch.cuda.stream(self._ext)) if stream else contextlib.nullcontext
        self.h = pwa_create(w.res_chan, w.data_mass, w.data_amp, w.data_weight, w.mc_mass, w.mc_amp, borrow=borrow,
                            device=device, stream=stream, rich=rich)
        self.P = pwa_n_params(self.h)
        self._keep_R = int(w.mc_amp.shape[0]) if rich is None else int(len(rich["ls_chan"]))  # fractions returned
        with self._on():
            self.nll_t = torch.zeros(1, dtype=torch.float64, device=self.dev)
            self.grad_t = torch.zeros(self.P, dtype=torch.float64, device=self.dev)
            self.hv_t = torch.zeros(self.P, dtype=torch.float64, device=self.dev)

    def _d(self, x):
        return self.torch.as_tensor(x, dtype=self.torch.float64).to(self.dev).contiguous()

    def nll(self, theta):
        with self._on():
            pwa_nll(self.h, self._d(theta), self.nll_t)
            return self.nll_t.item()

    def nll_grad(self, theta):
        with self._on():
            pwa_nll_grad(self.h, self._d(theta), self.nll_t, self.grad_t)
            return self.nll_t.item(), self.grad_t.cpu().numpy().copy()

    def hvp(self, theta, v):
        with self._on():
            pwa_hvp(self.h, self._d(theta), self._d(v), self.hv_t)
            return self.hv_t.cpu().numpy().copy()

    def nll_grad_hvp(self, theta, v):
        with self._on():
            pwa_nll_grad_hvp(self.h, self._d(theta), self._d(v), self.nll_t, self.grad_t, self.hv_t)
            return self.nll_t.item(), self.grad_t.cpu().numpy().copy(), self.hv_t.cpu().numpy().copy()

    def raw_sums(self, theta, v=None):
        with self._on():
            raw = self.torch.zeros(4 + 4 * self.P, dtype=self.torch.float64, device=self.dev)
            pwa_raw_sums(self.h, self._d(theta), None if v is None else self._d(v), raw)
            return raw

    def nll_grad_for_hvp(self, theta):
        with self._on():
            pwa_nll_grad_for_hvp(self.h, self._d(theta), self.nll_t, self.grad_t)
            return self.nll_t.item(), self.grad_t.cpu().numpy().copy()

    def hvp_cached(self, v):
        with self._on():
            pwa_hvp_cached(self.h, self._d(v), self.hv_t)
            return self.hv_t.cpu().numpy().copy()

    def nll_batch(self, thetas):
        with self._on():
            th = self._d(thetas)
            K = th.shape[0]
            out = self.torch.zeros(K, dtype=self.torch.float64, device=self.dev)
            pwa_nll_batch(self.h, K, th, out)
            return out.cpu().numpy()

    def hvp_cached_batch(self, vs):
        with self._on():
            v = self._d(vs)
            K = v.shape[0]
            out = self.torch.zeros(K, self.P, dtype=self.torch.float64, device=self.dev)
            pwa_hvp_cached_batch(self.h, K, v, out)
            return out.cpu().numpy()

    def hessian(self, theta):
        with self._on():
            out = self.torch.zeros(self.P, self.P, dtype=self.torch.float64, device=self.dev)
            pwa_hessian(self.h, self._d(theta), out)
            return out.cpu().numpy()

    def fit_fractions(self, theta):
        with self._on():
            frac = self.torch.zeros(int(self._keep_R), dtype=self.torch.float64, device=self.dev)
            pwa_fit_fractions(self.h, self._d(theta), frac)
            return frac.cpu().numpy()

    def fit(self, theta0, opts: Optional[pwa_fit_opts] = None):
        with self._on():
            th = self._d(theta0).clone()
            res = pwa_fit_newton_cg(self.h, th, opts)
            return th.cpu().numpy().copy(), res

    def close(self):
        if self.h:
            pwa_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
