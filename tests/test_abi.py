"""The C-ABI boundary without a GPU: libpwa_b200.so builds and loads, exports every function include/pwa.h
declares (and the binding lists the same names), the calls that need no device behave as documented, and the
product path fails loudly - never falls back to a CPU path - when no CUDA device is usable."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pwa():
    import paper_2403_09225_b200 as p
    from paper_2403_09225_b200.build import build
    build()
    p.load()
    return p


def _declared():
    src = open(os.path.join(ROOT, "include", "pwa.h")).read()
    src = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)
    names = re.findall(r"\b(pwa_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_header_symbols_are_exported_and_bound(pwa):
    declared = _declared()
    assert "pwa_create" in declared and "pwa_fit_newton_cg" in declared and len(declared) >= 20
    lib = ctypes.CDLL(pwa.lib_path())
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/pwa.h but not exported"
        assert hasattr(pwa, name), f"{name} has no Python binding of the same name"
    assert sorted(pwa.EXPORTS) == declared


def test_calls_that_need_no_device(pwa):
    assert pwa.pwa_version()
    o = pwa.pwa_fit_opts_default()
    assert (o.max_outer, o.max_cg, o.max_backtrack) == (500, 50, 40)
    assert (o.gtol, o.xtol, o.ftol, o.armijo_c1, o.backtrack) == (1e-5, 1e-8, 1e-12, 1e-4, 0.5)
    assert (o.gamma_min, o.gamma_max, o.mass_min, o.mass_max, o.gconv) == (5e-3, 2.0, 0.1, 4.0, 1.0)
    lib = pwa.load()
    assert lib.pwa_n_params(None) == -1 and lib.pwa_raw_size(None) == -1
    assert lib.pwa_destroy(None) == pwa.PWA_OK
    assert lib.pwa_nll(None, None, None) == pwa.PWA_ERR_INVALID_ARG


def _desc(pwa, R=2, H=2, C=1, n=8, **over):
    keep = {}
    keep["ch"] = np.zeros(R, dtype=np.int32)
    keep["mass"] = np.ones((C, n))
    keep["amp"] = np.ones((R, H, n, 2))
    d = pwa.pwa_model_desc()
    d.n_res, d.n_hel, d.n_chan = R, H, C
    d.res_chan = keep["ch"].ctypes.data
    for s in (d.data, d.mc):
        s.n_events, s.stride = n, 0
        s.mass = keep["mass"].ctypes.data
        s.amp = keep["amp"].ctypes.data
        s.weight = None
    d.mem, d.borrow, d.device, d.stream = pwa.PWA_MEM_HOST, 0, 0, None
    for k, v in over.items():
        setattr(d, k, v)
    return d, keep


@pytest.mark.parametrize("bad", [dict(n_res=0), dict(n_res=513), dict(n_hel=0), dict(n_hel=9), dict(n_chan=0),
                                 dict(n_chan=17), dict(borrow=1), dict(mem=7)])
def test_descriptor_validation_needs_no_device(pwa, bad):
    lib = pwa.load()
    d, keep = _desc(pwa, **bad)
    h = ctypes.c_void_p()
    assert lib.pwa_create(ctypes.byref(d), ctypes.byref(h)) == pwa.PWA_ERR_INVALID_ARG
    assert not h.value and pwa.pwa_last_error(None)


def test_no_device_means_a_loud_failure_not_a_cpu_path(pwa):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    lib = pwa.load()
    d, keep = _desc(pwa)
    h = ctypes.c_void_p()
    assert lib.pwa_create(ctypes.byref(d), ctypes.byref(h)) == pwa.PWA_ERR_CUDA
    assert not h.value and "CUDA" in pwa.pwa_last_error(None)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2403_09225_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "pwa_oracle" not in text, f
