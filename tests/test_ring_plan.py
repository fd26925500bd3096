"""Host logic of the shared-memory ring (csrc/pwa_sweep_lanes.cu: producers_for, ring_stages), no GPU:
the invariants that make the parity waits on the ring's barriers safe.

  * a stage is always refilled by the same producer thread          <=>  the producer count divides the stage count
  * tiles that share a stage are consumed by the same warps in turn <=>  the stage count is a multiple of the number of
                                                                         tiles consumed at the same time (`group`)
The functions are internal C++ (namespace pwa), reached here through their mangled names in the shared library."""
import ctypes

import pytest


@pytest.fixture(scope="module")
def lib():
    import paper_2403_09225_b200 as p
    from paper_2403_09225_b200.build import build
    build()
    l = ctypes.CDLL(p.lib_path())
    l._ZN3pwa13producers_forEi.argtypes = [ctypes.c_int]
    l._ZN3pwa13producers_forEi.restype = ctypes.c_int
    l._ZN3pwa11ring_stagesEii.argtypes = [ctypes.c_int, ctypes.c_int]
    l._ZN3pwa11ring_stagesEii.restype = ctypes.c_int
    return l


def test_producer_count_divides_the_stage_count(lib, monkeypatch):
    monkeypatch.delenv("PWA_NPROD", raising=False)
    want = {1: 1, 2: 2, 3: 3, 4: 4, 5: 1, 6: 3, 7: 1, 8: 4, 9: 3, 12: 4}
    for stages, n in want.items():
        got = lib._ZN3pwa13producers_forEi(stages)
        assert got == n and stages % got == 0 and 1 <= got <= 4, (stages, got)
    for cap in (1, 2, 3):
        monkeypatch.setenv("PWA_NPROD", str(cap))
        for stages in range(1, 13):
            got = lib._ZN3pwa13producers_forEi(stages)
            assert 1 <= got <= cap and stages % got == 0, (cap, stages, got)
    monkeypatch.delenv("PWA_NPROD")


def test_ring_depth_is_a_multiple_of_the_tiles_consumed_together(lib, monkeypatch):
    monkeypatch.delenv("PWA_NPROD", raising=False)
    for group in (1, 2, 4):
        for fit in range(0, 33):
            s = lib._ZN3pwa11ring_stagesEii(fit, group)
            if fit < max(2, group):
                assert s == 0, (fit, group, s)  # the shape cannot run
                continue
            assert max(2, group) <= s <= fit and s % group == 0 and fit - s < 2 * group, (fit, group, s)
    # one stage less where that admits more producers
    assert lib._ZN3pwa11ring_stagesEii(5, 1) == 4 and lib._ZN3pwa11ring_stagesEii(7, 1) == 6
    assert lib._ZN3pwa11ring_stagesEii(8, 1) == 8 and lib._ZN3pwa11ring_stagesEii(6, 1) == 6 and lib._ZN3pwa11ring_stagesEii(3, 1) == 3
    assert lib._ZN3pwa11ring_stagesEii(6, 2) == 4 and lib._ZN3pwa11ring_stagesEii(8, 4) == 8 and lib._ZN3pwa11ring_stagesEii(7, 4) == 4
