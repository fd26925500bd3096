"""K evaluations per pass over the event store (include/pwa.h: pwa_nll_batch, pwa_hvp_cached_batch,
pwa_hessian) against the oracle: the oracle side is K plain calls of the existing oracle (no new arithmetic).
Tolerances are the north_star's: NLL 1e-10 relative, HVP 1e-8 relative L2 per set / direction."""
import numpy as np
import pytest
import torch

from helpers import rel_l2

pytestmark = pytest.mark.gpu

# (config index, n_mc, n_data): shapes with a batch kernel (2: rho 3 x 4 slices, 3: rho 4 x 8 slices, 6: R = 6) and
# one without (4: the 8-event-tile variant takes one pass per evaluation through the same entry points)
CASES = [(2, 20_011, 3_001), (3, 12_345, 1_537), (6, 30_001, 1_999), (4, 2_049, 517)]


@pytest.fixture(scope="module")
def pwa():
    import paper_2403_09225_b200 as p
    from paper_2403_09225_b200.build import build
    build()
    p.load()
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    return p


_CACHE = {}


def _case(pwa, oracle_mod, idx, n_mc, n_data):
    key = (idx, n_mc, n_data)
    if key not in _CACHE:
        import workloads
        cfg = workloads.CONFIGS[idx].scaled(n_mc, n_data)
        w = workloads.make_workload(cfg, "cpu", chunk=1 << 13)
        _CACHE[key] = (cfg, w, oracle_mod.model_from_workload(w), pwa.Model(w))
    return _CACHE[key]


@pytest.mark.parametrize("idx,n_mc,n_data", CASES)
@pytest.mark.parametrize("K", [1, 2, 4, 7])
def test_nll_batch_matches_oracle(pwa, oracle_mod, idx, n_mc, n_data, K):
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    thetas = np.stack([workloads.theta_true(cfg).numpy()] + [workloads.random_start(cfg, k).numpy() for k in range(K - 1)])
    l0 = pwa.pwa_kernel_launches(gm.h)
    got = gm.nll_batch(thetas)
    launches = pwa.pwa_kernel_launches(gm.h) - l0
    assert pwa.pwa_status_flags(gm.h) == 0
    for k in range(K):
        f0 = float(oracle_mod.nll(om, thetas[k], "ld"))
        assert abs(got[k] - f0) <= 1e-10 * max(1.0, abs(f0)), (idx, K, k, got[k], f0)
        assert abs(got[k] - gm.nll(thetas[k])) <= 1e-12 * max(1.0, abs(f0))   # same value as the single call, to rounding
    if idx != 4:  # passes: 4 + 2 + 1 -> (sweep + reduction) per group
        assert launches == 2 * {1: 1, 2: 1, 4: 1, 7: 3}[K]
    again = gm.nll_batch(thetas)
    assert again.tobytes() == got.tobytes()  # deterministic


@pytest.mark.parametrize("idx,n_mc,n_data", CASES)
@pytest.mark.parametrize("K", [2, 3, 5])
def test_hvp_cached_batch_matches_oracle(pwa, oracle_mod, idx, n_mc, n_data, K):
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    th = workloads.random_start(cfg, 1).numpy()
    vs = np.stack([workloads.direction(cfg, 10 + k).numpy() for k in range(K)])
    f, g = gm.nll_grad_for_hvp(th)
    got = gm.hvp_cached_batch(vs)
    assert pwa.pwa_status_flags(gm.h) == 0
    for k in range(K):
        _, _, h0 = oracle_mod.nll_grad_hvp(om, th, vs[k], "ld")
        assert rel_l2(got[k], h0) < 1e-8, (idx, K, k)
        assert rel_l2(got[k], gm.hvp_cached(vs[k])) < 1e-12
    again = gm.hvp_cached_batch(vs)
    assert again.tobytes() == got.tobytes()


def test_hvp_cached_batch_needs_a_keeping_call(pwa, oracle_mod):
    import workloads
    cfg, w, om, _ = _case(pwa, oracle_mod, *CASES[0])
    fresh = pwa.Model(w)
    with pytest.raises(pwa.PwaError):
        fresh.hvp_cached_batch(np.zeros((2, cfg.n_par)))
    with pytest.raises(pwa.PwaError):
        pwa.pwa_nll_batch(fresh.h, 0, fresh.grad_t, fresh.nll_t)
    fresh.close()


@pytest.mark.parametrize("idx,n_mc,n_data", [(1, 20_000, 4_000), CASES[0]])
def test_hessian_columns_are_oracle_hvps(pwa, oracle_mod, idx, n_mc, n_data):
    """pwa_hessian = P unit directions through the batched HVP: every column against the oracle's HVP with that unit
    vector, symmetry, and the gauge null vectors of the Hessian (pin P2: H 1_phi = 0, (H u)_a = -g_a)."""
    import workloads
    cfg, w, om, gm = _case(pwa, oracle_mod, idx, n_mc, n_data)
    th = workloads.random_start(cfg, 0).numpy()
    Hm = gm.hessian(th)
    P = cfg.n_par
    scale = np.abs(Hm).max()
    assert np.max(np.abs(Hm - Hm.T)) <= 1e-9 * scale
    for k in range(P):
        e = np.zeros(P); e[k] = 1.0
        _, _, h0 = oracle_mod.nll_grad_hvp(om, th, e, "ld")
        assert rel_l2(Hm[k], h0) < 1e-8, k
    ones_phi = np.zeros(P); ones_phi[1::4] = 1.0
    assert np.max(np.abs(Hm @ ones_phi)) <= 1e-8 * scale
    u = np.zeros(P); u[0::4] = th[0::4]
    _, g0, _ = oracle_mod.nll_grad_hvp(om, th, None, "ld")
    g0 = np.asarray(g0, dtype=np.float64)
    hu = Hm @ u
    assert np.max(np.abs(hu[0::4] + g0[0::4])) <= 1e-8 * max(scale, np.abs(g0).max())
