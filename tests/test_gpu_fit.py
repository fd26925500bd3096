"""GPU fit (pwa_fit_newton_cg, a-8) against the reference fit oracle/fit.py (S15/S19).

The fit is an iteration whose end point is not unique (S14: global phase, common scale, local minima), so
raw theta is never compared.  What is unique and compared:
  * from the same start, with the same options, both sides run the same algorithm: the NLL reached agrees to
    1e-7 relative, the convergence classification is the same, and the sweep counts agree closely (rounding may
    shift a CG exit by an iteration);
  * at the point the CUDA fit returns, the ORACLE's gradient is small and its NLL equals the reported one
    (north_star tolerances): the result is checked by the oracle, not by the kernel that produced it;
  * the NLL never increased (Armijo) and the S19 box holds at the returned point; with a box that cuts the free
    minimum off both sides end on the same bounds with the same NLL (projected Newton-CG, S15');
  * fits run to their own stop from 12 random starts on both sides: same convergence class, same NLL where the
    trajectories stay together; starts that rounding sends to different basins are counted and bounded;
  * a start with a non-finite NLL (all couplings zero: ln 0) is reported as PWA_ERR_NONFINITE.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def setup(oracle_mod):
    import paper_2403_09225_b200 as pwa
    import workloads
    from paper_2403_09225_b200.build import build
    build()
    pwa.load()
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    out = {}
    for idx, n_mc, n_data in ((1, 20_000, 4_000), (2, 30_000, 3_000)):
        cfg = workloads.CONFIGS[idx].scaled(n_mc, n_data)
        w = workloads.make_workload(cfg, "cpu", chunk=1 << 13, imax_events=n_mc)
        out[idx] = (cfg, w, oracle_mod.model_from_workload(w), pwa.Model(w))
    return pwa, workloads, out


def _opts(pwa, **kw):
    o = pwa.pwa_fit_opts_default()
    for k, v in kw.items():
        setattr(o, k, v)
    return o


@pytest.mark.parametrize("idx", [1, 2])
def test_fit_from_theta_true_matches_the_reference_fit(oracle_mod, setup, idx):
    from oracle.fit import FitOpts, fit_newton_cg
    pwa, workloads, models = setup
    cfg, w, om, gm = models[idx]
    th0 = workloads.theta_true(cfg).numpy()
    ref = fit_newton_cg(om, th0, FitOpts(), prec="d", threads=oracle_mod.max_threads())
    th, res = gm.fit(th0)
    assert ref.converged and res.status == 0, (ref.stop_reason, res.stop_reason, res.status)
    assert res.stop_reason in (1, 2, 3)
    assert abs(res.nll - ref.nll) <= 1e-7 * max(1.0, abs(ref.nll)), (res.nll, ref.nll)
    assert abs(res.outer_iters - ref.outer_iters) <= max(2, ref.outer_iters // 5)
    assert abs(res.n_hvp - ref.n_hvp) <= max(5, ref.n_hvp // 4)
    # the oracle's verdict on the point the CUDA fit returned
    f0, g0, _ = oracle_mod.nll_grad_hvp(om, th, None, "ld")
    assert abs(float(f0) - res.nll) <= 1e-10 * max(1.0, abs(float(f0)))
    assert float(np.max(np.abs(np.asarray(g0, dtype=np.float64)))) <= max(10 * res.grad_inf_norm, 1e-3)
    assert res.nll < float(oracle_mod.nll(om, th0, "d"))
    o = FitOpts()
    assert np.all(th[3::4] >= o.gamma_min) and np.all(th[3::4] <= o.gamma_max)
    assert np.all(th[2::4] >= o.mass_min) and np.all(th[2::4] <= o.mass_max)
    assert res.n_grad >= res.outer_iters and res.n_hvp == res.cg_iters and res.seconds > 0.0


def test_fit_from_random_starts_follows_the_reference(oracle_mod, setup):
    """Random starts (S16) wander through many iterations; with a short budget both sides must have descended
    to nearly the same NLL, and the CUDA value must be the oracle's NLL at the returned point."""
    from oracle.fit import FitOpts, fit_newton_cg
    pwa, workloads, models = setup
    cfg, w, om, gm = models[1]
    for k in range(3):
        th0 = workloads.random_start(cfg, k).numpy()
        ref = fit_newton_cg(om, th0, FitOpts(max_outer=6), prec="d", threads=oracle_mod.max_threads())
        th, res = gm.fit(th0, _opts(pwa, max_outer=6))
        f_start = float(oracle_mod.nll(om, th0, "d"))
        assert res.nll <= f_start and ref.nll <= f_start
        assert abs(res.nll - ref.nll) <= 1e-6 * max(1.0, abs(ref.nll)), (k, res.nll, ref.nll)
        assert res.outer_iters == ref.outer_iters and res.stop_reason == ref.stop_reason
        f0 = float(oracle_mod.nll(om, th, "ld"))
        assert abs(f0 - res.nll) <= 1e-10 * max(1.0, abs(f0))


def test_active_bounds_match_the_reference_fit(oracle_mod, setup):
    """A box that cuts the unconstrained minimum off (widths capped below the fitted ones, a mass floor above a fitted
    mass): both sides must end on the same bounds, with the same NLL, and the oracle's projected gradient at the CUDA
    point must vanish while the frozen entries push outward (KKT)."""
    from oracle.fit import FitOpts, bounds, fit_newton_cg, projected_gradient
    pwa, workloads, models = setup
    cfg, w, om, gm = models[1]
    th0 = workloads.theta_true(cfg).numpy()
    th_free, r_free = gm.fit(th0)
    assert r_free.status == 0 and r_free.n_active == 0
    gmax, mmin = 0.8 * float(th_free[3::4].min()), float(th_free[2::4].min()) + 0.02
    ref = fit_newton_cg(om, th0, FitOpts(gamma_max=gmax, mass_min=mmin), prec="d", threads=oracle_mod.max_threads())
    th, res = gm.fit(th0, _opts(pwa, gamma_max=gmax, mass_min=mmin))
    assert ref.converged and res.status == 0 and res.n_active == ref.n_active >= 2
    assert abs(res.nll - ref.nll) <= 1e-7 * max(1.0, abs(ref.nll)) and res.nll > r_free.nll
    lo, hi = bounds(len(th), FitOpts(gamma_max=gmax, mass_min=mmin))
    assert np.all(th >= lo) and np.all(th <= hi)
    assert np.array_equal(th <= lo, np.asarray(ref.theta, dtype=np.float64) <= lo)
    assert np.array_equal(th >= hi, np.asarray(ref.theta, dtype=np.float64) >= hi)
    _, g0, _ = oracle_mod.nll_grad_hvp(om, th, None, "ld")
    g0 = np.asarray(g0, dtype=np.float64)
    gP, free = projected_gradient(th, g0, lo, hi)
    assert float(np.max(np.abs(gP))) <= max(10 * res.grad_inf_norm, 1e-3)
    assert np.all(g0[~free & (th <= lo)] > 0) and np.all(g0[~free & (th >= hi)] < 0)


def test_start_outside_the_box_is_projected(setup):
    pwa, workloads, models = setup
    cfg, w, om, gm = models[1]
    th0 = workloads.theta_true(cfg).numpy().copy()
    th0[3] = 5.0
    th0[6] = 0.01
    o = _opts(pwa, max_outer=0)
    th, res = gm.fit(th0, o)
    assert th[3] == o.gamma_max and th[6] == o.mass_min and res.stop_reason == 4
    want = th0.copy(); want[3] = o.gamma_max; want[6] = o.mass_min
    assert np.array_equal(th, want) and abs(res.nll - gm.nll(th)) <= 1e-13 * abs(res.nll)  # different kernel modes


@pytest.mark.parametrize("idx,n_starts", [(1, 8), (2, 4)])
def test_fits_to_completion_on_both_sides(oracle_mod, setup, idx, n_starts, capsys):
    """north_star: "Newton-CG fits reach the oracle's minimum".  Both sides run the SAME algorithm (S15') from the same
    random starts (S16) to their own stop.  Required of every start: the same convergence class, the CUDA value equal to
    the oracle's NLL at the CUDA point, and - where the CUDA fit converged - a vanishing oracle projected gradient
    there.  Where both converge the final NLLs agree to 1e-6 relative unless rounding has sent the two trajectories
    (100+ iterations through saddle regions) into different local minima, which PAPER.md:133 describes; those starts
    are printed.  On the config-1 shape (P = 8) they must stay a minority (measured: 0 of 8).  On the config-2 shape
    (P = 40 on 3 000 data events: dozens of local minima) the oracle's own end point changes with its OpenMP thread
    count (start 1: -1688.68 on 8 threads, -1692.18 on 16), so per-start agreement is not a property of either
    side there (measured: 1 of 4 agree); what is required is that every CUDA end point is a KKT point by the oracle."""
    from oracle.fit import FitOpts, bounds, fit_newton_cg, projected_gradient
    pwa, workloads, models = setup
    cfg, w, om, gm = models[idx]
    nt = oracle_mod.max_threads()
    lo, hi = bounds(cfg.n_par, FitOpts())
    same, different, rows = 0, [], []
    for k in range(n_starts):
        th0 = workloads.random_start(cfg, k).numpy()
        ref = fit_newton_cg(om, th0, FitOpts(), prec="d", threads=nt)
        th, res = gm.fit(th0)
        rows.append((k, ref.nll, ref.stop_reason, ref.converged, res.nll, res.stop_reason, res.status))
        assert (res.status == 0) == ref.converged, rows[-1]
        f0, g0, _ = oracle_mod.nll_grad_hvp(om, th, None, "d", threads=nt)
        assert abs(float(f0) - res.nll) <= 1e-10 * max(1.0, abs(float(f0)))
        assert np.all(th >= lo) and np.all(th <= hi)
        if res.status == 0:
            gP, _ = projected_gradient(th, np.asarray(g0, dtype=np.float64), lo, hi)
            assert float(np.max(np.abs(gP))) <= FitOpts().gconv
            if abs(res.nll - ref.nll) <= 1e-6 * max(1.0, abs(ref.nll)):
                same += 1
                assert res.stop_reason in (1, 2, 3) and ref.stop_reason in (1, 2, 3)
            else:
                different.append(k)
    with capsys.disabled():
        print(f"\nconfig-{idx} shape, {n_starts} random starts: {same} end at the reference fit's NLL, "
              f"different basins: {different}")
        for r in rows:
            print("  start %d: oracle nll %.6f stop %d conv %s | cuda nll %.6f stop %d status %d" % r)
    if idx == 1:
        assert len(different) <= n_starts // 2


def test_nonfinite_start_is_reported(setup):
    pwa, workloads, models = setup
    cfg, w, om, gm = models[1]
    th0 = workloads.theta_true(cfg).numpy().copy()
    th0[0::4] = 0.0  # all couplings zero: I = 0 on every event, ln I = -inf (S8)
    th, res = gm.fit(th0)
    assert res.status == 4  # PWA_ERR_NONFINITE, reported in the result, theta left at the start point
    assert np.array_equal(th, th0)
    assert pwa.pwa_status_flags(gm.h) & 1


def test_wall_time_cap_stops_the_fit(setup):
    """PAPER.md:135 ("early stopping"): max_seconds ends the fit at the next outer iteration with stop_reason 5."""
    pwa, workloads, models = setup
    cfg, w, om, gm = models[2]
    th0 = workloads.random_start(cfg, 0).numpy()
    th, res = gm.fit(th0, _opts(pwa, max_seconds=1e-7))
    assert res.stop_reason == 5 and res.status == 5 and res.outer_iters <= 1
    assert np.isfinite(res.nll) and res.nll <= gm.nll(th0) + 1e-9 * abs(res.nll)


def test_handles_on_their_own_streams_give_the_same_bits(setup):
    """Two fits in flight on two handles and streams over the same event store (bench.py --concurrent) must reproduce,
    bit for bit, what one handle on the default stream gives: nothing is shared between handles."""
    import concurrent.futures as cf
    pwa, workloads, models = setup
    cfg, w, om, gm = models[2]
    wd = type(w)(**{k: (v.cuda() if isinstance(v, torch.Tensor) and k != "res_chan" and k != "theta_true" else v)
                    for k, v in w.__dict__.items()})
    streams = [torch.cuda.Stream() for _ in range(2)]
    hs = [pwa.Model(wd, borrow=True, stream=s.cuda_stream) for s in streams]
    ref = pwa.Model(wd, borrow=True)
    try:
        starts = [workloads.random_start(cfg, k).numpy() for k in range(4)]
        o = _opts(pwa, max_outer=8)
        want = [ref.fit(s, o) for s in starts]
        with cf.ThreadPoolExecutor(max_workers=2) as ex:
            got = list(ex.map(lambda k: hs[k % 2].fit(starts[k], o), range(4)))
        for (th0, r0), (th1, r1) in zip(want, got):
            assert th0.tobytes() == th1.tobytes() and r0.nll == r1.nll and r0.n_hvp == r1.n_hvp
    finally:
        for x in hs + [ref]:
            x.close()
