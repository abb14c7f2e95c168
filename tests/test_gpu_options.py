"""GPU parity tests for the driver options added in round 2 (readings A21, A26-A28): the
flux-constrained projection, the Eq.25 minimum-error stop, the Gaussian-smoothed constant start, refresh_every and the
host-pointer OSEM entry points -- each against the CPU oracle on the same seeded inputs, through the C ABI."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402  (test infrastructure)
from paper_1210_2258_b200 import binding as B  # noqa: E402
from paper_1210_2258_b200 import synth  # noqa: E402

from test_gpu_parity import _need_gpu, dev, rel_l2, gpu_plan, oracle_opts, oracle_problem, run_both  # noqa: E402

SMALL = {
    "C0": lambda: synth.make("C0"),
    "C2": lambda: synth.make("C2", n=128),
    "C3": lambda: synth.make("C3", s=256, sbar=320, n_stars=150, max_iter=60, fwhm=64.0),
}


def oracle_run(w, alg="sgp", truth=None, **optkw):
    oo = oracle_opts(w, **optkw)
    P = oracle_problem(w, oo)
    ge = P.embed(w["g"]); be = [np.full((P.ny, P.nx), float(v)) for v in w["b"]]
    f, r = {"sgp": P.sgp, "rl": P.rl, "osem": P.osem}[alg](ge, be, opts=oo, truth=truth)
    return f, r, P


# ------------------------------------------------------------------------------------------------ flux-constrained projection
@pytest.mark.parametrize("dt,tol1,tol", [(np.float32, 1e-5, 1e-3), (np.float64, 1e-11, 1e-9)])
@pytest.mark.parametrize("cfg", ["C0", "C2", "C3"])
def test_flux_constrained_sgp(cfg, dt, tol1, tol):
    """Bonettini et al. 2009: projection on { f >= 0, sum_R f = c }.  One iteration at north_star's
    1e-5, 15 iterations over the un-branched stretch; sum_R f(k) = c to 1e-6 for every k tried; mu found by Newton steps on
    the device equals the oracle's exact (sorted) root through the iterate it produces."""
    _need_gpu()
    w = SMALL[cfg]()
    g = [dev(a, dt) for a in w["g"]]
    for iters, t in ((1, tol1), (15, tol)):
        plan, o = gpu_plan(w, dt, max_iter=iters, stop_rule=0, flux_constraint=1)
        fg, rg = plan.sgp(g, w["b"], opts=o)
        plan.close()
        fo, ro, P = oracle_run(w, max_iter=iters, stop_rule=0, flux_constraint=1)
        fg = fg.cpu().numpy()
        assert rg.iterations == ro.iterations == iters
        assert rel_l2(fg, fo) <= t, (cfg, iters, rel_l2(fg, fo))
        assert abs(rg.J0_final - ro.J0_final) <= (1e-5 if dt == np.float32 else 1e-11) * abs(ro.J0_final)
        c = max(0.0, sum(float((np.maximum(gj, 0) - bj).sum()) for gj, bj in zip(w["g"], w["b"])) / len(w["g"]))
        assert abs(fg.astype(np.float64).sum() - c) <= (1e-6 if dt == np.float64 else 2e-6) * c
        assert (fg >= 0).all()
    # a flux given by the caller
    plan, o = gpu_plan(w, dt, max_iter=5, stop_rule=0, flux_constraint=1, flux_value=1e6)
    fg, rg = plan.sgp(g, w["b"], opts=o)
    plan.close()
    assert abs(fg.double().sum().item() - 1e6) <= 2e-6 * 1e6
    fo, ro, P = oracle_run(w, max_iter=5, stop_rule=0, flux_constraint=1, flux_value=1e6)
    assert rel_l2(fg.cpu().numpy(), fo) <= tol


# ------------------------------------------------------------------------------------------------ Eq.25
@pytest.mark.parametrize("dt", [np.float32, np.float64])
@pytest.mark.parametrize("alg", ["sgp", "rl"])
def test_minimum_error_stop_eq25(alg, dt):
    """Eq.25 on the device: the error trace rho(k) against the oracle's, the stop at the first k whose
    next step would increase rho, and the iterate returned = f(k) of the run stopped there by max_iter"""
    _need_gpu()
    w = synth.make("C1", n=256, max_iter=300, stop_rule=0)
    # few counts (the object dimmed 300 times, Poisson noise drawn again): semiconvergence within a few dozen iterations
    rng = np.random.default_rng(25)
    truth = w["truth"] / 300.0
    K = np.fft.rfft2(np.fft.ifftshift(w["psf"][0]))
    w["g"] = [rng.poisson(np.maximum(np.fft.irfft2(K * np.fft.rfft2(truth), s=truth.shape) + w["b"][0], 0)).astype(np.float64)]
    w["name"] += "_dim"
    K = 300
    fo, ro, P = oracle_run(w, alg, truth=truth, max_iter=K, stop_rule=oracle.STOP_MINERR)
    assert ro.stop_reason == 4, "the oracle run must stop by Eq.25 for this test to mean anything"
    plan, o = gpu_plan(w, dt, max_iter=K, stop_rule=B.STOP_MINERR)
    g = [dev(a, dt) for a in w["g"]]
    run = plan.sgp if alg == "sgp" else plan.rl
    fg, rg = run(g, w["b"], opts=o, truth=dev(truth, dt))
    assert rg.stop_reason == 4 and abs(rg.iterations - ro.iterations) <= 1
    n = min(rg.iterations, ro.iterations)
    np.testing.assert_allclose(rg.err[:n + 1], ro.err[:n + 1], rtol=2e-4 if dt == np.float32 else 1e-9)
    assert abs(rg.err_final - ro.err_final) <= (1e-4 if dt == np.float32 else 1e-9) * ro.err_final
    assert rg.err[rg.iterations + 1] > rg.err[rg.iterations] == rg.err_final           # the discarded step would have increased it
    # the iterate returned is f(k), not the discarded f(k+1)
    o2 = B.default_options(**{**w["opts"], "max_iter": rg.iterations, "stop_rule": 0})
    fk, rk = run(g, w["b"], opts=o2, truth=dev(truth, dt))       # with the true object given both runs take the launch-per-pass path (small grids: csrc/small.cuh)
    assert torch.equal(fk, fg) and rk.J0_final == rg.J0_final
    if rg.iterations == ro.iterations:
        assert rel_l2(fg.cpu().numpy(), fo) <= (1e-3 if dt == np.float32 else 1e-8)
    # error trace without the stopping rule; the rule without a true object is refused
    f3, r3 = run(g, w["b"], opts=B.default_options(**{**w["opts"], "max_iter": 10, "stop_rule": 0}), truth=dev(truth, dt))
    np.testing.assert_allclose(r3.err[:11], ro.err[:11], rtol=2e-4 if dt == np.float32 else 1e-9)
    _, r4 = run(g, w["b"], opts=o, check=False)
    assert r4.rc == B.ERR_ARG
    plan.close()


@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_minimum_error_stop_eq25_osem(dt):
    """Eq.25 for OSEM on the device, per cycle (reading A27; the paper stops OSEM at the minimum r.m.s. error in its
    diffuse-object experiments): the error trace against the oracle's, the stop at the first cycle that would
    increase rho, the iterate returned = h(k) of the run stopped there by max_iter (bit for bit), J0 at that iterate."""
    _need_gpu()
    w = synth.make("C2", n=128)
    # few counts (the object dimmed 3000 times, Poisson noise drawn again): semiconvergence after 16 cycles
    rng = np.random.default_rng(26)
    truth = w["truth"] / 3000.0
    g = []
    for j, k in enumerate(w["psf"]):
        K = np.fft.rfft2(np.fft.ifftshift(k / k.sum()))
        g.append(rng.poisson(np.maximum(np.fft.irfft2(K * np.fft.rfft2(truth), s=truth.shape) + w["b"][j], 0)).astype(np.float64))
    w["g"] = g
    w["name"] += "_dim"
    K = 60
    fo, ro, P = oracle_run(w, "osem", truth=truth, max_iter=K, stop_rule=oracle.STOP_MINERR)
    assert ro.stop_reason == 4 and 3 < ro.iterations < K, "the oracle run must stop by Eq.25 for this test to mean anything"
    plan, o = gpu_plan(w, dt, max_iter=K, stop_rule=B.STOP_MINERR)
    gd = [dev(a, dt) for a in w["g"]]
    fg, rg = plan.osem(gd, w["b"], opts=o, truth=dev(truth, dt))
    assert rg.stop_reason == 4 and rg.iterations == ro.iterations, (rg.stop_reason, rg.iterations, ro.iterations)
    n = rg.iterations
    np.testing.assert_allclose(rg.err[:n + 2], ro.err[:n + 2], rtol=1e-5 if dt == np.float32 else 1e-11)
    assert rg.err[n + 1] > rg.err[n] == rg.err_final                      # the discarded cycle would have increased it
    assert abs(rg.J0_final - ro.J0_final) <= (1e-4 if dt == np.float32 else 1e-10) * abs(ro.J0_final)
    assert rel_l2(fg.cpu().numpy(), fo) <= (1e-4 if dt == np.float32 else 1e-10)
    assert rg.n_fft2 == ro.n_fft2 == 4 * len(g) * (rg.iterations + 1), (rg.n_fft2, ro.n_fft2)      # the discarded cycle was computed too
    # the iterate returned is h(k), not the discarded h(k+1)
    o2 = B.default_options(**{**w["opts"], "max_iter": n, "stop_rule": 0})
    fk, rk = plan.osem(gd, w["b"], opts=o2)
    assert torch.equal(fk, fg) and rk.J0_final == rg.J0_final and rk.iterations == n
    # the error trace without the stopping rule; the rule without a true object is refused
    f3, r3 = plan.osem(gd, w["b"], opts=B.default_options(**{**w["opts"], "max_iter": 8, "stop_rule": 0}), truth=dev(truth, dt))
    np.testing.assert_allclose(r3.err[:9], ro.err[:9], rtol=1e-5 if dt == np.float32 else 1e-11)
    assert r3.iterations == 8 and r3.stop_reason == 1
    _, r4 = plan.osem(gd, w["b"], opts=o, check=False)
    assert r4.rc == B.ERR_ARG
    plan.close()


# ------------------------------------------------------------------------------------------------ smoothed constant start
@pytest.mark.parametrize("dt,tol", [(np.float32, 2e-6), (np.float64, 1e-12)])
def test_gaussian_smoothed_constant_start(dt, tol):
    """PAPER.md:264 / reading A28: f(0) = M_R o max(0, G_sigma * (c M_R)) against the oracle (max_iter = 0 returns f(0)), then
    10 iterations from it; without boundary correction the smoothed constant is the constant"""
    _need_gpu()
    w = SMALL["C3"]()
    g = [dev(a, dt) for a in w["g"]]
    for sig in (2.0, 5.5):
        plan, o = gpu_plan(w, dt, max_iter=0, init=B.INIT_CONST_SMOOTH, init_sigma=sig)
        f0g, r0 = plan.sgp(g, w["b"], opts=o)
        fo0, ro0, P = oracle_run(w, max_iter=0, init=oracle.INIT_CONST_SMOOTH, init_sigma=sig)
        MR = P.info()["MR"]
        f0g = f0g.cpu().numpy()
        assert np.abs(f0g - fo0).max() <= tol * fo0.max() and (f0g[MR == 0] == 0).all() and (f0g >= 0).all()
        assert abs(r0.J0_final - ro0.J0_final) <= (1e-6 if dt == np.float32 else 1e-12) * ro0.J0_final
        o10 = B.default_options(**{**w["opts"], "max_iter": 10, "stop_rule": 0, "init": B.INIT_CONST_SMOOTH, "init_sigma": sig})
        fg, rg = plan.sgp(g, w["b"], opts=o10)
        fo, ro, _ = oracle_run(w, max_iter=10, stop_rule=0, init=oracle.INIT_CONST_SMOOTH, init_sigma=sig)
        assert rel_l2(fg.cpu().numpy(), fo) <= (1e-4 if dt == np.float32 else 1e-10)
        plan.close()
    w = SMALL["C0"]()
    pa, oa = gpu_plan(w, dt, max_iter=3, init=B.INIT_CONST_SMOOTH)
    pb, ob = gpu_plan(w, dt, max_iter=3, init=B.INIT_CONST)
    g = [dev(a, dt) for a in w["g"]]
    assert torch.equal(pa.sgp(g, w["b"], opts=oa)[0], pb.sgp(g, w["b"], opts=ob)[0])
    pa.close(); pb.close()


# ------------------------------------------------------------------------------------------------ refresh_every (reading A21)
@pytest.mark.parametrize("dt,tol", [(np.float32, 1e-3), (np.float64, 1e-10)])
@pytest.mark.parametrize("cfg,fuse", [("C0", 4), ("C0", 8), ("C2", 8), ("C3", 4)])
def test_refresh_every(cfg, fuse, dt, tol):
    """A_j f and J0 recomputed from f after every n-th iteration (separate and fused line-search schedules): parity with the
    oracle's branch over the un-branched stretch, p + 1 transforms more per refresh, and J0 at the refreshed iterations
    equal to the objective evaluated from the returned image itself"""
    _need_gpu()
    w = SMALL[cfg]()
    p = len(w["g"])
    g = [dev(a, dt) for a in w["g"]]
    iters, every = 20, 5
    plan, o = gpu_plan(w, dt, max_iter=iters, stop_rule=0, refresh_every=every, use_graph=1 | fuse)
    fg, rg = plan.sgp(g, w["b"], opts=o)
    plan.close()
    fo, ro, P = oracle_run(w, max_iter=iters, stop_rule=0, refresh_every=every)
    assert rg.iterations == ro.iterations == iters
    assert rg.n_fft2 == ro.n_fft2 == iters * (2 * p + 2) + (iters // every) * (p + 1)
    assert rel_l2(fg.cpu().numpy(), fo) <= tol
    np.testing.assert_allclose(rg.J, ro.J, rtol=1e-4 if dt == np.float32 else 1e-11)
    ge = P.embed(w["g"]); be = [np.full((P.ny, P.nx), float(v)) for v in w["b"]]
    Jf = P.J0_of_f(fg.cpu().numpy().astype(np.float64), ge, be)          # iteration 20 is a refreshed one
    assert abs(rg.J0_final - Jf) <= (2e-6 if dt == np.float32 else 1e-12) * Jf
    # refresh after every iteration, with a stopping rule that must now be evaluated by the refresh kernel
    plan, o = gpu_plan(w, dt, max_iter=200, stop_rule=1, tol=1e-3, refresh_every=1, use_graph=1 | fuse)
    fg, rg = plan.sgp(g, w["b"], opts=o)
    plan.close()
    fo, ro, P = oracle_run(w, max_iter=200, stop_rule=1, tol=1e-3, refresh_every=1)
    assert rg.stop_reason == ro.stop_reason == 2 and abs(rg.iterations - ro.iterations) <= 1


# ------------------------------------------------------------------------------------------------ OSEM through host pointers
def test_osem_host_entry_points():
    _need_gpu()
    w = synth.make("C2", n=128)
    o = B.default_options(**{**w["opts"], "max_iter": 6, "stop_rule": 0})
    g32 = [a.astype(np.float32) for a in w["g"]]; k32 = [a.astype(np.float32) for a in w["psf"]]
    fh, rh = B.osem_multi(g32, k32, w["b"], opts=o, host=True)
    fd, rd = B.osem_multi([dev(a, np.float32) for a in g32], [dev(a, np.float32) for a in k32], w["b"], opts=o)
    assert np.array_equal(fh, fd.cpu().numpy()) and rh.iterations == rd.iterations == 6 and rh.J0_final == rd.J0_final
    w = synth.make("C3", s=64, sbar=128, n_stars=30, max_iter=5, fwhm=8.0)
    o = B.default_options(**{**w["opts"], "stop_rule": 0})
    g32 = [a.astype(np.float32) for a in w["g"]]; k32 = [a.astype(np.float32) for a in w["psf"]]
    oy, ox, sy, sx = w["S"]
    fh, rh = B.osem_boundary(g32, k32, w["b"], oy, ox, opts=o, host=True)
    fo, ro = oracle.osem_boundary(w["g"], w["psf"], w["b"], oy, ox, opts=oracle.default_options(**{**w["opts"], "stop_rule": 0}))
    assert rh.iterations == 5 and rel_l2(fh, fo) <= 1e-4 and (fh[rh.maskR == 0] == 0).all()


# ------------------------------------------------------------------------------------------------ workspace estimate
@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_workspace_estimate_bounds_what_a_plan_allocates(dt):
    """sgp_workspace_bytes is an upper bound of what sgp_plan_create allocates, and a tight one (within 2 %) at the large sizes"""
    _need_gpu()
    import ctypes as C
    L = B.lib()
    L.sgp_workspace_bytes.restype = C.c_size_t
    L.sgp_workspace_bytes.argtypes = [C.c_int] * 5
    code = B.F32 if dt == np.float32 else B.F64
    for (ny, nx, p, S) in [(64, 64, 1, None), (256, 256, 1, None), (128, 320, 3, None), (320, 256, 2, (50, 10, 200, 232)), (1000, 400, 1, None),
                           (2048, 2048, 1, None), (2048, 2048, 3, None), (1280, 1280, 1, (128, 128, 1024, 1024))]:
        psf = synth.psf_gaussian(ny, nx, 2.0)
        plan = B.Plan([dev(psf, dt)] * p, S=S)
        kind = B.KIND_BOUNDARY if S is not None else (B.KIND_SINGLE if p == 1 else B.KIND_MULTI)
        est, got = L.sgp_workspace_bytes(kind, p, ny, nx, code), plan.workspace_bytes()
        plan.close()
        assert got <= est, (ny, nx, p, S, got, est)
        if ny * nx >= 2048 * 2048:
            assert est <= 1.02 * got
