"""GPU parity tests for the one-cluster-per-problem SGP kernel of the small grids (csrc/small.cuh; SURVEY.md 8(f) item 2,
"small grids"): the whole of Algorithm 1 inside one kernel, the transposes of the 2-D transforms through
distributed shared memory.  Every run is checked against the fp64 oracle at north_star's tolerances (1e-5 after one iteration,
1e-3 / 1e-10 over the un-branched stretch, identical rule / backtrack traces, same stopping iteration) and against the
launch-per-pass path (`use_graph` bit 7), which evaluates the same formulas with another grouping of the sums."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402  (test infrastructure)
from paper_1210_2258_b200 import binding as B  # noqa: E402
from paper_1210_2258_b200 import synth  # noqa: E402

from test_gpu_parity import _need_gpu, dev, rel_l2, oracle_run  # noqa: E402

NO_CLUSTER = 128          # use_graph bit 7 (include/sgp.h)
TOL = {np.float32: dict(one=1e-5, run=1e-3, J=1e-4, alpha=5e-3, pix=1e-3), np.float64: dict(one=1e-11, run=1e-10, J=1e-10, alpha=1e-9, pix=1e-10)}


def _oracle(w, n, **kw):
    P = oracle.Problem(w["psf"])
    return P.sgp(w["g"], [np.full((n, n), float(w["b"][0]))], opts=oracle.default_options(**kw))


def _gpu(w, dt, use_graph=1, **kw):
    o = B.default_options(**{**kw, "use_graph": use_graph})
    plan = B.Plan([dev(w["psf"][0], dt)], opts=o)
    f, r = plan.sgp([dev(w["g"][0], dt)], w["b"], opts=o)
    plan.close()
    return f.cpu().numpy(), r


@pytest.mark.parametrize("dt", [np.float32, np.float64])
@pytest.mark.parametrize("n", [128, 256])
def test_cluster_kernel_matches_the_oracle(n, dt):
    """C0 recipe (BASELINE.json configs[0]; 256^2 is its stated size): one iteration at 1e-5 / 1e-11; 15 iterations (C0 runs with
    D = f and BB steps of 1e2 ... 1e4: in float the J0 trace of ANY evaluation leaves 1e-4 of the fp64 sequence after 20-45
    iterations, sooner on the smaller grid): image, per-pixel bound, whole J0 trace, step lengths, identical rule
    and backtrack traces, the same count of 2-D transforms (2p + 2 per iteration)"""
    _need_gpu()
    t = TOL[dt]
    w = synth.make("C0", n=n)
    for it in (1, 15):
        kw = {**w["opts"], "max_iter": it, "stop_rule": 0}
        fo, ro = _oracle(w, n, **kw)
        fg, rg = _gpu(w, dt, **kw)
        assert rg.fused_linesearch == 2, "this geometry must run through the cluster kernel"
        assert rg.iterations == ro.iterations == it and rg.n_fft2 == ro.n_fft2 == 4 * it
        e = rel_l2(fg, fo)
        print(f"[measured] cluster_{n} {np.dtype(dt).name} rel_l2_{it}it = {e:.3e}")
        assert e <= (t["one"] if it == 1 else t["run"])
        assert np.max(np.abs(fg - fo)) <= t["pix"] * np.max(fo)
        assert np.all(fg >= 0)
        assert np.max(np.abs(rg.J - ro.J) / np.abs(ro.J)) <= t["J"]
        assert np.array_equal(rg.rule, ro.rule) and np.array_equal(rg.backtracks, ro.backtracks)
        assert np.max(np.abs(rg.alpha - ro.alpha) / np.abs(ro.alpha)) <= t["alpha"]
        assert np.array_equal(rg.lam, ro.lam)


@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_cluster_kernel_backtracks_like_the_oracle(dt):
    """alpha0 = 1e5, alpha_min = 1e3: lambda = 1 overshoots in every iteration, so every iteration runs the Armijo loop
     inside the kernel -- one reduction per trial, q, u, g in registers.  Backtrack counts and accepted
    lambdas equal the oracle's; image and J0 at the tolerance of an un-branched run"""
    _need_gpu()
    n = 256
    t = TOL[dt]
    w = synth.make("C0", n=n)
    kw = {**w["opts"], "alpha0": 1e5, "alpha_min": 1e3, "alpha_max": 1e6, "max_iter": 10, "stop_rule": 0}
    fo, ro = _oracle(w, n, **kw)
    fg, rg = _gpu(w, dt, **kw)
    assert rg.fused_linesearch == 2 and ro.total_backtracks >= 10
    assert np.array_equal(rg.backtracks, ro.backtracks) and np.array_equal(rg.lam, ro.lam) and rg.total_backtracks == ro.total_backtracks
    # (J0 jumps between 3e5 and 1.7e6 along this run: its trace is held to the tolerance of the image, not to 1e-4)
    assert rel_l2(fg, fo) <= t["run"] and np.max(np.abs(rg.J - ro.J) / np.abs(ro.J)) <= t["run"]
    # the Armijo bound holds for every accepted step (Alg.1 step 5), whatever the rounding
    Jref = np.array([max(rg.J[max(0, k - int(kw["armijo_memory"]) + 1): k + 1]) for k in range(rg.iterations)])
    assert np.all(rg.J[1:] <= Jref * (1 + 1e-6))


def test_cluster_kernel_gives_up_like_the_launch_per_pass_path():
    """A16: with max_backtracks = 1 and an overshooting first step the line search fails; both paths report the same status and
    leave the same iterate"""
    _need_gpu()
    w = synth.make("C0", n=128)
    kw = {**w["opts"], "alpha0": 1e7, "alpha_min": 1e6, "alpha_max": 1e8, "max_iter": 5, "stop_rule": 0, "max_backtracks": 1}
    out = []
    for ug in (1, 1 | NO_CLUSTER):
        try:
            f, r = _gpu(w, np.float64, use_graph=ug, **kw)
            out.append(("ok", r.rc, r.iterations, f))
        except Exception as e:      # the binding raises on a negative status
            out.append(("raised", type(e).__name__, str(e)[:60], None))
    assert out[0][:3] == out[1][:3], (out[0][:3], out[1][:3])
    if out[0][0] == "ok":
        assert np.allclose(out[0][3], out[1][3], rtol=1e-12, atol=0)


@pytest.mark.parametrize("dt", [np.float32, np.float64])
@pytest.mark.parametrize("rule", ["relj", "disc"])
def test_cluster_kernel_stops_where_the_oracle_stops(rule, dt):
    """Eq.24 (relative change of J0) and Eq.26 (discrepancy; the threshold is the oracle's D(18), so that the rule fires inside
    the un-branched stretch): the kernel tests the rules itself and leaves at the same iteration as the oracle (fp32: +-1)"""
    _need_gpu()
    n = 256
    w = synth.make("C0", n=n)
    if rule == "relj":
        kw = {**w["opts"], "max_iter": 300, "stop_rule": 1, "tol": 3e-3}
    else:
        _, r18 = _oracle(w, n, **{**w["opts"], "max_iter": 18, "stop_rule": 0})
        kw = {**w["opts"], "max_iter": 300, "stop_rule": 2, "disc_threshold": float(2.0 * r18.J0_final / (n * n))}
    fo, ro = _oracle(w, n, **kw)
    fg, rg = _gpu(w, dt, **kw)
    assert rg.fused_linesearch == 2 and 0 < ro.iterations < 300
    assert rg.stop_reason == ro.stop_reason
    assert abs(rg.iterations - ro.iterations) <= (1 if dt == np.float32 else 0)
    if rg.iterations == ro.iterations:
        assert rel_l2(fg, fo) <= (3e-3 if dt == np.float32 else 1e-9)


@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_cluster_kernel_C1_recipe_to_its_discrepancy_stop(dt):
    """C1 recipe (galaxies + stars, Airy PSF, b = 20) at 256^2 with the paper's default options: adaptive bounds (L1, L2) from one
    RL step, monotone Armijo rule, discrepancy stop (Eq.26) -- same bounds, same stopping iteration, image and
    J0 trace at north_star's tolerances"""
    _need_gpu()
    n = 256
    t = TOL[dt]
    w = synth.make("C1", n=n)
    kw = dict(w["opts"])
    fo, ro = _oracle(w, n, **kw)
    fg, rg = _gpu(w, dt, **kw)
    assert rg.fused_linesearch == 2 and ro.stop_reason == 3 and 0 < ro.iterations < kw["max_iter"]
    assert rg.stop_reason == ro.stop_reason and rg.iterations == ro.iterations
    lt = 1e-4 if dt == np.float32 else 1e-10      # the bounds are the extreme values of one RL step, taken in the working precision
    assert abs(rg.L1_used - ro.L1_used) <= lt * ro.L1_used and abs(rg.L2_used - ro.L2_used) <= lt * ro.L2_used
    e = rel_l2(fg, fo)
    print(f"[measured] cluster_C1_256 {np.dtype(dt).name} rel_l2_{ro.iterations}it = {e:.3e}")
    # J0 trace in float: the oracle's own float build is 2.5e-4 off its double build on this recipe (at the steep 5th step)
    assert e <= t["run"] and np.max(np.abs(rg.J - ro.J) / np.abs(ro.J)) <= (1e-3 if dt == np.float32 else t["J"])
    assert abs(rg.J0_final - ro.J0_final) <= t["J"] * ro.J0_final
    assert np.array_equal(rg.rule, ro.rule) and np.array_equal(rg.backtracks, ro.backtracks)


@pytest.mark.parametrize("dt,tol", [(np.float32, 2e-5), (np.float64, 1e-12)])
def test_cluster_kernel_and_launch_per_pass_path_agree(dt, tol):
    """The same problem through both paths: same formulas, other grouping of the global sums -- rounding-level agreement over 12
    iterations, identical branches; max_iter = 0 returns the start point in both"""
    _need_gpu()
    n = 256
    w = synth.make("C0", n=n)
    kw = {**w["opts"], "max_iter": 12, "stop_rule": 0}
    fc, rc_ = _gpu(w, dt, use_graph=1, **kw)
    fp, rp = _gpu(w, dt, use_graph=1 | NO_CLUSTER, **kw)
    assert rc_.fused_linesearch == 2 and rp.fused_linesearch != 2
    assert rel_l2(fc, fp) <= tol and np.array_equal(rc_.rule, rp.rule) and np.array_equal(rc_.backtracks, rp.backtracks)
    assert rc_.n_fft2 == rp.n_fft2 and rc_.kernel_launches < rp.kernel_launches
    kw0 = {**w["opts"], "max_iter": 0, "stop_rule": 0}
    f0c, r0c = _gpu(w, dt, use_graph=1, **kw0)
    f0p, r0p = _gpu(w, dt, use_graph=1 | NO_CLUSTER, **kw0)
    assert np.array_equal(f0c, f0p) and r0c.iterations == r0p.iterations == 0 and r0c.J0_final == r0p.J0_final


def test_cluster_kernel_in_batched_plans():
    """A batched plan runs one cluster per problem up to 32 problems of 256^2: 6 problems of 256^2 each equal --
    bit for bit -- the same problem run alone (every problem is summed by its own cluster in the same order), with different
    backgrounds and stopping iterations; 12 problems run in the two-CTAs-per-SM form of the kernel; 40 problems take the launch-per-pass
    path and match the oracle all the same"""
    _need_gpu()
    n, dt = 256, np.float32
    ws = [synth.make("C0", n=n, seed_idx=60 + i) for i in range(40)]
    psf = ws[0]["psf"]
    kw = {**ws[0]["opts"], "max_iter": 200, "stop_rule": 1, "tol": 2e-3}
    o = B.default_options(**kw)
    nb = 6
    g = [[dev(w["g"][0], dt)] for w in ws[:nb]]
    b = [[10.0 + i] for i in range(nb)]
    bp = B.BatchedPlan(nb, [dev(psf[0], dt)], opts=o)
    fb, rb = bp.run_batched(B.ALG_SGP, g, b, opts=o)
    bp.close()
    single = B.Plan([dev(psf[0], dt)], opts=o)
    for i in range(nb):
        fs, rs = single.run(B.ALG_SGP, g[i], b[i], opts=o)
        assert rb[i].fused_linesearch == 2 and rs.fused_linesearch == 2
        assert torch.equal(fb[i], fs) and rb[i].iterations == rs.iterations and np.array_equal(rb[i].J, rs.J)
    single.close()
    assert len({r.iterations for r in rb}) > 1
    # 12 problems: more than the device holds clusters of the one-CTA-per-SM form, so the two-CTAs-per-SM form runs them
    nb2 = 12
    g = [[dev(w["g"][0], dt)] for w in ws[:nb2]]
    for it, tol in ((1, 1e-5), (12, 1e-3)):
        oi = B.default_options(**{**ws[0]["opts"], "max_iter": it, "stop_rule": 0})
        bp = B.BatchedPlan(nb2, [dev(psf[0], dt)], opts=oi)
        fb, rb = bp.run_batched(B.ALG_SGP, g, [[10.0]] * nb2, opts=oi)
        bp.close()
        assert all(r.fused_linesearch == 2 for r in rb)
        for i in (0, 5, 11):
            fo, ro = _oracle(ws[i], n, **{**ws[0]["opts"], "max_iter": it, "stop_rule": 0})
            assert rel_l2(fb[i].cpu().numpy(), fo) <= tol and np.array_equal(rb[i].rule, ro.rule) and np.array_equal(rb[i].backtracks, ro.backtracks)
    # many problems: launch-per-pass
    o1 = B.default_options(**{**ws[0]["opts"], "max_iter": 1, "stop_rule": 0})
    g = [[dev(w["g"][0], dt)] for w in ws]
    bp = B.BatchedPlan(len(ws), [dev(psf[0], dt)], opts=o1)
    fb, rb = bp.run_batched(B.ALG_SGP, g, [[10.0]] * len(ws), opts=o1)
    bp.close()
    assert all(r.fused_linesearch != 2 for r in rb)
    for i in (0, 17, 39):
        fo, ro = _oracle(ws[i], n, **{**ws[0]["opts"], "max_iter": 1, "stop_rule": 0})
        assert rel_l2(fb[i].cpu().numpy(), fo) <= 1e-5


@pytest.mark.parametrize("dt", [np.float32, np.float64])
@pytest.mark.parametrize("s_,sbar", [(160, 256), (96, 128)])
def test_cluster_kernel_with_boundary_effect_correction(s_, sbar, dt):
    """Eq.16-23 inside the cluster kernel: a 160^2 image reconstructed on a 256^2 object grid -- the size of the paper's
    sub-domain problems -- and 96^2 in 128^2 (C3 recipe: stars also outside the image, Gauss + Moffat PSF,
    b = 5, paper-default options incl. the adaptive bounds).  One iteration at 1e-5 / 1e-11; 20 iterations: image over R, zero
    outside R, J0 trace, identical rule / backtrack traces; and the launch-per-pass path to rounding"""
    _need_gpu()
    t = TOL[dt]
    w = synth.make("C3", s=s_, sbar=sbar, n_stars=150, max_iter=20, fwhm=8.0)
    S = w["S"]
    for it in (1, 20):
        kw = {**w["opts"], "max_iter": it, "stop_rule": 0}
        fo, ro = oracle_run(w, max_iter=it, stop_rule=0)
        out = {}
        for ug in (1, 1 | NO_CLUSTER):
            o = B.default_options(**{**kw, "use_graph": ug})
            plan = B.Plan([dev(w["psf"][0], dt)], S=S, opts=o)
            f, r = plan.sgp([dev(w["g"][0], dt)], w["b"], opts=o)
            out[ug] = (f.cpu().numpy(), r)
            plan.close()
        fg, rg = out[1]
        fp, rp = out[1 | NO_CLUSTER]
        assert rg.fused_linesearch == 2 and rp.fused_linesearch != 2
        e = rel_l2(fg, fo)
        print(f"[measured] cluster_boundary_{s_}in{sbar} {np.dtype(dt).name} rel_l2_{it}it = {e:.3e}")
        assert e <= (t["one"] if it == 1 else t["run"]) and np.max(np.abs(fg - fo)) <= t["pix"] * np.max(fo)
        assert np.array_equal(fg == 0, fo == 0) or np.count_nonzero((fg == 0) != (fo == 0)) <= (8 if dt == np.float32 else 0)   # R (alpha_j >= sigma_R, Eq.20)
        assert np.max(np.abs(rg.J - ro.J) / np.abs(ro.J)) <= (1e-3 if dt == np.float32 else t["J"])
        assert np.array_equal(rg.rule, ro.rule) and np.array_equal(rg.backtracks, ro.backtracks) and rg.n_fft2 == ro.n_fft2
        assert rel_l2(fg, fp) <= (1e-4 if dt == np.float32 else 1e-11) and np.array_equal(rg.rule, rp.rule)


def test_mosaic_runs_its_sub_domains_through_the_cluster_kernel():
    """a 256^2 image as four overlapping 160^2 sub-images, each reconstructed on a 256^2 grid with boundary-effect
    correction -- one batched plan, one cluster per sub-domain.  Both paths against the oracle's mosaic (north_star: 1e-3 over a run)
    wherever a tile took the oracle's branches (same number of backtracks: reading A23); the two paths against each other when all
    their tiles did"""
    _need_gpu()
    w = synth.make("C1", n=256, max_iter=15, stop_rule=0)
    kw = {**w["opts"], "max_iter": 15, "stop_rule": 0}
    mo, ro = oracle.mosaic("sgp", w["g"], w["psf"], w["b"], 2, 2, (160, 160), opts=oracle.default_options(**kw))
    lay = oracle.mosaic_layout(256, 256, 2, 2, 160, 160, 256, 256)
    res = {}
    for ug in (1, 1 | NO_CLUSTER):
        o = B.default_options(**{**kw, "use_graph": ug})
        m, r = B.mosaic(B.ALG_SGP, [dev(a, np.float32) for a in w["g"]], [dev(k, np.float32) for k in w["psf"]], w["b"], 2, 2, (160, 160), opts=o)
        res[ug] = (m.cpu().numpy(), r)
    rs, rp = res[1][1], res[1 | NO_CLUSTER][1]
    assert all(x.fused_linesearch == 2 for x in rs) and all(x.fused_linesearch != 2 for x in rp)
    same = {}
    for ug, (m, rr) in res.items():
        same[ug] = [x.iterations == y.iterations == 15 and x.total_backtracks == y.total_backtracks for x, y in zip(rr, ro)]
        assert sum(same[ug]) >= 3, (ug, same[ug])                    # a flipped Armijo test in one tile is a valid run; more is a defect
        for t, x, y, ok in zip(lay, rr, ro, same[ug]):
            assert x.iterations == 15 and np.isfinite(x.J0_final)
            if not ok:
                continue
            y0, x0, hy, hx = t["out"]
            e = rel_l2(m[y0:y0 + hy, x0:x0 + hx], mo[y0:y0 + hy, x0:x0 + hx])
            print(f"[measured] mosaic_tile use_graph={ug} rel_l2_15it = {e:.3e}")
            assert e <= 1e-3 and abs(x.J0_final - y.J0_final) <= 1e-3 * abs(y.J0_final)      # fp32 J0 of a boundary problem: as in the test above
    if all(same[1]) and all(same[1 | NO_CLUSTER]):
        e = rel_l2(res[1][0], res[1 | NO_CLUSTER][0])
        print(f"[measured] mosaic cluster_vs_passes rel_l2_15it = {e:.3e}")
        assert e <= 1e-3


# ------------------------------------------------------------------------------------------------ Richardson-Lucy rounds in the cluster kernel
def _rl_both(w, dt, S=None, **kw):
    """(f, result) of rl_* through the cluster kernel and through the launch-per-pass path"""
    out = []
    for ug in (1, 1 | NO_CLUSTER):
        o = B.default_options(**{**kw, "use_graph": ug})
        plan = B.Plan([dev(w["psf"][0], dt)], S=S, opts=o)
        f, r = plan.rl([dev(w["g"][0], dt)], w["b"], opts=o)
        out.append((f.cpu().numpy(), r))
        plan.close()
    return out


@pytest.mark.parametrize("dt", [np.float32, np.float64])
@pytest.mark.parametrize("variant", ["plain", "relax", "linear", "boundary"])
def test_cluster_kernel_richardson_lucy(variant, dt):
    """Eq.1 (plain), Eq.3 (multiplicative relaxation, exponent 1.5), Eq.4 (linear relaxation, lambda = 1.4) at 256^2 and Eq.21
    (boundary-effect correction, 160^2 in 256^2): one update at 1e-5 / 1e-11, 30 updates at 1e-4 / 1e-10 with the whole J0 trace
    (RL does not branch: DESIGN.md 3a), against the oracle; and the launch-per-pass path to rounding"""
    _need_gpu()
    if variant == "boundary":
        w = synth.make("C3", s=160, sbar=256, n_stars=150, max_iter=30, fwhm=8.0)
    else:
        w = synth.make("C0", n=256)
    extra = {"relax": {"rl_relax": 1.5}, "linear": {"rl_linear": 1.4}}.get(variant, {})
    for it in (1, 30):
        kw = {**w["opts"], "max_iter": it, "stop_rule": 0, **extra}
        fo, ro = oracle_run(w, alg="rl", **{"max_iter": it, "stop_rule": 0, **extra})
        (fg, rg), (fp, rp) = _rl_both(w, dt, S=w.get("S"), **kw)
        assert rg.fused_linesearch == 2 and rp.fused_linesearch != 2
        assert rg.iterations == ro.iterations == it and rg.n_fft2 == ro.n_fft2 == rp.n_fft2
        e = rel_l2(fg, fo)
        print(f"[measured] cluster_rl_{variant} {np.dtype(dt).name} rel_l2_{it}it = {e:.3e}")
        assert e <= ((1e-5 if it == 1 else 1e-4) if dt == np.float32 else (1e-11 if it == 1 else 1e-10))
        assert np.max(np.abs(fg - fo)) <= (1e-3 if dt == np.float32 else 1e-9) * np.max(fo) and np.all(fg >= 0)
        assert np.max(np.abs(rg.J - ro.J) / np.abs(ro.J)) <= (1e-4 if dt == np.float32 else 1e-10)
        assert rel_l2(fg, fp) <= (2e-5 if dt == np.float32 else 1e-12)


@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_cluster_kernel_rl_stop_rule_and_batches(dt):
    """RL with the Eq.24 rule stops at the oracle's iteration; a batch of 5 problems (different backgrounds, different stopping
    iterations) equals the same problems run alone, bit for bit"""
    _need_gpu()
    n, nb = 128, 5
    ws = [synth.make("C0", n=n, seed_idx=90 + i) for i in range(nb)]
    kw = {**ws[0]["opts"], "max_iter": 400, "stop_rule": 1, "tol": 1e-3}
    o = B.default_options(**kw)
    g = [[dev(w["g"][0], dt)] for w in ws]
    b = [[10.0 + i] for i in range(nb)]
    bp = B.BatchedPlan(nb, [dev(ws[0]["psf"][0], dt)], opts=o)
    fb, rb = bp.run_batched(B.ALG_RL, g, b, opts=o)
    bp.close()
    single = B.Plan([dev(ws[0]["psf"][0], dt)], opts=o)
    for i in range(nb):
        fs, rs = single.run(B.ALG_RL, g[i], b[i], opts=o)
        assert rb[i].fused_linesearch == 2 and rs.fused_linesearch == 2
        assert torch.equal(fb[i], fs) and rb[i].iterations == rs.iterations and np.array_equal(rb[i].J, rs.J)
        P = oracle.Problem(ws[0]["psf"])
        fo, ro = P.rl(ws[i]["g"], [np.full((n, n), b[i][0])], opts=oracle.default_options(**kw))
        assert rb[i].stop_reason == ro.stop_reason == 2 and abs(rb[i].iterations - ro.iterations) <= (1 if dt == np.float32 else 0)
        if rb[i].iterations == ro.iterations:
            assert rel_l2(fb[i].cpu().numpy(), fo) <= (1e-3 if dt == np.float32 else 1e-9)
    single.close()
    assert len({r.iterations for r in rb}) > 1
