"""GPU parity tests for the batched plan and the mosaic driver: every problem
of a batch against the oracle run of that problem alone, and the mosaic against the oracle's mosaic."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402  (test infrastructure)
from paper_1210_2258_b200 import binding as B  # noqa: E402
from paper_1210_2258_b200 import synth  # noqa: E402

from test_gpu_parity import _need_gpu, dev, rel_l2  # noqa: E402


@pytest.mark.parametrize("dt,tol1,tol", [(np.float32, 1e-5, 1e-3), (np.float64, 1e-11, 1e-10)])
@pytest.mark.parametrize("alg", ["sgp", "rl"])
def test_batched_plan_every_problem_matches_its_own_oracle_run(alg, dt, tol1, tol):
    """5 different star fields (different seeds, different backgrounds) through ONE batched plan: each problem keeps its own
    step lengths, backtracks and stopping iteration (Eq.24 stop: the problems stop at different iterations), and equals --
    bit for bit -- the same problem run alone through an ordinary plan; against the oracle: 1e-5 after one iteration, traces
    equal over the un-branched stretch (10 iterations: at 128^2 in float the J0 of the C0 recipe leaves 1e-4 of the fp64 sequence
    between iterations 10 and 15, whatever evaluates it -- DESIGN.md 3a, reading A23)."""
    _need_gpu()
    nb, n = 5, 128
    ws = [synth.make("C0", n=n, seed_idx=40 + i) for i in range(nb)]
    psf = ws[0]["psf"]
    g = [[dev(w["g"][0], dt)] for w in ws]
    b = [[10.0 + i] for i in range(nb)]
    algc = B.ALG_SGP if alg == "sgp" else B.ALG_RL
    for kw in (dict(max_iter=1, stop_rule=0), dict(max_iter=10, stop_rule=0), dict(max_iter=300, stop_rule=1, tol=3e-4)):
        okw = {**ws[0]["opts"], **kw}
        o = B.default_options(**okw)
        bp = B.BatchedPlan(nb, [dev(psf[0], dt)], opts=o)
        fb, rb = bp.run_batched(algc, g, b, opts=o)
        bp.close()
        single = B.Plan([dev(psf[0], dt)], opts=o)
        its = []
        for i in range(nb):
            fs, rs = single.run(algc, g[i], b[i], opts=o)
            assert torch.equal(fb[i], fs) and rb[i].iterations == rs.iterations and np.array_equal(rb[i].J, rs.J)
            assert np.array_equal(rb[i].backtracks, rs.backtracks) and rb[i].stop_reason == rs.stop_reason
            its.append(rb[i].iterations)
            if kw["max_iter"] <= 10:
                P = oracle.Problem(psf)
                oo = oracle.default_options(**okw)
                fo, ro = (P.sgp if alg == "sgp" else P.rl)(ws[i]["g"], [np.full((n, n), b[i][0])], opts=oo)
                t = tol1 if kw["max_iter"] == 1 else tol
                assert rel_l2(fb[i].cpu().numpy(), fo) <= t and abs(rb[i].J0_final - ro.J0_final) <= (1e-4 if dt == np.float32 else 1e-11) * ro.J0_final
                if alg == "sgp":
                    assert np.array_equal(rb[i].backtracks, ro.backtracks) and np.array_equal(rb[i].rule, ro.rule)
        single.close()
        if kw["stop_rule"] == 1:
            assert len(set(its)) > 1, "the problems must stop at different iterations for this test to mean anything"
            assert all(r.stop_reason == 2 for r in rb)


def test_batched_plan_multi_image_boundary_and_bad_data():
    """p = 2 with boundary-effect correction in a batch of 3; one problem with a NaN pixel reports SGP_ERR_DATA in its own
    result while the others are solved; options that batched plans do not take are refused"""
    _need_gpu()
    dt = np.float32
    ws = [synth.make("C3", s=64, sbar=128, n_stars=30, max_iter=8, fwhm=8.0, seed_idx=50 + i) for i in range(3)]
    w2 = synth.make("C3", s=64, sbar=128, n_stars=30, max_iter=8, fwhm=14.0, seed_idx=60)
    psf = [ws[0]["psf"][0], w2["psf"][0]]
    S = ws[0]["S"]
    o = B.default_options(**{**ws[0]["opts"], "max_iter": 8, "stop_rule": 0})
    g = [[dev(w["g"][0], dt), dev(w["g"][0][::-1].copy(), dt)] for w in ws]
    b = [[5.0, 6.0]] * 3
    bp = B.BatchedPlan(3, [dev(k, dt) for k in psf], S=S, opts=o)
    fb, rb = bp.run_batched(B.ALG_SGP, g, b, opts=o)
    P = oracle.Problem(psf, masked=True, S=S, sigma_R=o.sigma_R)
    for i, w in enumerate(ws):
        ge = P.embed([w["g"][0], w["g"][0][::-1]]); be = [np.full((P.ny, P.nx), 5.0), np.full((P.ny, P.nx), 6.0)]
        fo, ro = P.sgp(ge, be, opts=oracle.default_options(**{**w["opts"], "max_iter": 8, "stop_rule": 0}))
        assert rb[i].iterations == 8 and rel_l2(fb[i].cpu().numpy(), fo) <= 1e-3
    gbad = [[t.clone() for t in prob] for prob in g]
    gbad[1][0][3, 3] = float("nan")
    fb2, rb2 = bp.run_batched(B.ALG_SGP, gbad, b, opts=o, check=False)
    assert [r.rc for r in rb2] == [B.OK, B.ERR_DATA, B.OK]
    assert torch.equal(fb2[0], fb[0]) and torch.equal(fb2[2], fb[2])
    for extra in ({"flux_constraint": 1}, {"refresh_every": 2}):
        with pytest.raises(B.SgpError) as ei:
            bp.run_batched(B.ALG_SGP, g, b, opts=B.default_options(**{**ws[0]["opts"], "max_iter": 8, "stop_rule": 0, **extra}))
        assert ei.value.code == B.ERR_UNSUPPORTED
    bp.close()


@pytest.mark.parametrize("dt,tol", [(np.float32, 1e-3), (np.float64, 1e-10)])
@pytest.mark.parametrize("alg", ["sgp", "rl", "osem"])
def test_mosaic_of_four_subdomains_matches_the_oracle(alg, dt, tol):
    """PAPER.md:385-389 at its own sizes: a 256 x 256 image cut into four 160 x 160 sub-images, each zero-padded into a 256 x 256
    array with the 256 x 256 PSF, 128 x 128 parts extracted; single image (Table 2) and three images (Table 6)"""
    _need_gpu()
    for p in (1, 3):
        w = synth.make("C1", n=256, max_iter=20, stop_rule=0) if p == 1 else synth.make("C2", n=256, max_iter=20)
        if alg == "osem" and p == 1:
            continue
        o = B.default_options(**{**w["opts"], "max_iter": 20, "stop_rule": 0})
        algc = {"sgp": B.ALG_SGP, "rl": B.ALG_RL, "osem": B.ALG_OSEM}[alg]
        m, res = B.mosaic(algc, [dev(a, dt) for a in w["g"]], [dev(k, dt) for k in w["psf"]], w["b"], 2, 2, (160, 160), opts=o)
        mo, ro = oracle.mosaic(alg, w["g"], w["psf"], w["b"], 2, 2, (160, 160), oracle.default_options(**{**w["opts"], "max_iter": 20, "stop_rule": 0}))
        assert len(res) == 4 and all(r.iterations == 20 for r in res)
        e = rel_l2(m.cpu().numpy(), mo)
        print(f"[measured] mosaic {alg} p={p} {np.dtype(dt).name} rel_l2 = {e:.3e}")
        assert e <= tol
        for r, r_o in zip(res, ro):
            assert abs(r.J0_final - r_o.J0_final) <= ((5e-3 if alg == "sgp" else 1e-5) if dt == np.float32 else 1e-10) * r_o.J0_final
    # host pointers
    w = synth.make("C1", n=256, max_iter=5, stop_rule=0)
    o = B.default_options(**{**w["opts"], "max_iter": 5, "stop_rule": 0})
    mh, _ = B.mosaic(B.ALG_SGP, [a.astype(dt) for a in w["g"]], [a.astype(dt) for a in w["psf"]], w["b"], 2, 2, (160, 160), opts=o, host=True)
    md, _ = B.mosaic(B.ALG_SGP, [dev(a, dt) for a in w["g"]], [dev(k, dt) for k in w["psf"]], w["b"], 2, 2, (160, 160), opts=o)
    assert np.array_equal(mh, md.cpu().numpy())
