"""A small tour of the library for `compute-sanitizer`: every kernel family on tiny grids, incl.
the Armijo backtracking (forced in every iteration), the fused and the separate line-search schedules, boundary masks, three images,
RL / OSEM on the fused schedule, a 5-smooth grid with padded thread groups, a batched plan, the flux-constrained projection, the
refresh round, the Eq.25 stop and the one-cluster-per-problem kernel of the small grids.  Not a pytest module: run as

    compute-sanitizer --tool memcheck  python tests/gpu_sanitize_case.py
    compute-sanitizer --tool racecheck python tests/gpu_sanitize_case.py
    compute-sanitizer --tool synccheck python tests/gpu_sanitize_case.py

and keep the tool's summary under profiles/.  Exit code 0 and "sanitize tour ok" mean the tour itself ran to the end."""
import sys
from pathlib import Path

import numpy as np
import torch

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))

from paper_1210_2258_b200 import binding as B  # noqa: E402
from paper_1210_2258_b200 import synth  # noqa: E402


def dev(a, dt=np.float32):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=dt), device="cuda")


def main():
    torch.cuda.set_device(0)
    for dt in (np.float32, np.float64):
        # single image 64^2, both schedules, graph replay on / off, backtracking in every iteration
        w = synth.make("C0", n=64)
        for bits in (1 | 4, 1 | 8, 8):
            kw = {**w["opts"], "max_iter": 12, "use_graph": bits, "alpha0": 1e5, "alpha_min": 1e3, "alpha_max": 1e6}
            plan = B.Plan([dev(w["psf"][0], dt)], opts=B.default_options(**kw))
            f, r = plan.sgp([dev(w["g"][0], dt)], w["b"])
            assert r.iterations == 12 and r.total_backtracks > 0 and torch.isfinite(f).all()
            f, r = plan.rl([dev(w["g"][0], dt)], w["b"])
            plan.close()
        # small grids: the whole iteration in one kernel, one cluster per problem (csrc/small.cuh) -- distributed shared memory,
        # st.async + mbarrier, cluster barriers; backtracking in every iteration; a batch of three problems
        w = synth.make("C0", n=128)
        kw = {**w["opts"], "max_iter": 8, "alpha0": 1e5, "alpha_min": 1e3, "alpha_max": 1e6}
        plan = B.Plan([dev(w["psf"][0], dt)], opts=B.default_options(**kw))
        f, r = plan.sgp([dev(w["g"][0], dt)], w["b"])
        assert r.fused_linesearch == 2 and r.iterations == 8 and r.total_backtracks > 0 and torch.isfinite(f).all()
        plan.close()
        ws = [synth.make("C0", n=128, seed_idx=80 + i) for i in range(3)]
        o = B.default_options(**{**ws[0]["opts"], "max_iter": 30, "stop_rule": 1, "tol": 1e-3})
        bp = B.BatchedPlan(3, [dev(ws[0]["psf"][0], dt)], opts=o)
        fb, rb = bp.run_batched(B.ALG_SGP, [[dev(x["g"][0], dt)] for x in ws], [[10.0]] * 3, opts=o)
        assert all(x.fused_linesearch == 2 for x in rb)
        bp.close()
        # three images, 128^2: SGP, RL, OSEM; flux constraint; refresh round; Eq.25
        w = synth.make("C2", n=128, max_iter=12)
        g = [dev(a, dt) for a in w["g"]]
        plan = B.Plan([dev(k, dt) for k in w["psf"]], opts=B.default_options(**w["opts"]))
        for run in (plan.sgp, plan.rl, plan.osem):
            f, r = run(g, w["b"])
            assert r.iterations == 12
        f, r = plan.sgp(g, w["b"], opts=B.default_options(**{**w["opts"], "flux_constraint": 1}))
        f, r = plan.sgp(g, w["b"], opts=B.default_options(**{**w["opts"], "refresh_every": 3}))
        f, r = plan.sgp(g, w["b"], opts=B.default_options(**{**w["opts"], "stop_rule": B.STOP_MINERR}), truth=dev(w["truth"], dt))
        f, r = plan.rl(g, w["b"], opts=B.default_options(**{**w["opts"], "stop_rule": B.STOP_MINERR}), truth=dev(w["truth"], dt))
        plan.close()
        # boundary-effect correction on a 5-smooth grid (80 x 200: radix 20 / 10 / 5 / 4, padded thread groups), smoothed start
        w = synth.make("C3", s=64, sbar=128, n_stars=30, max_iter=8, fwhm=8.0)
        plan = B.Plan([dev(k, dt) for k in w["psf"]], S=w["S"], opts=B.default_options(**{**w["opts"], "init": B.INIT_CONST_SMOOTH}))
        f, r = plan.sgp([dev(a, dt) for a in w["g"]], w["b"])
        f, r = plan.osem([dev(a, dt) for a in w["g"]], w["b"])
        plan.close()
        w = synth.make("C0r", ny=80, nx=200)
        plan = B.Plan([dev(w["psf"][0], dt)], opts=B.default_options(**{**w["opts"], "max_iter": 6}))
        f, r = plan.sgp([dev(w["g"][0], dt)], w["b"])
        f, r = plan.rl([dev(w["g"][0], dt)], w["b"])
        plan.close()
        # batched plan: 3 problems, Eq.24 stop (the problems stop at different iterations)
        ws = [synth.make("C0", n=64, seed_idx=70 + i) for i in range(3)]
        o = B.default_options(**{**ws[0]["opts"], "max_iter": 40, "stop_rule": 1, "tol": 1e-3})
        bp = B.BatchedPlan(3, [dev(ws[0]["psf"][0], dt)], opts=o)
        fb, rb = bp.run_batched(B.ALG_SGP, [[dev(x["g"][0], dt)] for x in ws], [[10.0]] * 3, opts=o)
        fb, rb = bp.run_batched(B.ALG_RL, [[dev(x["g"][0], dt)] for x in ws], [[10.0]] * 3, opts=o)
        bp.close()
    # mosaic (four sub-domains as one batched boundary plan)
    w = synth.make("C1", n=128, max_iter=6, stop_rule=0)
    o = B.default_options(**{**w["opts"], "max_iter": 6, "stop_rule": 0})
    m, res = B.mosaic(B.ALG_SGP, [dev(a) for a in w["g"]], [dev(k) for k in w["psf"]], w["b"], 2, 2, (80, 80), opts=o)
    assert torch.isfinite(m).all()
    # one-shot calls (the plan is kept between them, then released) and the entry point whose scratch is a static device array
    w = synth.make("C0", n=64)
    o = B.default_options(**{**w["opts"], "max_iter": 5})
    for _ in range(2):
        B.sgp_single(dev(w["g"][0]), dev(w["psf"][0]), w["b"][0], opts=o)
    B.release_cached_plans()
    rho = torch.zeros(1, dtype=torch.float64, device="cuda")
    for n in (1000, 70000, 400000):
        x = torch.rand(n, device="cuda") + 0.5
        B.rel_error_static(x, x + 0.1, rho)
        B.rel_error_static(x + 0.1, x, rho)
        assert 0.0 < float(rho.item()) < 1.0
    torch.cuda.synchronize()
    print("sanitize tour ok")


if __name__ == "__main__":
    main()
