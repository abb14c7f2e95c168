#!/usr/bin/env python
"""bench.py -- throughput of the SGP hot path (arXiv:1210.2258, Algorithm 1) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4c|C4a|C4b|C1|C0] [--alg sgp|rl] [--dtype f32|f64]
    python bench.py --impl reference ...     # the CPU oracle on the host cores (the tier's reference arm)

One STEP is one whole reconstruction of the workload through the plan form of the C ABI (sgp_plan_run):
the start-point phase (SURVEY.md 8(a) row a0'') followed by a FIXED number of SGP iterations (rows a1-a11;
200 for C4c, BASELINE.json configs[4]) with the inputs already resident in HBM.  The metric is SGP
iterations per second (BASELINE.json `metric`), whole job over all ranks; `gpixel_iter_per_s` = value x
object-grid pixels / 1e9.  The default workload is C4c: single image 2048 x 2048 fp32, galaxies + stars,
Airy PSF, b = 20, paper-default SGP options, 200 iterations -- the configuration the metric is quoted on.

The printed JSON line also carries
  e2e          the same metric through sgp_single_host / sgp_multi_host: HOST (pinned) buffers, PSF transfer functions,
               host->device and device->host copies all inside the timed region (the plan itself is the one the library
               keeps from the previous one-shot call of the same geometry: include/sgp.h);
  roofline     for the kernel with the largest share of the iteration: algorithmic bytes per launch
                / its mean duration, measured with CUDA event pairs around every launch
               in an instrumented pass of the same step right after the timed region (sgp_plan_set_profiling);
               `iteration` gives the same for the whole iteration from the un-instrumented timed region;
  cpu_baseline the oracle (oracle/, plain C, fp64, as it stands) on the host cores, on a bounded sample.
N > 1: independent replicas, one problem per GPU ("replicas only"), no collective on
the data path; time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import numpy as np  # noqa: E402

WORKLOADS = {
    # name: (synth config, kwargs, description)
    "C4c": ("C4c", {}, "C4c: single-image SGP 2048x2048, galaxies+stars, Airy PSF, b=20, Poisson, 200 iterations"),
    "C4a": ("C4a", {}, "C4a: single-image SGP 4096x4096, galaxies+stars, Airy PSF, b=20, Poisson, 200 iterations"),
    "C4b": ("C4b", {}, "C4b: multi-image SGP 3x2048x2048, rotated LBT PSFs, cluster+nebula, b_j=15, 200 iterations"),
    "C1": ("C1", dict(max_iter=200, stop_rule=0), "C1: single-image SGP 512x512, galaxies+stars, Airy PSF, b=20, 200 iterations"),
    "C0": ("C0", dict(), "C0: single-image SGP 256x256, 20 stars, Gaussian PSF, b=10, M=10, 100 iterations"),
}


def load_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        try:
            return float(json.loads(f.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def planes_per_launch(p: int, b_array: bool, masked: bool, backtracks_per_iter: float = 0.0, fused: bool = True):
    """algorithmic planes (n reals each) read + written per launch of the kernels as built, DESIGN.md section 6.
    K6 (fused line search) = spectrum, q, g read; u, q(k+1), ratio spectrum written.  K1 = g, q, u read; q, spectrum
    written: it returns at once unless the previous iteration backtracked (average over the launches of the run, the
    share of such iterations bounded by backtracks per iteration).  K3 = spectrum, f, d, grad read; f, grad written
    (lazy a10 for f).  K7 = q, u, g read once per Armijo trial (average over the launches of the run)."""
    ba = p if b_array else 0
    m = 1 if masked else 0
    k1 = (5 * p + ba) * (min(1.0, backtracks_per_iter) if fused else 1.0)
    k6 = (6 * p + ba) if fused else (4 * p + ba)
    return {
        "K1_ratio_rowfft": k1, "K2_col_conjsum": 2 * p + 1, "K3_rowifft_grad_bb": 6 + m,
        "K4_project_rowfft": 4 + m, "K5_col_mult": 2 * p + 1, "K6_rowifft_linesearch": k6,
        "K7_backtrack": (3 * p + ba) * backtracks_per_iter,
        # RL on the schedule of SURVEY.md 8(d) (7p + 6 planes): R3 = row C2R -> J0 -> ratio -> row R2C (spectrum_j, g_j read;
        # ratio spectrum_j written), R6 = row C2R -> update -> row R2C (spectrum, f read; f, spectrum written); R1 runs once per run
        "R1_rowfft": 2, "R2_col_mult": 2 * p + 1, "R3_rowifft_q_J": 3 * p + ba, "R4_ratio_rowfft": 3 * p + ba,
        "R5_col_conjsum": 2 * p + 1, "R6_rowifft_update": 4 + m,
    }


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md clocks line)"""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            c = [x.strip() for x in r.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def make_workload(name: str, rank: int):
    """rank r > 0 gets an independent replica: the same recipe drawn from another seed"""
    from paper_1210_2258_b200 import synth
    cfg, kw, desc = WORKLOADS[name]
    if rank == 0:
        return synth.make(cfg, **kw), desc
    sidx = 100 * rank
    if cfg == "C4c":
        w = synth.c1_galaxies_airy(2048, seed_idx=6 + sidx, max_iter=200, stop_rule=0)
    elif cfg == "C4a":
        w = synth.c1_galaxies_airy(4096, seed_idx=4 + sidx, max_iter=200, stop_rule=0)
    elif cfg == "C4b":
        w = synth.c2_lbt_multi(2048, seed_idx=5 + sidx, max_iter=200)
    elif cfg == "C1":
        w = synth.c1_galaxies_airy(512, seed_idx=1 + sidx, **kw)
    else:
        w = synth.c0_stars_gaussian(256, seed_idx=sidx)
    return w, desc


def max_over_ranks(x: float, world: int, device=None) -> float:
    """the slowest rank's time: all-reduce MAX over the process group (NCCL on GPUs; gloo in the CPU tests)"""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(ms_local: float, iters_per_step: int, steps: int, world: int, device=None) -> tuple:
    """(iterations/s over all ranks, ms of the slowest rank): replicas only, every rank does iters_per_step x steps"""
    ms = max_over_ranks(ms_local, world, device)
    return iters_per_step * steps * world / (ms * 1e-3), ms


def cufft_compare(w, dev, tdt, iters: int, warm: int = 5):
    """In-run comparison baseline named by north_star: the same SGP iteration (Alg.1, step lengths
    PAPER.md:130-155) written the way the paper's own GPU code is organised (one library call per
    vector operation, the host decides every branch), with cuFFT (torch.fft) for the 2p + 2 transforms and torch
    elementwise / reduction kernels for the rest.  Periodic (unmasked) workloads only.  Returns iterations/s over
    `iters` iterations after `warm` untimed ones, and J0 for a sanity comparison with the library's trace."""
    import torch
    fft = torch.fft
    o = w["opts"]
    p = len(w["g"]); ny, nx = w["psf"][0].shape
    g = [torch.as_tensor(np.ascontiguousarray(a), device=dev).to(tdt).clamp_(min=0) for a in w["g"]]
    b = [float(x) for x in w["b"]]
    K = []
    for k in w["psf"]:
        kk = torch.as_tensor(np.ascontiguousarray(k), device=dev).to(torch.float64)
        K.append(fft.rfft2(fft.ifftshift(kk / kk.sum()).to(tdt)))
    dsum = lambda x: float(x.sum(dtype=torch.float64).item())
    A = lambda F, j: fft.irfft2(K[j] * F, s=(ny, nx))
    def kl(gj, y):
        return torch.where(gj > 0, gj * torch.log(gj / y) + y - gj, y)
    def J0(q, lam=None, u=None):
        return sum(dsum(kl(g[j], (q[j] if u is None else q[j] + lam * u[j]) + b[j])) for j in range(p))
    def AT_ratio(q):
        F = None
        for j in range(p):
            t = torch.conj(K[j]) * fft.rfft2(g[j] / (q[j] + b[j]))
            F = t if F is None else F + t
        return fft.irfft2(F, s=(ny, nx))
    c0 = max(0.0, sum(dsum(g[j] - b[j]) for j in range(p)) / (p * ny * nx))
    f = torch.full((ny, nx), c0, dtype=tdt, device=dev)
    Ff = fft.rfft2(f)
    q = [A(Ff, j) for j in range(p)]
    J = J0(q)
    L1, L2 = float(o.get("L1", 1e-10)), float(o.get("L2", 1e10))
    if o.get("adaptive_L", 1):
        y = f * AT_ratio(q) / p
        ymin, ymax = float(y[y > 0].min().item()), float(y.max().item())
        L1, L2 = (ymin / 10, ymax * 10) if ymax / ymin < 50 else (ymin, ymax)
    beta, theta = float(o.get("beta", 1e-4)), float(o.get("theta", 0.4))
    amin, amax, alpha_prev, tau = 1e-5, 1e5, 1.3, 0.5
    m_alpha, M = int(o.get("m_alpha", 3)), int(o.get("armijo_memory", 1))
    ring, Jhist = [], [J]
    f_prev = grad_prev = None
    on_gpu = torch.device(dev).type == "cuda"
    if on_gpu:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for k in range(warm + iters):
        if k == warm:
            if on_gpu:
                torch.cuda.synchronize(); ev0.record()
            else:
                t0 = time.perf_counter()
        grad = p - AT_ratio(q)
        D = f.clamp(L1, L2) / p
        if k == 0:
            alpha = 1.3
        else:
            s_, z_ = f - f_prev, grad - grad_prev
            a_, c_, e_, h_ = dsum(s_ * s_ / (D * D)), dsum(s_ * z_ / D), dsum(s_ * z_ * D), dsum(z_ * z_ * D * D)
            a1 = min(10 * alpha_prev, amax) if c_ <= 0 else min(amax, max(amin, a_ / c_))
            a2 = min(10 * alpha_prev, amax) if e_ <= 0 else min(amax, max(amin, e_ / h_))
            ring = (ring + [a2])[-m_alpha:]
            if k <= 20 or a2 / a1 <= tau:
                alpha = min(ring)
                if k > 20: tau *= 0.9
            else:
                alpha = a1; tau *= 1.1
            alpha_prev = alpha
        d = (f - alpha * D * grad).clamp_(min=0) - f
        gd = dsum(grad * d)
        Fd = fft.rfft2(d)
        u = [A(Fd, j) for j in range(p)]
        lam, Jref = 1.0, max(Jhist[-M:])
        for _ in range(30):
            Jn = J0(q, lam, u)
            if np.isfinite(Jn) and Jn <= Jref + beta * lam * gd:
                break
            lam *= theta
        f_prev, grad_prev = f, grad
        f = f + lam * d
        q = [q[j] + lam * u[j] for j in range(p)]
        J = Jn; Jhist.append(J)
    if on_gpu:
        ev1.record(); torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1)
    else:
        ms = 1e3 * (time.perf_counter() - t0)
    return {"value": iters / (ms * 1e-3), "unit": "iterations/s", "iterations": iters, "warmup_iterations": warm,
            "J0_after": warm + iters, "J0": J,
            "impl": "torch.fft (cuFFT) rfft2/irfft2 + torch elementwise and reduction kernels, scalar logic on the host "
                    "(the organisation of the paper's GPUlib code, PAPER.md:302-310); comparison baseline only"}


def oracle_time(w, iters_a: int, iters_b: int):
    """wall time of the oracle for iters_a and iters_b SGP iterations of workload w (fp64, OpenMP over the host cores)"""
    import oracle
    oo = oracle.default_options(**{**w["opts"], "max_iter": iters_a})
    P = oracle.Problem(w["psf"], masked=w["S"] is not None, S=w["S"], sigma_R=oo.sigma_R)
    ge = P.embed(w["g"]); be = [np.full((P.ny, P.nx), float(v)) for v in w["b"]]
    out = []
    for it in (iters_a, iters_b):
        oo.max_iter = it
        t0 = time.perf_counter()
        _, r = P.sgp(ge, be, opts=oo)
        out.append(time.perf_counter() - t0)
        assert r.iterations == it
    return out


def oracle_time_single_thread(workload: str):
    """(seconds per SGP iteration, sample text) of the oracle on ONE host thread: t(1 iteration) - t(0 iterations) of the
    same workload, in a child process (the OpenMP thread count is fixed when the oracle library is loaded)"""
    code = ("import sys, time, json, numpy as np; sys.path.insert(0, %r)\n"
            "import oracle; from bench import make_workload\n"
            "w, _ = make_workload(%r, 0)\n"
            "oo = oracle.default_options(**{**w['opts'], 'max_iter': 0})\n"
            "P = oracle.Problem(w['psf'], masked=w['S'] is not None, S=w['S'], sigma_R=oo.sigma_R)\n"
            "ge = P.embed(w['g']); be = [np.full((P.ny, P.nx), float(v)) for v in w['b']]\n"
            "t = []\n"
            "for it in (0, 1):\n"
            "    oo.max_iter = it; t0 = time.perf_counter(); P.sgp(ge, be, opts=oo); t.append(time.perf_counter() - t0)\n"
            "print(json.dumps(t))\n") % (str(ROOT), workload)
    env = {**os.environ, "OMP_NUM_THREADS": "1"}
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=env, timeout=600)
    t0, t1 = json.loads(r.stdout.strip().splitlines()[-1])
    return t1 - t0, f"t(1 it) - t(0 it) = {t1:.2f}s - {t0:.2f}s, one thread"


def run_reference(args):
    """Reference arm of this tier: the CPU oracle as it stands, on the host cores; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    os.environ["OMP_NUM_THREADS"] = str(cores)
    import oracle
    w, desc = make_workload(args.workload, 0)
    p = len(w["g"]); ny, nx = w["psf"][0].shape
    m = args.ref_iters
    oo = oracle.default_options(**{**w["opts"], "max_iter": m})
    P = oracle.Problem(w["psf"], masked=w["S"] is not None, S=w["S"], sigma_R=oo.sigma_R)
    ge = P.embed(w["g"]); be = [np.full((P.ny, P.nx), float(v)) for v in w["b"]]
    fn = P.sgp if args.alg == "sgp" else P.rl
    for _ in range(args.warmup):
        fn(ge, be, opts=oo)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, r = fn(ge, be, opts=oo)
    dt = time.perf_counter() - t0
    value = m * args.steps / dt
    sample = (f"each step = {m} {args.alg.upper()} iterations of {args.workload} ({p}x{ny}x{nx}, fp64) from the constant start, "
              f"start-point phase (A f0, J0, adaptive bounds) inside the step; OpenMP over {cores} host threads")
    line = {"impl": "reference", "metric": "SGP iterations/s" if args.alg == "sgp" else "RL iterations/s", "value": value,
            "unit": "iterations/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "gpixel_iter_per_s": value * ny * nx / 1e9,
            "config": {"workload": desc, "iterations_per_step": m, "grid": [ny, nx], "images": p, "algorithm": args.alg},
            "cpu_baseline": {"value": value, "unit": "iterations/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "iterations/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def measure_other(name: str, alg_name: str, steps: int, dev, peak: float):
    """device-timed throughput of another workload of BASELINE.json configs[4] (north_star's target names 3 x 2048^2
    beside 2048^2; RL is timed separately): `steps` reconstructions after 3 warm-up ones, CUDA events on the launching
    stream; fractions of the roofline on SURVEY.md 8(d)'s bytes (SGP: schedule A, 14p + 14 planes; RL: 7p + 6)."""
    import torch
    from paper_1210_2258_b200 import binding as B
    w, desc = make_workload(name, 0)
    p = len(w["g"]); ny, nx = w["psf"][0].shape
    to_dev = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32), device=dev)
    opts = B.default_options(**{**w["opts"], "stop_rule": 0})
    plan = B.Plan([to_dev(k) for k in w["psf"]], S=w["S"], opts=opts)
    g = [to_dev(a) for a in w["g"]]
    f_out = torch.empty((ny, nx), dtype=torch.float32, device=dev)
    alg = B.ALG_SGP if alg_name == "sgp" else B.ALG_RL
    for _ in range(3):
        _, r = plan.run(alg, g, w["b"], opts=opts, f_out=f_out, traces=False)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(); ev0.record()
    loop_ms = 0.0
    for _ in range(steps):
        _, r = plan.run(alg, g, w["b"], opts=opts, f_out=f_out, traces=False)
        loop_ms += r.loop_ms
    ev1.record(); torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1)
    plan.close()
    iters = r.iterations
    masked = 1 if w["S"] is not None else 0
    planes = (14 * p + 14 + 2 * masked) if alg_name == "sgp" else (7 * p + 6 + masked)
    it_us = 1e3 * (loop_ms / steps) / iters
    gbs = planes * ny * nx * 4 / (it_us * 1e-6) / 1e9
    return {"workload": desc, "algorithm": alg_name, "dtype": "f32", "value": iters * steps / (ms * 1e-3), "unit": "iterations/s",
            "steps": steps, "iterations_per_step": iters, "ms_per_step": ms / steps, "iteration_us": round(it_us, 2),
            "planes": planes, "schedule": "SURVEY 8(d) schedule A (14p+14)" if alg_name == "sgp" else "SURVEY 8(d) RL schedule (7p+6)",
            "GBps": round(gbs, 1), "frac": round(gbs / peak, 4), "frac_nominal_8TBs": round(gbs / 8000.0, 4),
            "gpixel_iter_per_s": iters * steps / (ms * 1e-3) * ny * nx / 1e9, "backtracks_per_iteration": r.total_backtracks / max(1, iters),
            "fused_linesearch": int(r.fused_linesearch)}


def measure_batched(nb: int, steps: int, dev):
    """problems of the C0 recipe (256^2, different seeds) through ONE batched plan beside one C0 problem
    through an ordinary plan: aggregate iterations/s.  One problem and batches of up to 32 run one thread-block cluster per
    problem (csrc/small.cuh, `path` = cluster); the large batch runs launch-per-pass, every kernel launched once for all problems
    (blockIdx.z = problem)"""
    import torch
    from paper_1210_2258_b200 import binding as B, synth
    ws = [synth.c0_stars_gaussian(256, seed_idx=200 + i) for i in range(nb)]
    to_dev = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32), device=dev)
    opts = B.default_options(**ws[0]["opts"])
    out = {}
    for label, n_ in (("single", 1), ("batch_of_4", 4), ("batch_of_16", 16), ("batched", nb)):
        plan = B.BatchedPlan(n_, [to_dev(ws[0]["psf"][0])], opts=opts)
        g = [[to_dev(w["g"][0])] for w in ws[:n_]]
        b = [[10.0]] * n_
        for _ in range(3):
            _, rs = plan.run_batched(B.ALG_SGP, g, b, opts=opts)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); ev0.record()
        its = 0
        for _ in range(steps):
            _, rs = plan.run_batched(B.ALG_SGP, g, b, opts=opts)
            its += sum(r.iterations for r in rs)
        ev1.record(); torch.cuda.synchronize()
        plan.close()
        out[label] = {"problems": n_, "value": its / (ev0.elapsed_time(ev1) * 1e-3), "unit": "iterations/s (sum over the problems)",
                      "ms_per_step": ev0.elapsed_time(ev1) / steps, "iterations_per_problem": rs[0].iterations,
                      "path": "cluster" if rs[0].fused_linesearch == 2 else "launch-per-pass"}
    out["aggregate_speedup"] = out["batched"]["value"] / out["single"]["value"]
    out["aggregate_speedup_vs_round1_single"] = out["batched"]["value"] / 18700.0
    out["workload"] = (f"C0 recipe, 256x256 fp32, 100 SGP iterations per problem (start-point phase and result copies inside), 1 / 4 / 16 / {nb} problems in "
                       "one sgp_plan_run_batched call; round 1 ran one such problem at 18.7 kit/s (profiles/r1j_bench_lines.md)")
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1210_2258_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus != world:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch N > 1 as `python -m torch.distributed.run --nnodes=1 "
                         f"--nproc-per-node N --master-addr 127.0.0.1 bench.py --gpus N ...` (one rank per GPU)")
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.lib()   # fail loudly if the CUDA library is missing

    w, desc = make_workload(args.workload, rank)
    p = len(w["g"]); ny, nx = w["psf"][0].shape
    npdt, tdt = (np.float32, torch.float32) if args.dtype == "f32" else (np.float64, torch.float64)
    esz = np.dtype(npdt).itemsize
    iters = int(w["opts"]["max_iter"])
    okw = {**w["opts"], "stop_rule": 0}
    if args.tile_cols: okw["tile_cols"] = args.tile_cols
    if args.rows_per_block: okw["rows_per_block"] = args.rows_per_block
    okw["use_graph"] = args.graph
    opts = B.default_options(**okw)
    alg = B.ALG_SGP if args.alg == "sgp" else B.ALG_RL

    to_dev = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=npdt), device=dev)
    psfs = [to_dev(k) for k in w["psf"]]
    g = [to_dev(a) for a in w["g"]]
    plan = B.Plan(psfs, S=w["S"], opts=opts)
    f_out = torch.empty((ny, nx), dtype=tdt, device=dev)

    def step():
        _, r = plan.run(alg, g, w["b"], opts=opts, f_out=f_out, traces=False)
        return r

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        r = step()
    assert r.iterations == iters, (r.iterations, iters)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    backtracks = 0
    loop_ms = 0.0
    sync_all()
    with ClockSampler(local) as clk:
        ev0.record()
        for _ in range(args.steps):
            r = step()
            launches += r.kernel_launches; backtracks += r.total_backtracks; loop_ms += r.loop_ms
        ev1.record()
        sync_all()
    value, ms = whole_job_rate(ev0.elapsed_time(ev1), iters, args.steps, world, dev)
    J_final = r.J0_final

    # ---- instrumented pass: CUDA event pair around every launch of the same step (not part of `value`)
    plan.set_profiling(True)
    step()
    rp = step()
    kms = plan.kernel_ms()
    plan.set_profiling(False)
    bt_per_iter = rp.total_backtracks / max(1, rp.iterations)
    planes = planes_per_launch(p, False, w["S"] is not None, bt_per_iter, fused=bool(rp.fused_linesearch))
    plane_bytes = ny * nx * esz
    peak, peak_src = load_peaks()
    per_kernel = {}
    tot_ms = sum(v[0] for v in kms.values()) or 1.0
    for name, (msum, cnt) in kms.items():
        avg_us = 1e3 * msum / cnt
        gbs = planes[name] * plane_bytes / (avg_us * 1e-6) / 1e9
        per_kernel[name] = {"avg_us": round(avg_us, 2), "launches": cnt, "planes": round(planes[name], 3), "GBps": round(gbs, 1),
                            "frac": round(gbs / peak, 4), "share": round(msum / tot_ms, 4)}
    dom = max(kms, key=lambda k: kms[k][0])
    traffic = None          # DRAM read + write bytes of that kernel per launch, ncu --set full (profiles/traffic.md)
    traffic_source = None
    tf = ROOT / "profiles" / "traffic.csv"
    if tf.exists():
        try:
            for line in tf.read_text().splitlines()[1:]:
                wl, dt_, alg_, kern, nbytes = [c.strip() for c in line.split(",")]
                if (wl, dt_, alg_, kern) == (args.workload, args.dtype, args.alg, dom):
                    traffic = float(nbytes)
                    traffic_source = ("NOT measured in this run (ncu cannot run inside it): profiles/traffic.csv, written from the "
                                      "ncu --set full capture named in profiles/traffic.md (another box of the same pool, cold cache)")
        except Exception:
            traffic = None
    # schedule A (14p + 14 planes, the primary denominator); the kernels as built move 10p + 12 (+ 5p + 3p per backtracked iteration)
    iter_planes = (14 * p + 14 + (2 if w["S"] is not None else 0)) if args.alg == "sgp" else (
        7 * p + 6 + (1 if w["S"] is not None else 0))
    built_planes = sum(planes[k] for k in planes if k.startswith("K")) if args.alg == "sgp" else (
        sum(planes[k] for k in kms if k.startswith("R") and k != "R1_rowfft"))
    it_us = 1e3 * (loop_ms / args.steps) / iters          # loop only (library's own events), local rank
    it_gbs = iter_planes * plane_bytes / (it_us * 1e-6) / 1e9
    # the event pairs of the instrumented pass serialise the launches (no graph replay, no overlap of one kernel's tail with
    # the next one's head), so the kernel times add up to more than the iteration: `us_in_iteration` apportions the
    # un-instrumented iteration time by the measured shares, and those do add up to iteration.us
    sum_us = sum(v["avg_us"] * v["launches"] for v in per_kernel.values()) / max(1, iters)
    for name, v in per_kernel.items():
        v["us_in_iteration"] = round(v["share"] * it_us, 2)
        # the kernel's duration INSIDE the timed region (graph replay, no event pairs between the launches): its share of the
        # instrumented pass x the un-instrumented iteration time, per launch; the instrumented figures stay beside it
        lpi = v["launches"] / max(1, iters)                  # launches per iteration (OSEM / multi-launch kernels)
        us_timed = v["us_in_iteration"] / max(lpi, 1e-9)
        v["GBps_instrumented"], v["frac_instrumented"] = v["GBps"], v["frac"]
        v["GBps"] = round(planes[name] * plane_bytes / (us_timed * 1e-6) / 1e9, 1)
        v["frac"] = round(v["GBps"] / peak, 4)
        v["frac_nominal_8TBs"] = round(v["GBps"] / 8000.0, 4)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": per_kernel[dom]["GBps"], "peak": peak, "unit": "GB/s",
                "frac": per_kernel[dom]["frac"], "frac_nominal_8TBs": round(per_kernel[dom]["GBps"] / 8000.0, 4),
                "achieved_instrumented": per_kernel[dom]["GBps_instrumented"], "frac_instrumented": per_kernel[dom]["frac_instrumented"],
                "duration_source": "achieved = algorithmic bytes per launch / the kernel's duration inside the timed region: its share of "
                                   "the per-kernel CUDA-event times (instrumented pass of one step, no graph replay, right after the timed "
                                   "region) x the iteration time of the timed region itself; these add up to iteration.us.  "
                                   "*_instrumented divides by the event-pair time of the instrumented pass as it is (launch gaps serialised, "
                                   "sum_of_kernel_us_instrumented per iteration)",
                "traffic": traffic, "traffic_source": traffic_source, "peak_source": peak_src,
                "note": "2048^2 single image: the 10-plane working set largely stays in the 126 MB L2, the kernels are latency / "
                        "issue-bound, not HBM-bound (DESIGN.md section 6); `frac` divides ALGORITHMIC bytes by time",
                "sum_of_kernel_us_instrumented": round(sum_us, 2),
                "algorithmic_bytes_per_launch": planes[dom] * plane_bytes,
                "iteration": {"planes": iter_planes, "bytes": iter_planes * plane_bytes, "us": round(it_us, 2),
                              "GBps": round(it_gbs, 1), "frac": round(it_gbs / peak, 4), "frac_nominal_8TBs": round(it_gbs / 8000.0, 4),
                              "planes_as_built": round(built_planes, 2),
                              "frac_as_built": round(built_planes * plane_bytes / (it_us * 1e-6) / 1e9 / peak, 4),
                              "backtracks_per_iteration": backtracks / max(1, iters * args.steps)},
                "kernels": per_kernel}

    # ---- e2e: host (pinned) buffers through the one-shot host entry points; copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=npdt)).pin_memory().numpy()
        hg = [pin(a) for a in w["g"]]; hk = [pin(a) for a in w["psf"]]
        hf = torch.empty((ny, nx), dtype=tdt).pin_memory().numpy()

        def e2e_step():
            if w["S"] is not None:
                return B._one_shot("sgp_boundary" if args.alg == "sgp" else "rl_boundary", hg, hk, w["b"], None, opts,
                                   boundary=(w["S"][0], w["S"][1]), host=True, f_out=hf)[1]
            if p == 1:
                return (B.sgp_single if args.alg == "sgp" else B.rl_single)(hg[0], hk[0], w["b"][0], opts=opts, host=True, f_out=hf)[1]
            return (B.sgp_multi if args.alg == "sgp" else B.rl_multi)(hg, hk, w["b"], opts=opts, host=True, f_out=hf)[1]

        e2e_step(); e2e_step()
        sync_all()
        n_e2e = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            re = e2e_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, world, dev)
        sbytes = sum(a.nbytes for a in hg) + sum(a.nbytes for a in hk)
        e2e = {"value": re.iterations * n_e2e * world / dt, "unit": "iterations/s", "h2d_bytes_per_step": sbytes,
               "d2h_bytes_per_step": hf.nbytes, "steps": n_e2e, "ms_per_step": 1e3 * dt / n_e2e,
               "api": "sgp_single_host" if p == 1 and w["S"] is None else ("sgp_boundary_host" if w["S"] is not None else "sgp_multi_host"),
               "includes": "PSF transfer functions, H2D of g and PSF from pinned memory, all iterations, D2H of f; the plan (workspace, "
                           "tables, instantiated graph) is the one the library keeps from the previous one-shot call of the same "
                           "geometry (two untimed warm-up calls precede the timed ones)"}

    # ---- CPU baseline: the oracle on the host cores, bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cores = os.cpu_count() or 1
        os.environ["OMP_NUM_THREADS"] = str(cores)
        ia, ib = 1, 1 + args.cpu_iters
        ta, tb = oracle_time(w, ia, ib)
        per_it = (tb - ta) / (ib - ia)
        cpu = {"value": 1.0 / per_it, "unit": "iterations/s", "cores": cores, "kind": "oracle",
               "sample": f"{args.workload} ({p}x{ny}x{nx}) fp64 oracle: (t({ib} it) - t({ia} it)) / {ib - ia}, start-point phase excluded; "
                         f"t({ia})={ta:.2f}s t({ib})={tb:.2f}s; OpenMP over {cores} threads"}
        if not args.no_cpu_single:
            try:        # SURVEY.md 8(d) "Timing the oracle beside it": (i) single thread and (ii) all cores
                st, stxt = oracle_time_single_thread(args.workload)
                cpu["single_thread"] = {"value": 1.0 / st, "unit": "iterations/s", "cores": 1, "sample": stxt}
            except Exception as e:
                cpu["single_thread"] = {"error": f"{type(e).__name__}: {e}"}

    # ---- in-run comparison: the same iteration on cuFFT + torch kernels (north_star: "cuFFT ... in-run comparison baseline")
    cufft = None
    if rank == 0 and world == 1 and args.alg == "sgp" and w["S"] is None and not args.no_cufft:
        try:
            cufft = cufft_compare(w, dev, tdt, args.cufft_iters)
            cufft["speedup_of_this_library"] = value / cufft["value"]
        except Exception as e:      # a comparison leg must never take the bench line down
            cufft = {"error": f"{type(e).__name__}: {e}"}

    # ---- the other workloads of BASELINE.json configs[4] (north_star's target names 3 x 2048^2 as well; RL timed separately)
    others = None
    if rank == 0 and world == 1 and not args.no_others and args.workload == "C4c" and args.alg == "sgp" and args.dtype == "f32":
        others = []
        for nm, al in (("C4b", "sgp"), ("C4c", "rl"), ("C4b", "rl")):
            try:
                others.append(measure_other(nm, al, max(2, min(args.steps, 3)), dev, peak))
            except Exception as e:
                others.append({"workload": nm, "algorithm": al, "error": f"{type(e).__name__}: {e}"})

    batched = None
    if rank == 0 and world == 1 and not args.no_others and args.workload == "C4c" and args.alg == "sgp" and args.dtype == "f32":
        try:
            batched = measure_batched(64, 3, dev)
        except Exception as e:
            batched = {"error": f"{type(e).__name__}: {e}"}

    if rank == 0:
        line = {"metric": "SGP iterations/s" if args.alg == "sgp" else "RL iterations/s", "value": value, "unit": "iterations/s",
                "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
                "gpixel_iter_per_s": value * ny * nx / 1e9,
                "config": {"workload": desc, "iterations_per_step": iters, "grid": [ny, nx], "images": p, "algorithm": args.alg,
                           "parallelism": "replicas only" if world > 1 else "single GPU",
                           "l2": f"no flush: per-iteration working set {(7 * p + 4) * plane_bytes / 1e6:.0f} MB "
                                 f"({7 * p + 4} planes) vs 126 MB L2",
                           "tile_cols": int(opts.tile_cols), "rows_per_block": int(opts.rows_per_block),
                           "J0_final": J_final, "backtracks": backtracks // args.steps,
                           "fused_linesearch": int(r.fused_linesearch),
                           "path": ("one cluster per problem, whole iteration in one kernel (csrc/small.cuh); the per-kernel table of `roofline` is the "
                                    "launch-per-pass path of the instrumented pass") if int(r.fused_linesearch) == 2 else "launch-per-pass"},
                "clocks": clk.summary(), "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
                "cufft_compare": cufft, "other_workloads": others, "batched_small_grids": batched}
        print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4c", choices=sorted(WORKLOADS))
    ap.add_argument("--alg", default="sgp", choices=["sgp", "rl"])
    ap.add_argument("--dtype", default="f32", choices=["f32", "f64"])
    ap.add_argument("--tile-cols", type=int, default=0)
    ap.add_argument("--rows-per-block", type=int, default=0)
    ap.add_argument("--cpu-iters", type=int, default=5, help="oracle iterations timed for cpu_baseline")
    ap.add_argument("--ref-iters", type=int, default=3, help="oracle iterations per step of --impl reference")
    ap.add_argument("--graph", type=int, default=1, help="1 = replay the iterations as CUDA graphs of 10 (default), 0 = plain launches; +4 / +8 = force the separate / fused line-search kernel (experiment)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-cpu-single", action="store_true", help="skip the single-thread timing of the oracle")
    ap.add_argument("--no-others", action="store_true", help="skip the C4b / RL lines of other_workloads")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT + torch comparison leg")
    ap.add_argument("--cufft-iters", type=int, default=40, help="iterations timed by the cuFFT comparison leg")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
