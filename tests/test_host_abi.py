"""CPU tests (no GPU): the C-ABI library loads and exports every symbol include/sgp.h declares, the host-side
logic that needs no device (option defaults = the paper's values, argument checks, workspace size, error strings),
the seeded input generators, and the multi-rank path of bench.py (replicas only) on the gloo backend, world size 2."""
import ctypes as C
import json
import os
import re
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

from paper_1210_2258_b200 import binding as B  # noqa: E402
from paper_1210_2258_b200 import synth  # noqa: E402


@pytest.fixture(scope="module")
def lib():
    B.build()
    return B.lib()


def declared_functions():
    """names of the functions include/sgp.h declares"""
    txt = (ROOT / "include" / "sgp.h").read_text()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    names = re.findall(r"^(?:int|void|size_t|const char \*)\s*\*?\s*((?:sgp|rl|osem)_\w+)\s*\(", txt, flags=re.M)
    return sorted(set(names))


def test_library_exports_every_declared_symbol(lib):
    names = declared_functions()
    assert len(names) >= 31
    for n in names:
        assert hasattr(lib, n), f"libsgp_b200.so does not export {n}"
    assert sorted(B.EXPORTS) == names, "binding.EXPORTS and include/sgp.h disagree"


def test_option_defaults_are_the_papers(lib):
    o = B.default_options()
    # PAPER.md:271 (Sect. 3.2): beta = 1e-4, theta = 0.4, alpha_0 = 1.3, tau_1 = 0.5, alpha_max = 1e5, M_alpha = 3, alpha_min = 1e-5
    assert (o.beta, o.theta, o.alpha0, o.tau1, o.alpha_max, o.m_alpha, o.alpha_min) == (1e-4, 0.4, 1.3, 0.5, 1e5, 3, 1e-5)
    assert o.alt_start == 20                       # alternation after the first 20 iterations
    assert o.armijo_memory == 1                    # monotone line search
    assert o.adaptive_L == 1
    assert o.disc_threshold == 1.0 and o.max_backtracks == 30 and o.sigma_R == 1e-2      # readings A7, A16, A13
    assert o.rl_relax == 1.0 and o.rl_linear == 1.0        # plain RL (Eq.1) unless Eq.3 / Eq.4 is asked for


def test_strings_and_workspace(lib):
    lib.sgp_version.restype = C.c_char_p
    lib.sgp_strerror.restype = C.c_char_p
    assert b"sm_100a" in lib.sgp_version()
    msgs = {lib.sgp_strerror(c) for c in range(0, -10, -1)}
    assert len(msgs) >= 9 and all(m for m in msgs)
    lib.sgp_workspace_bytes.restype = C.c_size_t
    lib.sgp_workspace_bytes.argtypes = [C.c_int] * 5
    w1 = lib.sgp_workspace_bytes(B.KIND_SINGLE, 1, 2048, 2048, B.F32)
    w3 = lib.sgp_workspace_bytes(B.KIND_MULTI, 3, 2048, 2048, B.F32)
    w64 = lib.sgp_workspace_bytes(B.KIND_SINGLE, 1, 2048, 2048, B.F64)
    plane = 2048 * 2048 * 4
    assert 11 * plane <= w1 <= 12 * plane          # 7p + 4 planes + tables (q is double-buffered)
    assert 25 * plane <= w3 <= 26 * plane
    assert abs(w64 / w1 - 2.0) < 0.01
    assert lib.sgp_workspace_bytes(B.KIND_SINGLE, 1, 100, 100, B.F32) == 0       # unsupported size
    assert lib.sgp_workspace_bytes(B.KIND_SINGLE, 0, 256, 256, B.F32) == 0


def test_plan_create_rejects_bad_arguments_before_touching_the_device(lib):
    lib.sgp_plan_create.restype = C.c_int
    plan = C.c_void_p()
    o = B.default_options()

    def create(kind, p, ny, nx, oy=0, ox=0, sy=0, sx=0, dtype=B.F32, opt=o):
        return lib.sgp_plan_create(C.byref(plan), kind, p, ny, nx, oy, ox, sy, sx, dtype, C.byref(opt) if opt is not None else None)

    assert create(B.KIND_SINGLE, 1, 100, 256) == B.ERR_ARG            # size not of the form 2^a 5^b within 64..4096
    assert create(B.KIND_SINGLE, 2, 256, 256) == B.ERR_ARG            # single image means p = 1
    assert create(B.KIND_MULTI, 0, 256, 256) == B.ERR_ARG
    assert create(B.KIND_BOUNDARY, 1, 320, 320, 100, 100, 256, 256) == B.ERR_ARG   # S sticks out of S-bar
    assert create(B.KIND_SINGLE, 1, 256, 256, dtype=7) == B.ERR_ARG
    bad = B.default_options(); bad.theta = 1.5
    assert create(B.KIND_SINGLE, 1, 256, 256, opt=bad) == B.ERR_ARG
    bad = B.default_options(); bad.adaptive_L = 0; bad.L1 = 2.0; bad.L2 = 1.0
    assert create(B.KIND_SINGLE, 1, 256, 256, opt=bad) == B.ERR_ARG
    bad = B.default_options(); bad.rl_linear = 0.0                    # Eq.4: lambda_k > 0
    assert create(B.KIND_SINGLE, 1, 256, 256, opt=bad) == B.ERR_ARG
    bad = B.default_options(); bad.rl_linear = 1.2; bad.rl_relax = 1.2   # Eq.3 and Eq.4 are alternatives
    assert create(B.KIND_SINGLE, 1, 256, 256, opt=bad) == B.ERR_ARG
    assert plan.value is None


def test_binding_fails_loudly_without_the_library(tmp_path, monkeypatch):
    """no CPU fallback: a missing library is an error, never a silent detour"""
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_1210_2258_b200 import binding as B\n"
            "B._LIB = None; B.LIB_PATH = B.Path(%r)\n"
            "try:\n    B.lib()\nexcept Exception as e:\n    print('RAISED', type(e).__name__)\n") % (str(ROOT), str(tmp_path / "nope.so"))
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, cwd=tmp_path)
    assert "RAISED" in out.stdout, out.stdout + out.stderr


# ------------------------------------------------------------------------------------------------ generators
@pytest.mark.parametrize("cfg,kw,p", [("C0", {}, 1), ("C1", dict(n=128), 1), ("C2", dict(n=64), 3),
                                      ("C3", dict(s=64, sbar=128, n_stars=20, fwhm=8.0), 1)])
def test_synth_is_seeded_and_well_formed(cfg, kw, p):
    a, b = synth.make(cfg, **kw), synth.make(cfg, **kw)
    assert len(a["g"]) == len(a["psf"]) == len(a["b"]) == p
    for ga, gb, k in zip(a["g"], b["g"], a["psf"]):
        np.testing.assert_array_equal(ga, gb)                  # same seed, same data
        assert ga.min() >= 0 and np.all(ga == np.round(ga))    # Poisson counts
        assert k.min() >= 0 and abs(k.sum() - 1.0) < 1e-9      # PSF normalised to unit volume
        cy, cx = np.unravel_index(np.argmax(k), k.shape)
        assert abs(cy - k.shape[0] // 2) <= 1 and abs(cx - k.shape[1] // 2) <= 1    # centred (A18)
    if a["S"] is not None:
        oy, ox, sy, sx = a["S"]
        assert a["g"][0].shape == (sy, sx) and a["psf"][0].shape[0] >= oy + sy
    # mean counts are consistent with "object flux + background"
    assert a["g"][0].mean() > a["b"][0]


# ------------------------------------------------------------------------------------------------ N > 1 (gloo)
_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch.distributed as dist
import bench
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank, world = dist.get_rank(), dist.get_world_size()
w, _ = bench.make_workload("C0", rank)
ms_local = 10.0 * (rank + 1)                      # rank 1 is the slow one
value, ms = bench.whole_job_rate(ms_local, 100, 2, world)
print(json.dumps({"rank": rank, "value": value, "ms": ms, "gsum": float(w["g"][0].sum())}))
dist.destroy_process_group()
"""


def test_replicas_only_aggregation_world_size_2(tmp_path):
    """bench.py --gpus N: independent replicas (another seed per rank), time = max over ranks, value = whole job"""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % str(ROOT))
    env = {**os.environ, "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": "29611", "WORLD_SIZE": "2"}
    procs = [subprocess.Popen([sys.executable, str(script)], env={**env, "RANK": str(r)}, stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = []
    for pr in procs:
        so, se = pr.communicate(timeout=300)
        assert pr.returncode == 0, se
        outs.append(json.loads(so.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    assert outs[0]["ms"] == outs[1]["ms"] == 20.0                       # the slowest rank's time, on every rank
    assert outs[0]["value"] == outs[1]["value"] == 100 * 2 * 2 / 20e-3  # iterations of BOTH replicas / that time
    assert outs[0]["gsum"] != outs[1]["gsum"]                           # rank 1 works on its own replica


def test_reference_arm_runs_on_rank_0_only():
    env = {**os.environ, "RANK": "1", "WORLD_SIZE": "2"}
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_cufft_comparison_leg_computes_the_same_iteration_as_the_oracle():
    """bench.py's in-run comparison baseline (torch.fft + torch elementwise, run here on the CPU in fp64) is a third
    statement of Algorithm 1: after 25 iterations its J0 must agree with the oracle's trace (C0, M = 10, fixed L; and
    a 3-image problem with the adaptive bounds of PAPER.md:273-275)."""
    import torch
    import bench
    import oracle
    for cfg, kw in (("C0", {}), ("C2", {"n": 128})):
        w = synth.make(cfg, **kw)
        r = bench.cufft_compare(w, "cpu", torch.float64, 20, warm=5)
        oo = oracle.default_options(**{**w["opts"], "max_iter": 25, "stop_rule": 0})
        P = oracle.Problem(w["psf"], masked=False, S=None, sigma_R=oo.sigma_R)
        ge = P.embed(w["g"]); be = [np.full((P.ny, P.nx), float(v)) for v in w["b"]]
        _, ro = P.sgp(ge, be, opts=oo)
        assert ro.iterations == 25
        assert abs(r["J0"] - ro.J0_final) <= 1e-6 * abs(ro.J0_final), (cfg, r["J0"], ro.J0_final)
