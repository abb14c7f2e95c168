"""sgp_rel_error_static (include/sgp.h): the entry point that allocates nothing -- the relative reconstruction error of
Eq.25 with its scratch in a static device array -- against the existing path (the plan's err_kernel,
reported as trace_err[0] of a run that is given the true object and a user start point), on two calls in a row.

Collected last on purpose (the file name): the suite runs with `pytest -x`."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1210_2258_b200 import binding as B  # noqa: E402
from paper_1210_2258_b200 import synth  # noqa: E402


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def _dev(a, dt):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=dt), device="cuda")


def _existing_path(plan, w, g, f, truth):
    """rho(0) of a run that starts from f: err_kernel (extra.cuh) with the plan's workspace as scratch"""
    o = B.default_options(**{**w["opts"], "max_iter": 0, "stop_rule": 0, "init": B.INIT_USER})
    _, r = plan.sgp(g, w["b"], f0=f, opts=o, truth=truth)
    return float(r.err[0])


# (ny, nx): one CTA row short of the grid cap, a 5-smooth grid with a ragged last CTA, and a grid-stride case (n > 1184 x 256)
@pytest.mark.parametrize("dt", [np.float32, np.float64])
@pytest.mark.parametrize("shape", [(256, 256), (200, 320), (1024, 2048)])
def test_rel_error_static_matches_plan_path_twice(shape, dt):
    _need_gpu()
    ny, nx = shape
    w = synth.make("C0r", ny=ny, nx=nx)
    plan = B.Plan([_dev(w["psf"][0], dt)], opts=B.default_options(**w["opts"]))
    g = [_dev(w["g"][0], dt)]
    truth = _dev(w["truth"], dt)
    rng = np.random.default_rng(1210)
    # two different images, so that the second call cannot pass on what the first left in the array
    fa = _dev(np.maximum(w["truth"] * (1.0 + 0.05 * rng.standard_normal((ny, nx))), 0.0) + 1.0, dt)
    fb = _dev(np.full((ny, nx), float(np.mean(w["truth"]))), dt)
    rho = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    got = []
    for f in (fa, fb):                                   # two calls in a row on one stream
        assert B.rel_error_static(f, truth, rho) == B.OK
        got.append(float(rho.item()))
    want = [_existing_path(plan, w, g, f, truth) for f in (fa, fb)]
    plan.close()
    t64 = truth.double().cpu().numpy()
    for f, a, b in zip((fa, fb), got, want):
        # same kernel arithmetic, same grid and reduction order: the tests of the existing path use 1e-9 (fp64) / 2e-4 (fp32)
        # against the oracle; the two device paths agree far inside that
        assert abs(a - b) <= 1e-12 * b, (shape, dt, a, b)
        ref = np.linalg.norm(f.double().cpu().numpy() - t64) / np.linalg.norm(t64)      # the definition, in double
        assert abs(a - ref) <= 1e-9 * ref
    assert got[0] != got[1]


def test_rel_error_static_small_after_large_and_limits():
    """a small call after a large one (the array still holds the large call's partials), then the argument checks: beyond the
    maximum nothing is launched and the error text says why"""
    _need_gpu()
    rng = np.random.default_rng(2258)
    rho = torch.zeros(1, dtype=torch.float64, device="cuda")
    for n in (2048 * 2048, 1000, 1, 4096 * 4096):
        t = _dev(rng.random(n) + 0.5, np.float32)
        f = _dev(rng.random(n) + 0.5, np.float32)
        for _ in range(2):
            assert B.rel_error_static(f, t, rho) == B.OK
            ref = float(torch.linalg.vector_norm(f.double() - t.double()) / torch.linalg.vector_norm(t.double()))
            assert abs(float(rho.item()) - ref) <= 1e-9 * ref, n
        del t, f
    L = B.lib()
    assert L.sgp_rel_error_static_max() == B.STATIC_MAX_ELEMS == 4096 * 4096
    x = torch.ones(16, dtype=torch.float32, device="cuda")
    rho.fill_(-7.0)
    p = C.c_void_p(x.data_ptr())
    rc = L.sgp_rel_error_static(p, p, B.STATIC_MAX_ELEMS + 1, B.F32, C.c_void_p(rho.data_ptr()), None)
    assert rc == B.ERR_ARG and b"exceeds SGP_STATIC_MAX_ELEMS" in L.sgp_last_cuda_error()
    torch.cuda.synchronize()
    assert float(rho.item()) == -7.0                     # nothing ran
    assert L.sgp_rel_error_static(p, p, 0, B.F32, C.c_void_p(rho.data_ptr()), None) == B.ERR_ARG
    assert L.sgp_rel_error_static(None, p, 16, B.F32, C.c_void_p(rho.data_ptr()), None) == B.ERR_ARG
    assert L.sgp_rel_error_static(p, p, 16, 7, C.c_void_p(rho.data_ptr()), None) == B.ERR_ARG
    with pytest.raises(B.SgpError, match="exceeds SGP_STATIC_MAX_ELEMS"):
        big = torch.empty(B.STATIC_MAX_ELEMS + 256, dtype=torch.float32, device="cuda")
        B.rel_error_static(big, big, rho)
