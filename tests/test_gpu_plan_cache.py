"""The plan the one-shot entry points keep between calls (include/sgp.h, "Each host thread keeps the plan of its last one-shot
call"): results do not depend on whether the plan was found or created, a new PSF is transformed in every call, another
geometry replaces the plan, and sgp_release_cached_plans gives the device memory back."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1210_2258_b200 import binding as B  # noqa: E402
from paper_1210_2258_b200 import synth  # noqa: E402

from test_gpu_parity import _need_gpu, dev  # noqa: E402


def _plan_path(w, dt, opts, psf=None):
    plan = B.Plan([dev(k, dt) for k in (psf or w["psf"])], S=w["S"], opts=opts)
    f, r = plan.sgp([dev(a, dt) for a in w["g"]], w["b"], opts=opts)
    plan.close()
    return f, r


@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_one_shot_calls_reuse_their_plan(dt):
    _need_gpu()
    B.release_cached_plans()
    w = synth.make("C0", n=256)
    o = B.default_options(**{**w["opts"], "max_iter": 25})
    g, k = dev(w["g"][0], dt), dev(w["psf"][0], dt)
    want, rw = _plan_path(w, dt, o)
    f1, r1 = B.sgp_single(g, k, w["b"][0], opts=o)               # creates the plan
    f2, r2 = B.sgp_single(g, k, w["b"][0], opts=o)               # finds it
    assert torch.equal(f1, want) and torch.equal(f2, want)
    assert r1.iterations == r2.iterations == rw.iterations and r1.J0_final == r2.J0_final == rw.J0_final
    assert r1.kernel_launches == r2.kernel_launches > 0
    # same geometry, another PSF (wider) and another algorithm: the transfer function is rebuilt in the call
    yy, xx = np.mgrid[:256, :256]
    psf2 = np.exp(-((yy - 128.0) ** 2 + (xx - 128.0) ** 2) / (2 * 3.0 ** 2))
    want2, _ = _plan_path(w, dt, o, psf=[psf2])
    f3, _ = B.sgp_single(g, dev(psf2, dt), w["b"][0], opts=o)
    assert torch.equal(f3, want2) and not torch.equal(f3, want)
    fr1, _ = B.rl_single(g, k, w["b"][0], opts=o)
    fr2, _ = B.rl_single(g, k, w["b"][0], opts=o)
    assert torch.equal(fr1, fr2) and not torch.equal(fr1, f1)
    # host-pointer variant: same numbers
    hf = np.empty((256, 256), dt)
    fh, rh = B.sgp_single(np.ascontiguousarray(w["g"][0], dt), np.ascontiguousarray(w["psf"][0], dt), w["b"][0], opts=o, host=True, f_out=hf)
    assert np.array_equal(np.asarray(fh), want.cpu().numpy())
    # another geometry replaces the plan; a boundary problem after it
    w3 = synth.make("C0r", ny=128, nx=320)
    o3 = B.default_options(**{**w3["opts"], "max_iter": 10})
    want3, _ = _plan_path(w3, dt, o3)
    f4, _ = B.sgp_single(dev(w3["g"][0], dt), dev(w3["psf"][0], dt), w3["b"][0], opts=o3)
    assert torch.equal(f4, want3)
    w4 = synth.make("C3", s=64, sbar=128, n_stars=30, max_iter=8, fwhm=8.0)
    o4 = B.default_options(**w4["opts"])
    want4, _ = _plan_path(w4, dt, o4)
    for _ in range(2):
        f5, r5 = B.sgp_boundary([dev(a, dt) for a in w4["g"]], [dev(a, dt) for a in w4["psf"]], w4["b"], w4["S"][0], w4["S"][1], opts=o4)
        assert torch.equal(f5, want4)
    f6, _ = B.sgp_single(g, k, w["b"][0], opts=o)                # and back
    assert torch.equal(f6, want)
    B.release_cached_plans()


def test_release_cached_plans_returns_the_memory():
    _need_gpu()
    B.release_cached_plans()
    w = synth.make("C0", n=1024)
    o = B.default_options(**{**w["opts"], "max_iter": 3})
    g, k = dev(w["g"][0], np.float32), dev(w["psf"][0], np.float32)
    out = torch.empty_like(g)                                       # so that torch's own allocator is not part of the measurement
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    B.sgp_single(g, k, w["b"][0], opts=o, f_out=out)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    ws = B.lib().sgp_workspace_bytes(B.KIND_SINGLE, 1, 1024, 1024, B.F32)
    assert free0 - free1 >= 11 * 1024 * 1024 * 4, (free0, free1)     # the plan (7p + 4 planes and more) is still there
    B.release_cached_plans()
    torch.cuda.synchronize()
    free2 = torch.cuda.mem_get_info()[0]
    assert free2 - free1 >= 11 * 1024 * 1024 * 4 and free0 - free2 < 8 * 1024 * 1024, (free0, free1, free2, ws)
    B.release_cached_plans()                                        # nothing to free: a no-op


def test_mosaic_keeps_its_sub_domain_plan_between_calls():
    """sgp_mosaic keeps the batched sub-domain plan and the sub-image buffers of the calling thread's last call: repeated calls give
    the same bits (also after a call with another geometry in between, which replaces the plan), other data of the same geometry
    give that data's result, and sgp_release_cached_plans returns the memory"""
    _need_gpu()
    B.release_cached_plans()
    dt = np.float32
    w = synth.make("C1", n=256, max_iter=8, stop_rule=0)
    w2 = synth.make("C1", n=256, seed_idx=9, max_iter=8, stop_rule=0)
    o = B.default_options(**{**w["opts"], "max_iter": 8, "stop_rule": 0})
    run = lambda x, sub: B.mosaic(B.ALG_SGP, [dev(a, dt) for a in x["g"]], [dev(k, dt) for k in x["psf"]], x["b"], 2, 2, sub, opts=o)[0]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    m1 = run(w, (160, 160))
    free1 = torch.cuda.mem_get_info()[0]
    assert free0 - free1 >= 4 * 11 * 256 * 256 * 4                  # four sub-domain workspaces are still there
    m2 = run(w, (160, 160))
    assert torch.equal(m1, m2)
    other = run(w2, (160, 160))
    assert not torch.equal(other, m1)
    m3 = run(w, (144, 144))                                         # another window: a new plan
    assert not torch.equal(m3, m1)
    m4 = run(w, (160, 160))
    assert torch.equal(m4, m1)
    B.release_cached_plans()
    fresh = run(w2, (160, 160))                                     # and a plan created afresh gives what the kept one gave
    assert torch.equal(fresh, other)
    B.release_cached_plans()
    torch.cuda.synchronize()
    assert free0 - torch.cuda.mem_get_info()[0] < 8 * 1024 * 1024
