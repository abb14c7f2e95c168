"""Pins P15..P19: the parts of the CPU oracle added in round 2 (start points, data cleaning, refresh_every,
flux-constrained projection, Eq.25 stop, Gaussian-smoothed start, mosaic), checked against what the paper and the
mathematics fix -- never against the oracle's own formulas and never against the CUDA path.  All CPU.
"""
import itertools
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

import oracle
from paper_1210_2258_b200 import synth

ROOT = Path(__file__).resolve().parents[1]
RNG = np.random.default_rng(20121023)


def _psf(ny, nx, rng, width=1.5):
    y = np.arange(ny)[:, None] - ny // 2
    x = np.arange(nx)[None, :] - nx // 2
    k = np.exp(-(y * y + x * x) / (2 * width * width)) * (1.0 + 0.3 * rng.random((ny, nx)))
    return k / k.sum()


def _problem(ny=12, nx=10, p=1, S=None, rng=RNG, b=3.0, flux=300.0, sigma_R=1e-3):
    psfs = [_psf(ny, nx, rng, 1.0 + 0.4 * j) for j in range(p)]
    P = oracle.Problem(psfs, masked=S is not None, S=S, sigma_R=sigma_R)
    info = P.info()
    truth = flux * rng.random((ny, nx)) ** 3 * info["MR"]
    oy, ox, sy, sx = P.S
    MS = np.zeros((ny, nx)); MS[oy:oy + sy, ox:ox + sx] = 1
    g = [rng.poisson(q + b) * MS for q in P.all_A(truth)]
    bb = [np.full((ny, nx), b) for _ in range(p)]
    return P, g, bb, truth, MS, info


# ---------------------------------------------------------------------------------- P15: start points
@pytest.mark.parametrize("p,S", [(1, None), (3, None), (1, (2, 1, 8, 7)), (2, (1, 2, 9, 6))])
def test_P15_start_points_written_out(p, S):
    """max_iter = 0 returns f(0): the null image, the noisy image g_1, the constant image (background-subtracted mean
    flux per pixel, on R only with boundary correction) and a user image, each written out here in numpy."""
    P, g, bb, truth, MS, info = _problem(p=p, S=S)
    MR = info["MR"].astype(float)
    o = lambda **kw: oracle.default_options(max_iter=0, adaptive_L=0, **kw)
    f, r = P.sgp(g, bb, opts=o(init=oracle.INIT_ZERO))
    assert r.iterations == 0 and np.array_equal(f, np.zeros_like(f))
    f, _ = P.sgp(g, bb, opts=o(init=oracle.INIT_G))
    assert np.array_equal(f, np.maximum(g[0], 0) * MS * MR)                 # g_1, "the first PSF K_1"
    if p > 1:
        assert not np.array_equal(f, np.maximum(g[1], 0) * MS * MR)
    f, _ = P.sgp(g, bb, opts=o(init=oracle.INIT_CONST))
    c = max(0.0, np.mean([((gj - bj) * MS).sum() / MS.sum() for gj, bj in zip(g, bb)]))
    assert np.allclose(f, c * MR, rtol=1e-14, atol=0)
    if S is not None:
        assert (f[MR == 0] == 0).all() and MR.sum() > MS.sum()              # "only the pixels in the object array R"
    u = 5.0 + RNG.random(f.shape)
    f, _ = P.sgp(g, bb, f0=u, opts=o(init=oracle.INIT_USER))
    assert np.array_equal(f, u * MR)
    u[3, 3] = -1e-3                                                          # "any non-negative image is allowed"
    _, r = P.sgp(g, bb, f0=u, opts=o(init=oracle.INIT_USER), check=False)
    assert r.rc == -3
    _, r = P.sgp(g, bb, f0=None, opts=o(init=oracle.INIT_USER), check=False)
    assert r.rc == -1
    # the same start points serve RL and OSEM
    f, _ = P.rl(g, bb, opts=o(init=oracle.INIT_G))
    assert np.array_equal(f, np.maximum(g[0], 0) * MS * MR)
    f, _ = P.osem(g, bb, opts=o(init=oracle.INIT_CONST))
    assert np.allclose(f, c * MR, rtol=1e-14, atol=0)


def test_P15_negative_data_are_clamped_unless_strict():
    """reading A17: g < 0 (possible after background subtraction by the caller) is taken as 0; strict = 1 refuses it.
    A run on data with negative pixels equals, bit for bit, the run on the data clamped by numpy; values outside S are ignored."""
    P, g, bb, truth, MS, info = _problem(S=(2, 1, 8, 7))
    gn = [a.copy() for a in g]
    gn[0][4, 4] = -7.0; gn[0][5, 2] = -0.5
    gn[0][0, 0] = -3.0                                                       # outside S: never read
    o = oracle.default_options(max_iter=6)
    for run in (P.sgp, P.rl, P.osem):
        fa, ra = run(gn, bb, opts=o)
        gc = [np.maximum(a, 0) for a in gn]
        fb, rb = run(gc, bb, opts=o)
        assert np.array_equal(fa, fb) and ra.J0_final == rb.J0_final
        _, r = run(gn, bb, opts=oracle.default_options(max_iter=6, strict=1), check=False)
        assert r.rc == -3
    gx = [a.copy() for a in g]; gx[0][4, 4] = np.nan
    _, r = P.sgp(gx, bb, opts=o, check=False)
    assert r.rc == -3


def test_P15_refresh_every_recomputes_Af_and_measures_the_drift():
    """reading A21: q <- q + lambda u is A f(k+1) in exact arithmetic.  With refresh_every = 1 the carried q is replaced
    by A f after every step: the J trace must then be J0 evaluated from f itself (Eq.2 through Eq.16 only), and the
    run without refresh must stay within rounding of it; drift over 200 iterations is reported."""
    P, g, bb, truth, MS, info = _problem(ny=16, nx=16, p=2)
    o1 = oracle.default_options(max_iter=12, refresh_every=1)
    f1, r1 = P.sgp(g, bb, opts=o1)
    assert abs(r1.J0_final - P.J0_of_f(f1, g, bb)) <= 1e-13 * r1.J0_final   # J of the last iterate recomputed from f
    o0 = oracle.default_options(max_iter=12)
    f0, r0 = P.sgp(g, bb, opts=o0)
    assert np.allclose(r0.J, r1.J, rtol=1e-11) and np.allclose(f0, f1, rtol=0, atol=1e-9 * f1.max())
    assert abs(r0.J0_final - P.J0_of_f(f0, g, bb)) <= 1e-12 * r0.J0_final   # the carried q is A f to rounding
    # refresh every 5: J(5), J(10) are recomputed values, the iterations in between carry q
    f5, r5 = P.sgp(g, bb, opts=oracle.default_options(max_iter=10, refresh_every=5))
    assert abs(r5.J[10] - P.J0_of_f(f5, g, bb)) <= 1e-13 * r5.J[10]
    assert r5.n_fft2 == 10 * (2 * 2 + 2) + 2 * (2 + 1)                      # each refresh costs p + 1 transforms more
    # drift of the carried q over 200 iterations (fp64): reported, bounded well below the fp32 tolerances
    fl, rl = P.sgp(g, bb, opts=oracle.default_options(max_iter=200))
    drift = abs(rl.J0_final - P.J0_of_f(fl, g, bb)) / rl.J0_final
    print(f"drift of J0 from the carried q after 200 iterations (fp64): {drift:.2e}")
    assert drift <= 1e-10


def test_P15_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    """the oracle built with -fsanitize=address,undefined runs SGP / RL / OSEM, masked and unmasked, flux projection,
    smoothed start and the Eq.25 stop without a report (sanitizers)"""
    exe = tmp_path / "oracle_asan"
    src = ROOT / "tests" / "oracle_sanitize_main.c"
    cmd = ["gcc", "-std=c99", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
           "-fno-omit-frame-pointer", "-Wno-unknown-pragmas", "-I", str(ROOT / "oracle"), str(src),
           str(ROOT / "oracle" / "sgp_oracle.c"), "-lm", "-o", str(exe)]
    subprocess.run(cmd, check=True)
    r = subprocess.run([str(exe)], capture_output=True, text=True, env={"ASAN_OPTIONS": "detect_leaks=1"})
    assert r.returncode == 0, r.stdout + r.stderr
    assert "ERROR" not in r.stderr and "runtime error" not in r.stderr
    assert "sanitize-run ok" in r.stdout


# ---------------------------------------------------------------------------------- P16: flux-constrained projection
def _project_flux_bruteforce(x, D, c):
    """min sum (y - x)^2 / D  s.t. y >= 0, sum y = c, by enumeration of the active sets: for a set A of free indices
    the stationary point is y_A = x_A - mu D_A with mu = (sum x_A - c) / sum D_A; keep the feasible one of least cost."""
    n = len(x)
    best, besty = np.inf, None
    for m in range(1, n + 1):
        for A in itertools.combinations(range(n), m):
            A = list(A)
            mu = (x[A].sum() - c) / D[A].sum()
            y = np.zeros(n); y[A] = x[A] - mu * D[A]
            if (y < -1e-13).any():
                continue
            cost = (((y - x) ** 2) / D).sum()
            if cost < best - 1e-13:
                best, besty = cost, y
    return np.maximum(besty, 0), best


def test_P16_flux_projection_bruteforce():
    """PAPER.md:60, :68 (Bonettini et al. 2009): the projection on { y >= 0, sum y = c } in the metric D^-1 against an
    enumeration of all active sets on vectors of length <= 6, incl. mu < 0 (c larger than the flux of x) and ties"""
    rng = np.random.default_rng(16)
    for trial in range(300):
        n = int(rng.integers(2, 7))
        x = rng.normal(size=n) * 3
        D = 0.1 + rng.random(n) * 3
        c = float(rng.choice([0.3, 1.0, 5.0, 40.0]))
        if trial % 7 == 0:
            x[1] = x[0]; D[1] = D[0]
        y, mu = oracle.project_flux(x, D, c)
        yb, cost_b = _project_flux_bruteforce(x, D, c)
        assert (y >= 0).all() and abs(y.sum() - c) <= 1e-12 * max(1.0, c)
        assert np.allclose(y, yb, atol=1e-10), (x, D, c, y, yb)
        assert np.allclose(y, np.maximum(0, x - mu * D), atol=1e-13)
    # D = 0 marks pixels outside R: they stay at 0 and carry no flux
    y, mu = oracle.project_flux([3.0, 9.0, 1.0], [1.0, 0.0, 1.0], 2.0)
    assert y[1] == 0 and abs(y.sum() - 2.0) < 1e-14
    # when c equals the flux of P+(x), the constraint is inactive: mu = 0 and the result is max(0, x) (Eq.6)
    x = np.array([2.0, -1.0, 0.5, 3.0]); D = np.array([1.0, 2.0, 0.5, 1.0])
    y, mu = oracle.project_flux(x, D, np.maximum(x, 0).sum())
    assert abs(mu) < 1e-15 and np.array_equal(y, np.maximum(x, 0))


@pytest.mark.parametrize("p,S", [(1, None), (2, None), (1, (2, 1, 8, 7))])
def test_P16_flux_constrained_sgp_keeps_the_flux_and_decreases_J(p, S):
    """with the flux constraint every iterate has sum_R f(k) = c (f(0) is rescaled to it, and f + lambda d is a
    convex combination of two points of the constraint set); J0 still decreases monotonically (M = 1)"""
    P, g, bb, truth, MS, info = _problem(p=p, S=S)
    c_default = max(0.0, sum(((gj - bj) * MS).sum() for gj, bj in zip(g, bb)) / p)
    for c, kw in ((c_default, {}), (1234.5, {"flux_value": 1234.5})):
        fs = []
        for k in (0, 1, 2, 7, 25):
            f, r = P.sgp(g, bb, opts=oracle.default_options(max_iter=k, flux_constraint=1, **kw))
            assert abs(f.sum() - c) <= 1e-10 * c and (f >= 0).all() and (f[info["MR"] == 0] == 0).all()
            fs.append(f)
        assert np.all(np.diff(r.J) < 0)
    # unconstrained run from the same data does not keep it
    f, r = P.sgp(g, bb, opts=oracle.default_options(max_iter=25))
    assert abs(f.sum() - c_default) > 1e-6 * c_default
    # one constrained step written out: y = argmin over the constraint set, f(1) = f(0) + lambda (y - f(0))
    o1 = oracle.default_options(max_iter=1, flux_constraint=1, adaptive_L=0, L1=1e-5, L2=1e5)
    f0, _ = P.sgp(g, bb, opts=oracle.default_options(max_iter=0, flux_constraint=1, adaptive_L=0, L1=1e-5, L2=1e5))
    f1, r1 = P.sgp(g, bb, opts=o1)
    grad = P.gradient(f0, g, bb)
    Dk = P.scaling(f0, 1e-5, 1e5)
    y, mu = oracle.project_flux(f0 - r1.alpha[0] * Dk * grad, Dk, c_default)
    assert np.allclose(f1, f0 + r1.lam[0] * (y - f0), rtol=0, atol=1e-12 * f0.max())


# ---------------------------------------------------------------------------------- P17: Eq.25
@pytest.mark.parametrize("alg", ["sgp", "rl", "osem"])
def test_P17_minimum_reconstruction_error_stop(alg):
    """Eq.25: rho(k) = ||f(k) - f~||_2 / ||f~||_2 written out in numpy along a free run; the MINERR
    run stops at the first k whose next step would increase rho and returns exactly f(k) of the free run"""
    rng = np.random.default_rng(17)
    P, g, bb, truth, MS, info = _problem(ny=16, nx=16, p=2, rng=rng, flux=100.0)      # few counts: early semiconvergence
    run = {"sgp": P.sgp, "rl": P.rl, "osem": P.osem}[alg]
    K = 120
    free = [run(g, bb, opts=oracle.default_options(max_iter=k), truth=truth) for k in (K,)][0]
    fK, rK = free
    rho = [np.linalg.norm(run(g, bb, opts=oracle.default_options(max_iter=k))[0] - truth) / np.linalg.norm(truth) for k in range(0, 12)]
    assert np.allclose(rK.err[:12], rho, rtol=1e-13)
    inc = np.nonzero(np.diff(rK.err[:K + 1]) > 0)[0]
    assert len(inc) > 0, "the recipe must show semiconvergence within the free run for this test to mean anything"
    kstar = int(inc[0])
    fm, rm = run(g, bb, opts=oracle.default_options(max_iter=K, stop_rule=oracle.STOP_MINERR), truth=truth)
    assert rm.stop_reason == 4 and rm.iterations == kstar
    fk, rk = run(g, bb, opts=oracle.default_options(max_iter=kstar))
    assert np.array_equal(fm, fk) and rm.J0_final == rk.J0_final
    assert rm.err_final == rK.err[kstar] and rm.err[kstar + 1] == rK.err[kstar + 1] > rm.err_final
    # without the true object the rule cannot be used
    _, r = run(g, bb, opts=oracle.default_options(max_iter=5, stop_rule=oracle.STOP_MINERR), check=False)
    assert r.rc == -1
    assert abs(oracle.rel_error(fk, truth) - np.linalg.norm(fk - truth) / np.linalg.norm(truth)) < 1e-15


# ---------------------------------------------------------------------------------- P18: Gaussian-smoothed constant start
def test_P18_smoothed_constant_start():
    """PAPER.md:264 ("the constant image will be convolved with a Gaussian to avoid the presence of sharp edges", reading
    A28): periodic problems: the smoothed constant IS the constant; boundary problems: M_R o (G_sigma * (c M_R)) with the
    Gaussian and the circular convolution written out here by shifts"""
    P, g, bb, truth, MS, info = _problem(p=2)
    fc, _ = P.sgp(g, bb, opts=oracle.default_options(max_iter=0, init=oracle.INIT_CONST))
    fs, _ = P.sgp(g, bb, opts=oracle.default_options(max_iter=0, init=oracle.INIT_CONST_SMOOTH, init_sigma=1.7))
    assert np.allclose(fs, fc, rtol=1e-13)
    P, g, bb, truth, MS, info = _problem(ny=14, nx=12, S=(3, 2, 8, 7), sigma_R=0.05)
    MR = info["MR"].astype(float)
    ny, nx = MR.shape
    assert 0 < MR.sum() < MR.size
    sig = 1.3
    fc, _ = P.sgp(g, bb, opts=oracle.default_options(max_iter=0, init=oracle.INIT_CONST, sigma_R=0.05))
    fs, _ = P.sgp(g, bb, opts=oracle.default_options(max_iter=0, init=oracle.INIT_CONST_SMOOTH, init_sigma=sig, sigma_R=0.05))
    dy = np.minimum(np.arange(ny), ny - np.arange(ny))[:, None]; dx = np.minimum(np.arange(nx), nx - np.arange(nx))[None, :]
    G = np.exp(-(dy ** 2 + dx ** 2) / (2 * sig * sig)); G /= G.sum()
    conv = sum(G[a, b_] * np.roll(fc, (a, b_), axis=(0, 1)) for a in range(ny) for b_ in range(nx))
    assert np.allclose(fs, np.maximum(conv, 0) * MR, rtol=1e-12, atol=1e-13 * fc.max())
    assert (fs[MR == 0] == 0).all() and fs[MR == 1].min() < fc.max() * 0.999       # the edge of R is no longer sharp
    _, r = P.sgp(g, bb, opts=oracle.default_options(max_iter=0, init=oracle.INIT_CONST_SMOOTH, init_sigma=0.0), check=False)
    assert r.rc == -1


# ---------------------------------------------------------------------------------- P19: mosaic
def test_P19_mosaic_layout_is_the_papers():
    """256 x 256 images, four partially overlapping 160 x 160 subdomains, each zero-padded into a
    256 x 256 array, 128 x 128 non-overlapping images extracted (tests/golden/mosaic_layout.txt)"""
    rows = [l.split() for l in (ROOT / "tests" / "golden" / "mosaic_layout.txt").read_text().splitlines() if l and not l.startswith("#")]
    N, T, s, nbar, part = (int(v) for v in rows[0])
    tiles = oracle.mosaic_layout(N, N, T, T, s, s, nbar, nbar)
    assert len(tiles) == T * T == 4
    cover = np.zeros((N, N), int)
    for t in tiles:
        yi, xi = t["img"]; y0, x0, hy, hx = t["out"]; ys, xs = t["src"]; oy, ox, sy, sx = t["S"]
        assert (hy, hx) == (part, part) and (sy, sx) == (s, s)
        assert 0 <= yi <= N - s and 0 <= xi <= N - s and yi in (0, N - s) and xi in (0, N - s)      # partially overlapping, inside the image
        # the extracted part lies inside the sub-image, and maps back to the right image pixels
        assert oy <= ys and ys + hy <= oy + sy and ox <= xs and xs + hx <= ox + sx
        assert (ys - oy + yi, xs - ox + xi) == (y0, x0)
        cover[y0:y0 + hy, x0:x0 + hx] += 1
    assert (cover == 1).all()                                                                     # non-overlapping, complete


def test_P19_mosaic_tiles_are_independent_and_free_of_boundary_effects():
    """each sub-domain is reconstructed from its own sub-image only; and the mosaic agrees with the
    reconstruction of the full image while a reconstruction of the sub-images WITHOUT boundary correction does not
    ("the mosaic of the four reconstructions does not exhibit visible boundary effects")"""
    rng = np.random.default_rng(19)
    N, s = 32, 20
    psf = synth.psf_gaussian(N, N, 3.0)
    truth = 200.0 * rng.random((N, N)) ** 2 + 50.0
    blur = np.fft.irfft2(np.fft.rfft2(np.fft.ifftshift(psf)) * np.fft.rfft2(truth), s=(N, N))
    g = [blur + 5.0]                                                       # noiseless: differences are boundary effects only
    o = oracle.default_options(max_iter=30, sigma_R=1e-2)
    m, res = oracle.mosaic("rl", g, [psf], [5.0], 2, 2, (s, s), o)
    full, _ = oracle.rl_single(g[0], psf, 5.0, None, o)
    # compared away from the outer frame of the image, where the full reconstruction sees the periodic wrap-around of
    # this synthetic image and the sub-domain reconstructions (rightly) do not
    inner = (slice(4, N - 4), slice(4, N - 4))
    err_mosaic = np.linalg.norm((m - full)[inner]) / np.linalg.norm(full[inner])
    # the same sub-images deconvolved as if periodic (no correction): edge artefacts inside the extracted parts
    naive = np.zeros_like(m)
    for t in oracle.mosaic_layout(N, N, 2, 2, s, s, N, N):
        yi, xi = t["img"]; y0, x0, hy, hx = t["out"]
        pk = synth.psf_gaussian(s, s, 3.0)
        fsub, _ = oracle.rl_single(g[0][yi:yi + s, xi:xi + s], pk, 5.0, None, o)
        naive[y0:y0 + hy, x0:x0 + hx] = fsub[y0 - yi:y0 - yi + hy, x0 - xi:x0 - xi + hx]
    err_naive = np.linalg.norm((naive - full)[inner]) / np.linalg.norm(full[inner])
    print(f"mosaic vs full-image reconstruction: {err_mosaic:.3e}; without boundary correction: {err_naive:.3e}")
    assert err_mosaic < 0.01 and err_naive > 2.5 * err_mosaic
    # independence: data outside sub-image 0 do not touch tile 0
    g2 = [g[0].copy()]; g2[0][s:, :] += 100.0; g2[0][:, s:] += 100.0
    m2, _ = oracle.mosaic("rl", g2, [psf], [5.0], 2, 2, (s, s), o)
    assert np.array_equal(m2[:N // 2, :N // 2], m[:N // 2, :N // 2]) and not np.array_equal(m2, m)
    # the SGP and OSEM drivers run through the same stitching
    ms, rs = oracle.mosaic("sgp", g, [psf], [5.0], 2, 2, (s, s), o)
    assert len(rs) == 4 and all(r.iterations == 30 for r in rs) and np.linalg.norm(ms - full) / np.linalg.norm(full) < 0.05
