"""Pins P1..P11 of SURVEY.md 8(c): the CPU oracle checked against what the paper and the
mathematics fix (closed forms, invariants, brute force, library routines) -- never against
itself and never against the CUDA path.  All CPU, run with -m "not gpu".
"""
import itertools

import numpy as np
import pytest

import oracle
from paper_1210_2258_b200 import synth

RNG = np.random.default_rng(20121022)


def _rand_psf(ny, nx, rng, width=1.5):
    y = np.arange(ny)[:, None] - ny // 2
    x = np.arange(nx)[None, :] - nx // 2
    k = np.exp(-(y * y + x * x) / (2 * width * width)) * (1.0 + 0.3 * rng.random((ny, nx)))
    return k / k.sum()


def _tiny_problem(ny=8, nx=8, p=1, masked=False, rng=RNG, b=3.0, flux=200.0, S=None):
    psfs = [_rand_psf(ny, nx, rng, 1.0 + 0.4 * j) for j in range(p)]
    P = oracle.Problem(psfs, masked=masked, S=S, sigma_R=1e-3)
    truth = flux * rng.random((ny, nx)) ** 3
    info = P.info()
    truth = truth * info["MR"]
    q = P.all_A(truth)
    oy, ox, sy, sx = P.S
    MS = np.zeros((ny, nx)); MS[oy:oy + sy, ox:ox + sx] = 1
    g = [rng.poisson(qq + b) * MS for qq in q]
    bb = [np.full((ny, nx), b) for _ in range(p)]
    return P, g, bb, truth, MS


# ---------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("shape", [(16, 16), (8, 20), (10, 16), (5, 7), (1, 12), (40, 10)])
def test_P1_fft_vs_direct_dft_and_numpy(shape):
    ny, nx = shape
    x = RNG.normal(size=shape) + 1j * RNG.normal(size=shape)
    X = oracle.fft2(x, -1)
    # the definition, written out as DFT matrices
    Fy = np.exp(-2j * np.pi * np.outer(np.arange(ny), np.arange(ny)) / ny)
    Fx = np.exp(-2j * np.pi * np.outer(np.arange(nx), np.arange(nx)) / nx)
    assert np.abs(X - Fy @ x @ Fx).max() <= 1e-12 * max(1, np.abs(X).max())
    assert np.abs(X - np.fft.fft2(x)).max() <= 1e-12 * max(1, np.abs(X).max())
    # inverse incl. 1/(ny nx), round trip
    assert np.abs(oracle.fft2(X, +1) - x).max() <= 1e-13
    assert np.abs(oracle.fft2(x, +1) - np.fft.ifft2(x)).max() <= 1e-13
    # Parseval
    assert np.isclose((np.abs(X) ** 2).sum(), ny * nx * (np.abs(x) ** 2).sum(), rtol=1e-12)


@pytest.mark.parametrize("n", [1280 // 16, 5 * 16, 3 * 5 * 4, 64])
def test_P1_fft_radix5_lengths_and_delta(n):
    d = np.zeros((4, n)); d[0, 0] = 1.0
    assert np.abs(oracle.fft2(d) - 1.0).max() <= 1e-14          # delta -> ones
    x = RNG.normal(size=(4, n))
    assert np.abs(oracle.fft2(x) - np.fft.fft2(x)).max() <= 1e-11


def test_P1_fft_convolution_vs_direct_16():
    ny = nx = 16
    psf = _rand_psf(ny, nx, RNG)
    x = RNG.random((ny, nx)) * 10
    P = oracle.Problem([psf])
    K0 = np.fft.ifftshift(psf)                                     # origin moved to (0,0), A18
    direct = oracle.conv2_direct(K0, x)
    assert np.abs(P.A(0, x) - direct).max() <= 1e-12 * np.abs(direct).max()
    # direct convolution itself against the definition in numpy
    ref = np.zeros_like(x)
    for my, mx in itertools.product(range(ny), range(nx)):
        for qy, qx in itertools.product(range(ny), range(nx)):
            ref[my, mx] += K0[(my - qy) % ny, (mx - qx) % nx] * x[qy, qx]
    assert np.abs(direct - ref).max() <= 1e-12 * np.abs(ref).max()
    # A^T = correlation: direct form
    corr = np.zeros_like(x)
    for ny_, nx_ in itertools.product(range(ny), range(nx)):
        for my, mx in itertools.product(range(ny), range(nx)):
            corr[ny_, nx_] += K0[(my - ny_) % ny, (mx - nx_) % nx] * x[my, mx]
    assert np.abs(P.AT(0, x) - corr).max() <= 1e-12 * np.abs(corr).max()


@pytest.mark.parametrize("shape", [(12, 10), (11, 9), (7, 12)])
@pytest.mark.parametrize("origin", [oracle.PSF_CENTER, oracle.PSF_CORNER])
def test_P1_delta_psf_is_identity(origin, shape):
    ny, nx = shape
    psf = np.zeros((ny, nx))
    if origin == oracle.PSF_CENTER:
        psf[ny // 2, nx // 2] = 7.0      # any positive volume: the library normalises (A18)
    else:
        psf[0, 0] = 7.0
    P = oracle.Problem([psf], psf_origin=origin)
    x = RNG.random((ny, nx))
    assert np.abs(P.A(0, x) - x).max() <= 1e-14
    assert np.abs(P.AT(0, x) - x).max() <= 1e-14


def test_P1_psf_shift_direction():
    """an off-centre delta PSF shifts the image the same way the convolution definition does"""
    ny, nx = 8, 8
    psf = np.zeros((ny, nx)); psf[ny // 2 + 2, nx // 2 - 1] = 1.0     # K(m) = delta(m - (2,-1))
    P = oracle.Problem([psf])
    x = RNG.random((ny, nx))
    assert np.abs(P.A(0, x) - np.roll(x, (2, -1), axis=(0, 1))).max() <= 1e-14
    assert np.abs(P.AT(0, x) - np.roll(x, (-2, 1), axis=(0, 1))).max() <= 1e-14


# ---------------------------------------------------------------------------------- P2
@pytest.mark.parametrize("masked,S", [(False, None), (True, (3, 2, 8, 10))])
@pytest.mark.parametrize("p", [1, 3])
def test_P2_adjointness(masked, S, p):
    ny, nx = 14, 16
    psfs = [_rand_psf(ny, nx, RNG, 1.2 + 0.5 * j) for j in range(p)]
    P = oracle.Problem(psfs, masked=masked, S=S, sigma_R=0.05)
    for j in range(p):
        x, y = RNG.normal(size=(ny, nx)), RNG.normal(size=(ny, nx))
        lhs, rhs = (P.A(j, x) * y).sum(), (x * P.AT(j, y)).sum()
        assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), 1.0)
    # the fused forms equal the separate applications of Eq.16 / Eq.17
    x = RNG.normal(size=(ny, nx))
    for j, out in enumerate(P.all_A(x)):
        assert np.abs(out - P.A(j, x)).max() <= 1e-13
    rs = [RNG.normal(size=(ny, nx)) for _ in range(p)]
    assert np.abs(P.sum_AT(rs) - sum(P.AT(j, rs[j]) for j in range(p))).max() <= 1e-13


def test_P2_masks_and_alpha_definition():
    """Eq.19 in reading A5: alpha_j(n) = sum_m K_j(m-n) M_S(m); R by Eq.20; W = M_R/alpha"""
    ny, nx = 12, 12
    S = (2, 3, 7, 6)
    rng = np.random.default_rng(1)
    psfs = [_rand_psf(ny, nx, rng, 0.6), _rand_psf(ny, nx, rng, 3.0)]
    sigma = 0.35
    P = oracle.Problem(psfs, masked=True, S=S, sigma_R=sigma)
    info = P.info()
    MS = np.zeros((ny, nx)); MS[2:9, 3:9] = 1
    alphas = []
    for k in psfs:
        K0 = np.fft.ifftshift(k / k.sum())
        a = np.zeros((ny, nx))
        for n_ in itertools.product(range(ny), range(nx)):
            for m in itertools.product(range(ny), range(nx)):
                a[n_] += K0[(m[0] - n_[0]) % ny, (m[1] - n_[1]) % nx] * MS[m]
        alphas.append(a)
    alpha = sum(alphas)
    MR = np.all([a >= sigma for a in alphas], axis=0)
    assert np.array_equal(info["MR"].astype(bool), MR)
    assert 0 < MR.sum() < ny * nx
    # the rule is "for all j" (Eq.20): it differs here from thresholding alpha_1 alone or the sum
    assert not any(np.array_equal(MR, a >= sigma) for a in (alphas[0], alphas[1], alpha))
    assert np.abs(info["alpha"] - alpha).max() <= 1e-13
    assert np.abs(info["W"] - np.where(MR, 1.0 / alpha, 0.0)).max() <= 1e-12
    assert info["nS"] == 42 and info["nR"] == MR.sum()
    # A_j zeroes outside S and ignores x outside R; A_j^T zeroes outside R
    x = RNG.random((ny, nx))
    assert np.all(P.A(0, x)[MS == 0] == 0)
    assert np.abs(P.A(0, x) - P.A(0, x * MR)).max() <= 1e-14
    assert np.all(P.AT(1, x)[~MR] == 0)


# ---------------------------------------------------------------------------------- P3
@pytest.mark.parametrize("p,masked,S", [(1, False, None), (3, False, None), (1, True, (1, 2, 6, 5)), (2, True, (2, 1, 5, 6))])
def test_P3_gradient_vs_finite_differences(p, masked, S):
    rng = np.random.default_rng(33 + p)
    P, g, b, truth, MS = _tiny_problem(8, 8, p, masked, rng, S=S)
    MR = P.info()["MR"].astype(bool)
    f = (truth + 5.0 + rng.random(truth.shape)) * MR
    grad = P.gradient(f, g, b)
    assert np.all(grad[~MR] == 0)
    num = np.zeros_like(f)
    for idx in zip(*np.nonzero(MR)):
        h = 1e-4 * max(1.0, f[idx])
        fp, fm = f.copy(), f.copy()
        fp[idx] += h; fm[idx] -= h
        num[idx] = (P.J0_of_f(fp, g, b) - P.J0_of_f(fm, g, b)) / (2 * h)
    assert np.abs(grad - num).max() <= 1e-6 * max(1.0, np.abs(num).max())


def test_P3_J0_definition_and_limits():
    """Eq.2 written out in numpy; the g = 0 summand is y; J0(f; g) = 0 iff Af + b = g"""
    ny, nx = 8, 8
    P, g, b, truth, MS = _tiny_problem(ny, nx, 2, False, np.random.default_rng(5))
    g[0][0, :] = 0.0
    f = truth + 1.0
    q = P.all_A(f)
    J = P.J0(q, g, b)
    ref = 0.0
    for j in range(2):
        y = q[j] + b[j]
        with np.errstate(divide="ignore", invalid="ignore"):
            t = np.where(g[j] > 0, g[j] * np.log(g[j] / y), 0.0)
        ref += (t + y - g[j]).sum()
    assert np.isclose(J, ref, rtol=1e-12)
    gz = [qq + bb for qq, bb in zip(q, b)]
    assert abs(P.J0(q, gz, b)) <= 1e-10
    assert J > 0


# ---------------------------------------------------------------------------------- P4
def _rl_formula(P, f, g, b, W):
    w = sum(P.AT(j, np.where(P.A(j, f) + b[j] > 0, g[j] / (P.A(j, f) + b[j]), 0.0)) for j in range(P.p))
    return W * f * w


@pytest.mark.parametrize("p,masked,S", [(1, False, None), (3, False, None), (1, True, (2, 2, 8, 8)), (3, True, (1, 3, 9, 7))])
def test_P4_sgp_with_alpha1_lambda1_is_RL(p, masked, S):
    """SGP with alpha_k = 1, lambda_k = 1, D = W o f is the RL update
    (Eq.1; Eq.13 with W = 1/p; Eq.21 with W = M_R/alpha)."""
    rng = np.random.default_rng(44 + p)
    P, g, b, truth, MS = _tiny_problem(12, 12, p, masked, rng, S=S)
    info = P.info()
    f0 = (1.0 + rng.random((12, 12)) * 50) * info["MR"]
    K = 3
    opts = oracle.default_options(max_iter=K, adaptive_L=0, L1=1e-300, L2=1e300, init=oracle.INIT_USER)
    f_sgp, res = P.sgp(g, b, f0, opts, force_alpha=[1.0] * K, force_lambda=[1.0] * K)
    f_rl = f0.copy()
    for _ in range(K):
        f_rl = _rl_formula(P, f_rl, g, b, info["W"])           # the printed formula, via Eq.16/17 only
    assert np.abs(f_sgp - f_rl).max() <= 1e-12 * np.abs(f_rl).max()
    # and the oracle's own RL entry point does the same
    f_rl2, _ = P.rl(g, b, f0, oracle.default_options(max_iter=K, init=oracle.INIT_USER))
    assert np.abs(f_rl2 - f_rl).max() <= 1e-12 * np.abs(f_rl).max()
    assert np.abs(P.rl_step(f0, g, b) - _rl_formula(P, f0, g, b, info["W"])).max() <= 1e-12 * np.abs(f_rl).max()
    if not masked:
        assert np.all(info["W"] == 1.0 / p) and np.all(info["alpha"] == p)     # A8


# ---------------------------------------------------------------------------------- P5
@pytest.mark.parametrize("p,masked,S", [(1, False, None), (3, False, None), (2, True, (2, 3, 9, 8))])
def test_P5_rl_flux_invariants_b0(p, masked, S):
    """with b = 0 and unit-volume periodic PSFs RL conserves flux:
    sum f(k+1) = sum g (single), (1/p) sum_j sum g_j (multi), sum_R alpha f(k+1) = sum_j sum_S g_j (boundary)."""
    rng = np.random.default_rng(55 + p)
    ny, nx = 14, 12
    psfs = [_rand_psf(ny, nx, rng, 1.0 + 0.6 * j) for j in range(p)]
    P = oracle.Problem(psfs, masked=masked, S=S, sigma_R=0.02)
    info = P.info()
    oy, ox, sy, sx = P.S
    MS = np.zeros((ny, nx)); MS[oy:oy + sy, ox:ox + sx] = 1
    g = [rng.poisson(30 + 100 * rng.random((ny, nx))) * MS for _ in range(p)]
    b = [np.zeros((ny, nx)) for _ in range(p)]
    f = (0.5 + rng.random((ny, nx))) * info["MR"]
    target = sum(gg.sum() for gg in g)
    for _ in range(4):
        f = P.rl_step(f, g, b)
        assert np.isclose((info["alpha"] * f).sum(), target, rtol=1e-12)
        assert np.all(f >= 0)
    if not masked:
        assert np.isclose(f.sum(), target / p, rtol=1e-12)


# ---------------------------------------------------------------------------------- P6
def test_P6_projection_bruteforce():
    """Eq.6: P+ in the metric of D^-1.  The minimiser of sum (y_i - x_i)^2 / D_i over y >= 0 is found by
    enumerating active sets (each y_i is either 0 or free); it must equal the oracle's y."""
    rng = np.random.default_rng(6)
    for n in (1, 2, 3, 5, 6):
        for _ in range(20):
            f = rng.random(n) * 3
            grad = rng.normal(size=n) * 4
            D = 0.1 + rng.random(n) * 5
            alpha = 10 ** rng.uniform(-2, 1)
            x = f - alpha * D * grad
            best, besty = np.inf, None
            for act in itertools.product([0, 1], repeat=n):
                y = np.where(np.array(act) == 1, x, 0.0)
                if np.any(y < 0):
                    continue
                val = ((y - x) ** 2 / D).sum()
                if val < best - 1e-15:
                    best, besty = val, y
            y_or = oracle.project(f, grad, D, alpha)
            assert np.allclose(y_or, besty, atol=1e-14)
            assert np.all(y_or >= 0)


def test_P6_scaling_eq10_eq23():
    ny, nx = 10, 10
    psfs = [_rand_psf(ny, nx, RNG, 1.0), _rand_psf(ny, nx, RNG, 1.5)]
    f = RNG.random((ny, nx)) * 10
    P = oracle.Problem(psfs)                               # unmasked, p = 2: D = clip(f)/p (A8)
    assert np.allclose(P.scaling(f, 2.0, 7.0), np.clip(f, 2.0, 7.0) / 2, rtol=1e-15)
    Pm = oracle.Problem(psfs, masked=True, S=(2, 2, 6, 6), sigma_R=0.1)
    info = Pm.info()
    ref = np.where(info["MR"] > 0, np.clip(f, 2.0, 7.0) / info["alpha"], 0.0)
    assert np.allclose(Pm.scaling(f, 2.0, 7.0), ref, rtol=1e-14)


# ---------------------------------------------------------------------------------- P7
@pytest.mark.parametrize("cfg", ["single", "multi", "boundary"])
def test_P7_iteration_invariants(cfg):
    rng = np.random.default_rng(77)
    if cfg == "single":
        w = synth.c0_stars_gaussian(32)
    elif cfg == "multi":
        w = synth.c2_lbt_multi(32, max_iter=60)
    else:
        w = synth.c3_boundary(24, 32, n_stars=30, max_iter=60)
    masked = w["S"] is not None
    P = oracle.Problem(w["psf"], masked=masked, S=w["S"], sigma_R=1e-2)
    g = P.embed(w["g"]); b = [np.full(P.psfs[0].shape, bj) for bj in w["b"]]
    opts = oracle.default_options(max_iter=60, armijo_memory=1)
    f, res = P.sgp(g, b, None, opts)
    assert res.iterations == 60 and res.stop_reason == 1
    assert np.all(f >= 0)
    assert np.all(f[P.info()["MR"] == 0] == 0)
    # monotone Armijo (M = 1): J(k+1) < J(k)
    assert np.all(np.diff(res.J) < 0)
    assert np.all((res.alpha >= opts.alpha_min) & (res.alpha <= opts.alpha_max))
    assert res.alpha[0] == opts.alpha0 and res.rule[0] == 0
    # lambda in {theta^i}
    i = np.round(np.log(res.lam) / np.log(opts.theta))
    assert np.allclose(res.lam, opts.theta ** i, rtol=1e-12)
    assert np.array_equal(i.astype(int), res.backtracks)
    assert res.total_backtracks == res.backtracks.sum()
    # first 20 iterations use the Eq.9 value (A9)
    assert np.all(res.rule[1:21] == 2)
    assert np.isclose(res.J0_final, res.J[-1])
    assert np.isclose(res.discrepancy_final, 2 * res.J[-1] / (P.p * P.info()["nS"]))
    # J reported by the run equals J0 recomputed from the returned f (reuse of q + lambda u, A21)
    assert np.isclose(P.J0_of_f(f, g, b), res.J0_final, rtol=1e-9)


def test_P7_descent_direction_bound():
    """grad'd <= -d'D^-1 d / alpha <= 0 for y = P+(f - alpha D grad) (projection inequality)"""
    rng = np.random.default_rng(78)
    P, g, b, truth, MS = _tiny_problem(10, 10, 2, False, rng)
    f = truth + rng.random(truth.shape)
    grad = P.gradient(f, g, b)
    for alpha in (1e-3, 0.7, 1.3, 50.0):
        D = P.scaling(f, 1e-3, 1e3)
        d = oracle.project(f, grad, D, alpha) - f
        gd = (grad * d).sum()
        assert gd <= -(d * d / D).sum() / alpha + 1e-9 * abs(gd)
        assert gd <= 0


@pytest.mark.parametrize("beta,alpha0", [(0.5, 1.3), (0.9, 40.0), (1e-4, 3e3)])
def test_P7_armijo_accepts_first_lambda_satisfying_the_inequality(beta, alpha0):
    """Alg.1 steps 4-5 re-evaluated here from the pinned building blocks:
    lambda_0 is the first theta^i with J0(f + lambda d) <= J0(f) + beta lambda grad'd."""
    rng = np.random.default_rng(79)
    P, g, b, truth, MS = _tiny_problem(10, 10, 1, False, rng)
    o = oracle.default_options(max_iter=1, beta=beta, alpha0=alpha0, alpha_max=1e5, adaptive_L=0, L1=1e-3, L2=1e3)
    f1, res = P.sgp(g, b, None, o)
    c0 = max(0.0, (g[0] - b[0]).mean())
    f0 = np.full((10, 10), c0)
    grad = P.gradient(f0, g, b)
    d = oracle.project(f0, grad, P.scaling(f0, 1e-3, 1e3), alpha0) - f0
    gd = (grad * d).sum()
    J0 = P.J0_of_f(f0, g, b)
    lam, nb = 1.0, 0
    while not P.J0_of_f(f0 + lam * d, g, b) <= J0 + beta * lam * gd:
        lam *= o.theta; nb += 1
    assert res.backtracks[0] == nb and np.isclose(res.lam[0], lam)
    assert np.allclose(f1, f0 + lam * d, rtol=1e-12, atol=1e-12)
    assert np.isclose(res.J[0], J0, rtol=1e-12) and np.isclose(res.J[1], P.J0_of_f(f1, g, b), rtol=1e-10)


def test_P7_nonmonotone_memory():
    """A15: with memory M the reference value is the max of the last M accepted J; M = 1 is the paper"""
    w = synth.c0_stars_gaussian(32)
    P = oracle.Problem(w["psf"])
    g = w["g"]; b = [np.full((32, 32), w["b"][0])]
    o = oracle.default_options(max_iter=150, armijo_memory=10, adaptive_L=0, L1=1e-10, L2=1e10)
    f, res = P.sgp(g, b, None, o)
    J = res.J
    for k in range(res.iterations):
        assert J[k + 1] <= J[max(0, k - 9): k + 1].max()
    # the memory is really used: some accepted steps increase J, and fewer backtracks are needed
    assert (np.diff(J) > 0).sum() >= 5
    o1 = oracle.default_options(max_iter=150, armijo_memory=1, adaptive_L=0, L1=1e-10, L2=1e10)
    _, res1 = P.sgp(g, b, None, o1)
    assert np.all(np.diff(res1.J) < 0) and res1.total_backtracks > res.total_backtracks
    # a memory of 2 must not behave like a longer one: every increase is bounded by the last 2 values
    o2 = oracle.default_options(max_iter=150, armijo_memory=2, adaptive_L=0, L1=1e-10, L2=1e10)
    _, res2 = P.sgp(g, b, None, o2)
    for k in range(res2.iterations):
        assert res2.J[k + 1] <= res2.J[max(0, k - 1): k + 1].max()


# ---------------------------------------------------------------------------------- P8
def test_P8_sgp_and_rl_reach_the_same_minimum_kkt():
    rng = np.random.default_rng(88)
    ny = nx = 8
    psf = _rand_psf(ny, nx, rng, 0.7)
    P = oracle.Problem([psf])
    truth = 50 * rng.random((ny, nx))
    b = [np.full((ny, nx), 2.0)]
    g = [rng.poisson(P.A(0, truth) + 2.0).astype(float)]
    f_sgp, rs = P.sgp(g, b, None, oracle.default_options(max_iter=4000, stop_rule=oracle.STOP_RELJ, tol=1e-15))
    f_rl, rr = P.rl(g, b, None, oracle.default_options(max_iter=60000))
    assert abs(rs.J0_final - rr.J0_final) <= 1e-9 * abs(rr.J0_final)
    grad = P.gradient(f_sgp, g, b)
    scale = np.abs(grad).max()
    pos = f_sgp > 1e-6 * f_sgp.max()
    assert np.abs(grad[pos]).max() <= 1e-5
    assert grad[~pos].min() >= -1e-5 if (~pos).any() else True
    # SGP needs (far) fewer iterations than RL to get there
    k_rl = np.argmax(rr.J <= rs.J0_final * (1 + 1e-9)) if (rr.J <= rs.J0_final * (1 + 1e-9)).any() else rr.iterations
    assert rs.iterations < k_rl


# ---------------------------------------------------------------------------------- P9
def test_P9_discrepancy_is_one_at_the_truth():
    """E[J0(f~; g)] ~ N^2/2, so 2 J0 /(p #S) ~ 1 at the true object and decreases from > 1"""
    w = synth.c2_lbt_multi(128, max_iter=30)
    P = oracle.Problem(w["psf"])
    b = [np.full((128, 128), bj) for bj in w["b"]]
    J = P.J0_of_f(w["truth"], w["g"], b)
    disc = 2 * J / (3 * 128 * 128)
    assert abs(disc - 1.0) <= 5 * np.sqrt(2.0 / (3 * 128 * 128)) + 0.02
    f, res = P.sgp(w["g"], b, None, oracle.default_options(max_iter=30))
    D = 2 * res.J / (3 * 128 * 128)
    assert D[0] > 1.0 and np.all(np.diff(D) < 0)
    # boundary problem: normalisation by #S (A6, A12)
    wb = synth.c3_boundary(96, 128, n_stars=60)
    Pb = oracle.Problem(wb["psf"], masked=True, S=wb["S"])
    gb = Pb.embed(wb["g"]); bb = [np.full((128, 128), wb["b"][0])]
    Jb = Pb.J0_of_f(wb["truth"], gb, bb)
    # truth outside R is dropped by M_R, so allow a small excess
    assert 0.9 <= 2 * Jb / (96 * 96) <= 1.25


def test_P9_discrepancy_stop_rule():
    w = synth.c1_galaxies_airy(64)
    P = oracle.Problem(w["psf"])
    b = [np.full((64, 64), w["b"][0])]
    o = oracle.default_options(max_iter=500, stop_rule=oracle.STOP_DISCREPANCY, disc_threshold=1.05)
    f, res = P.sgp(w["g"], b, None, o)
    D = 2 * res.J / (64 * 64)
    assert res.stop_reason == 3 and res.iterations < 500
    assert D[-1] <= 1.05 and np.all(D[:-1] > 1.05)          # first k with D(k) <= b (A7)
    o2 = oracle.default_options(max_iter=500, stop_rule=oracle.STOP_RELJ, tol=1e-4)
    f2, res2 = P.sgp(w["g"], b, None, o2)
    J = res2.J
    rel = np.abs(np.diff(J)) / J[:-1]
    assert res2.stop_reason == 2 and rel[-1] <= 1e-4 and np.all(rel[:-1] > 1e-4)      # Eq.24


# ---------------------------------------------------------------------------------- P10
def test_P10_bb_rules_by_hand():
    """Eq.7-9 and the safeguards of PAPER.md:132-153 on a 3-vector example worked out here by hand."""
    s = np.array([1.0, -2.0, 0.5]); z = np.array([0.5, -1.0, 1.0]); D = np.array([1.0, 2.0, 4.0])
    a = (s * s / D**2).sum(); c = (s * z / D).sum(); e = (s * z * D).sum(); h = (z * z * D**2).sum()
    assert (a, c, e, h) == (1.0 + 1.0 + 0.015625, 0.5 + 1.0 + 0.125, 0.5 + 4.0 + 2.0, 0.25 + 4.0 + 16.0)
    bb1, bb2 = a / c, e / h                                    # 1.2403846..., 0.3209876...
    o = oracle.default_options()
    bb = oracle.BB(o)
    # k = 1: ring = {bb2}: alpha = bb2 (first 20 iterations use Eq.9, tau unchanged)
    alpha, rule, a1, a2 = bb.next(1, a, c, e, h)
    assert np.isclose(a1, bb1) and np.isclose(a2, bb2) and rule == 2 and np.isclose(alpha, bb2)
    assert bb.s.tau == 0.5 and bb.s.alpha_prev == alpha
    # k = 2: c <= 0 -> alpha1 = min(10 alpha_prev, alpha_max); e <= 0 -> alpha2 likewise
    alpha2, rule, a1, a2 = bb.next(2, a, -1.0, -2.0, h)
    assert np.isclose(a1, 10 * bb2) and np.isclose(a2, 10 * bb2)
    assert np.isclose(alpha2, min(bb2, 10 * bb2))              # ring minimum over {bb2, 10 bb2}
    # clamps
    _, _, a1, a2 = bb.next(3, 1e9, 1.0, 1e-9, 1.0)
    assert a1 == o.alpha_max and a2 == o.alpha_min
    # ring holds the last M_alpha = 3 values only: {10 bb2, alpha_min, X}
    alpha4, _, _, a2 = bb.next(4, a, c, 50.0, 1.0)
    assert a2 == 50.0 and alpha4 == o.alpha_min
    alpha5, _, _, _ = bb.next(5, a, c, 60.0, 1.0)
    assert alpha5 == o.alpha_min                               # ring {alpha_min, 50, 60}
    alpha6, _, _, _ = bb.next(6, a, c, 70.0, 1.0)
    assert alpha6 == 50.0                                      # ring {50, 60, 70}
    assert bb.s.tau == 0.5
    # alternation after the first 20 iterations
    bb = oracle.BB(o)
    al, rule, a1, a2 = bb.next(21, a, c, e, h)                 # a2/a1 = 0.2588 <= 0.5 -> Eq.9, tau *= 0.9
    assert rule == 2 and np.isclose(al, bb2) and np.isclose(bb.s.tau, 0.45)
    al, rule, a1, a2 = bb.next(22, a, c, 0.9 * a / c * h, h)   # a2/a1 = 0.9 > tau -> BB1, tau *= 1.1
    assert rule == 1 and np.isclose(al, bb1) and np.isclose(bb.s.tau, 0.495)
    # 10 * alpha_{k-1} uses the alpha actually used (A10)
    al, rule, a1, a2 = bb.next(23, a, 0.0, e, h)
    assert np.isclose(a1, 10 * bb1)


def test_P10_adaptive_bounds_by_hand():
    """PAPER.md:273-275 (A19)"""
    assert oracle.adaptive_bounds(np.array([0.0, 2.0, 40.0, 0.0, 5.0])) == (0.2, 400.0)     # 20 < 50
    assert oracle.adaptive_bounds(np.array([0.0, 2.0, 400.0, -1.0])) == (2.0, 400.0)       # 200 >= 50
    assert oracle.adaptive_bounds(np.array([1.0, 50.0])) == (1.0, 50.0)                    # ratio == 50: not < 50


def test_P10_bb_sums_in_a_run_match_definition():
    """alpha_1 of a real run recomputed here from f(0), f(1), grad(0), grad(1) and Eq.7-9"""
    rng = np.random.default_rng(101)
    P, g, b, truth, MS = _tiny_problem(10, 10, 2, False, rng)
    o1 = oracle.default_options(max_iter=1, adaptive_L=0, L1=0.5, L2=40.0)
    o2 = oracle.default_options(max_iter=2, adaptive_L=0, L1=0.5, L2=40.0)
    f1, r1 = P.sgp(g, b, None, o1)
    f2, r2 = P.sgp(g, b, None, o2)
    c0 = max(0.0, np.mean([(gg - bb).mean() for gg, bb in zip(g, b)]))
    f0 = np.full((10, 10), c0)
    s = f1 - f0
    z = P.gradient(f1, g, b) - P.gradient(f0, g, b)
    D = np.clip(f1, 0.5, 40.0) / 2
    bb2 = (s * z * D).sum() / (z * z * D * D).sum()
    assert np.isclose(r2.alpha[1], np.clip(bb2, o2.alpha_min, o2.alpha_max), rtol=1e-9)
    assert r2.alpha[0] == 1.3


# ---------------------------------------------------------------------------------- P11
@pytest.mark.parametrize("p", [1, 3])
def test_P11_fft_count(p):
    """2p+2 two-dimensional transforms per SGP iteration and per RL step, none per backtrack"""
    w = synth.c2_lbt_multi(32, p=p)
    P = oracle.Problem(w["psf"])
    b = [np.full((32, 32), bj) for bj in w["b"]]
    counts = {}
    for K in (5, 9):
        _, res = P.sgp(w["g"], b, None, oracle.default_options(max_iter=K))
        counts[K] = res.n_fft2
    assert counts[5] == 5 * (2 * p + 2) and counts[9] == 9 * (2 * p + 2)
    # force backtracking with an absurd first step: the count must not change
    o = oracle.default_options(max_iter=3, alpha0=1e5, alpha_max=1e5)
    _, res = P.sgp(w["g"], b, None, o)
    assert res.total_backtracks > 0 and res.n_fft2 == 3 * (2 * p + 2)
    rl = {}
    for K in (4, 7):
        _, res = P.rl(w["g"], b, None, oracle.default_options(max_iter=K))
        rl[K] = res.n_fft2
    assert rl[7] - rl[4] == 3 * (2 * p + 2)


# ---------------------------------------------------------------------------------- entry points
# ---------------------------------------------------------------------------------- P12 (OSEM, Algorithm 2)
def _dense_operator(k, ny, nx, MS, MR):
    """the matrix of A_j written out from Eq.16: A[m, n] = M_S(m) K_j(m - n) M_R(n), K_j normalised, periodic, centre at ny/2, nx/2"""
    K0 = np.fft.ifftshift(k / k.sum())
    A = np.zeros((ny * nx, ny * nx))
    for my, mx in itertools.product(range(ny), range(nx)):
        if not MS[my, mx]:
            continue
        for qy, qx in itertools.product(range(ny), range(nx)):
            if MR[qy, qx]:
                A[my * nx + mx, qy * nx + qx] = K0[(my - qy) % ny, (mx - qx) % nx]
    return A


@pytest.mark.parametrize("p,masked,S", [(2, False, None), (3, False, None), (2, True, (1, 2, 6, 5))])
def test_P12_osem_cycle_is_eq15_eq22_written_out_with_dense_matrices(p, masked, S):
    """PAPER.md:178-191 (Algorithm 2, Eq.15) and :246 (Eq.22): the cycle over the images written with dense matrices
    built from the definition of A_j (Eq.16), its transpose, and alpha_j = A_j^T 1_S: h <- (M_R/alpha_j) h o A_j^T(g_j/(A_j h + b_j)),
    j = 1..p in this order, each sub-step seeing the previous one's h."""
    rng = np.random.default_rng(120 + p)
    ny, nx = 8, 7
    P, g, b, truth, MS = _tiny_problem(ny, nx, p, masked, rng, S=S)
    info = P.info()
    MR = info["MR"].astype(bool)
    f0 = (1.0 + 20 * rng.random((ny, nx))) * MR
    K = 3
    f_or, res = P.osem(g, b, f0, oracle.default_options(max_iter=K, init=oracle.INIT_USER))
    mats = [_dense_operator(k, ny, nx, MS, MR) for k in P.psfs] if hasattr(P, "psfs") else None
    if mats is None:
        pytest.skip("Problem does not keep its PSFs")
    h = f0.ravel().copy()
    ones_S = MS.ravel().astype(float)
    for _ in range(K):
        for j in range(p):
            A = mats[j]
            aj = A.T @ ones_S
            r = np.where(MS.ravel() > 0, g[j].ravel() / (A @ h + b[j].ravel()), 0.0)
            h = np.where(MR.ravel(), h * (A.T @ r) / np.where(MR.ravel(), aj, 1.0), 0.0)
    assert np.abs(f_or.ravel() - h).max() <= 1e-11 * np.abs(h).max()
    assert res.iterations == K and res.n_fft2 == 4 * p * K          # "4p FFTs" per OSEM iteration
    # the order of the cycle matters (so the pin would catch a reversed or simultaneous update)
    h2 = f0.ravel().copy()
    for _ in range(K):
        for j in reversed(range(p)):
            A = mats[j]
            aj = A.T @ ones_S
            r = np.where(MS.ravel() > 0, g[j].ravel() / (A @ h2 + b[j].ravel()), 0.0)
            h2 = np.where(MR.ravel(), h2 * (A.T @ r) / np.where(MR.ravel(), aj, 1.0), 0.0)
    assert np.abs(h2 - h).max() > 1e-6 * np.abs(h).max()
    # J0 reported at the final iterate is Eq.12 there
    q = [mats[j] @ h for j in range(p)]
    J = sum(float(np.sum(np.where(MS.ravel() > 0, np.where(g[j].ravel() > 0, g[j].ravel() * np.log(np.where(g[j].ravel() > 0, g[j].ravel(), 1.0) / (q[j] + b[j].ravel())), 0.0) + q[j] + b[j].ravel() - g[j].ravel(), 0.0))) for j in range(p))
    assert abs(res.J0_final - J) <= 1e-10 * abs(J)


@pytest.mark.parametrize("masked,S", [(False, None), (True, (2, 2, 8, 8))])
def test_P12_osem_with_one_image_is_RL_and_substeps_conserve_flux(masked, S):
    """p = 1: Algorithm 2 is Eq.1 / Eq.21.  b = 0: every sub-step j conserves sum_R alpha_j h(j) = sum_S g_j
    (the argument of PAPER.md:33 applied to image j), so after a full cycle the flux is that of the LAST image."""
    rng = np.random.default_rng(12)
    P, g, b, truth, MS = _tiny_problem(12, 12, 1, masked, rng, S=S)
    o = oracle.default_options(max_iter=5)
    f_rl, r_rl = P.rl(g, b, opts=o)
    f_os, r_os = P.osem(g, b, opts=o)
    assert np.abs(f_rl - f_os).max() <= 1e-13 * np.abs(f_rl).max() and abs(r_os.J0_final - r_rl.J0_final) <= 1e-12 * r_rl.J0_final
    p = 3
    psfs = [_rand_psf(12, 12, rng, 1.0 + 0.5 * j) for j in range(p)]
    P3 = oracle.Problem(psfs, masked=masked, S=S, sigma_R=0.02)
    oy, ox, sy, sx = P3.S
    M = np.zeros((12, 12)); M[oy:oy + sy, ox:ox + sx] = 1
    g3 = [rng.poisson(20 + 60 * (j + 1) * rng.random((12, 12))) * M for j in range(p)]
    b0 = [np.zeros((12, 12)) for _ in range(p)]
    f, _ = P3.osem(g3, b0, opts=oracle.default_options(max_iter=4))
    alpha_last = P3.AT(p - 1, M)
    assert np.isclose((alpha_last * f).sum(), g3[-1].sum(), rtol=1e-12)
    assert not np.isclose((alpha_last * f).sum(), g3[0].sum(), rtol=1e-3)
    assert np.all(f >= 0)


# ---------------------------------------------------------------------------------- P13 (multiplicative relaxation, Eq.3)
@pytest.mark.parametrize("p,masked,S", [(1, False, None), (2, False, None), (1, True, (2, 2, 8, 8))])
def test_P13_multiplicative_relaxation_is_eq3(p, masked, S):
    """PAPER.md:46, Eq.3: f(k+1) = f(k) o (A^T g/(A f(k) + b))^alpha written out with the operators of Eq.16/17 (for p
    images / boundary correction the bracket is the RL factor of Eq.13 / Eq.21, reading A24); alpha = 1 is RL itself;
    with alpha = 1.5 on a noiseless consistent problem the true object stays a fixed point and the iteration reaches a
    given J0 in fewer steps than RL ("a reduction in the number of iterations by a factor of alpha")."""
    rng = np.random.default_rng(130 + p)
    P, g, b, truth, MS = _tiny_problem(12, 12, p, masked, rng, S=S)
    info = P.info()
    f0 = (1.0 + rng.random((12, 12)) * 30) * info["MR"]
    K, a = 4, 1.5
    f_or, _ = P.rl(g, b, f0, oracle.default_options(max_iter=K, init=oracle.INIT_USER, rl_relax=a))
    f = f0.copy()
    for _ in range(K):
        w = sum(P.AT(j, np.where(P.A(j, f) + b[j] > 0, g[j] / (P.A(j, f) + b[j]), 0.0)) for j in range(P.p))
        f = f * (info["W"] * w) ** a
    assert np.abs(f_or - f).max() <= 1e-12 * np.abs(f).max()
    f1, r1 = P.rl(g, b, f0, oracle.default_options(max_iter=K, init=oracle.INIT_USER, rl_relax=1.0))
    f2, r2 = P.rl(g, b, f0, oracle.default_options(max_iter=K, init=oracle.INIT_USER))
    assert np.array_equal(f1, f2)
    # fixed point: noiseless data g_j = A_j truth + b
    gq = [q + b[j] for j, q in enumerate(P.all_A(truth))]
    ft, _ = P.rl(gq, b, truth, oracle.default_options(max_iter=3, init=oracle.INIT_USER, rl_relax=a))
    assert np.abs(ft - truth).max() <= 1e-11 * truth.max()
    # acceleration: J0 after 12 relaxed steps is below J0 after 12 plain steps (both monotone here)
    _, ra = P.rl(g, b, f0, oracle.default_options(max_iter=12, init=oracle.INIT_USER, rl_relax=a))
    _, rp = P.rl(g, b, f0, oracle.default_options(max_iter=12, init=oracle.INIT_USER))
    assert ra.J0_final < rp.J0_final
    with pytest.raises(oracle.OracleError):
        P.rl(g, b, f0, oracle.default_options(max_iter=1, init=oracle.INIT_USER, rl_relax=0.0))


# ---------------------------------------------------------------------------------- P14 (linear relaxation, Eq.4)
@pytest.mark.parametrize("p,masked,S", [(1, False, None), (2, False, None), (1, True, (2, 2, 8, 8))])
def test_P14_linear_relaxation_is_eq4(p, masked, S):
    """PAPER.md:50, Eq.4: f(k+1) = f(k) - lambda f(k) o (1 - A^T g/(A f(k) + b)) written out with the operators of
    Eq.16/17 (constant lambda_k, reading A25; for p images / boundary correction the bracket holds the RL factor of
    Eq.13 / Eq.21); lambda = 1 is RL itself; one step is the point (1 - lambda) f + lambda f_RL on the
    line through f and the RL step ("a line search along this descent direction"), projected on f >= 0
    (the paper's constraint); the flux invariant of
    RL survives for p = 1 unmasked (sum f(k+1) = sum(g - b) whenever sum f(k) is); the true object of a noiseless
    problem is a fixed point; J0 after a few relaxed steps is below plain RL."""
    rng = np.random.default_rng(140 + p)
    P, g, b, truth, MS = _tiny_problem(12, 12, p, masked, rng, S=S)
    info = P.info()
    f0 = (1.0 + rng.random((12, 12)) * 30) * info["MR"]
    K, lam = 4, 1.4
    f_or, _ = P.rl(g, b, f0, oracle.default_options(max_iter=K, init=oracle.INIT_USER, rl_linear=lam))
    f = f0.copy()
    for _ in range(K):
        w = sum(P.AT(j, np.where(P.A(j, f) + b[j] > 0, g[j] / (P.A(j, f) + b[j]), 0.0)) for j in range(P.p))
        f = np.maximum(0.0, f - lam * f * (1.0 - info["W"] * w))      # projected on f >= 0 (reading A25)
    assert np.abs(f_or - f).max() <= 1e-12 * np.abs(f).max()
    f1, _ = P.rl(g, b, f0, oracle.default_options(max_iter=K, init=oracle.INIT_USER, rl_linear=1.0))
    f2, _ = P.rl(g, b, f0, oracle.default_options(max_iter=K, init=oracle.INIT_USER))
    assert np.array_equal(f1, f2)
    # one step lies on the line through f0 and the plain RL step
    fl, _ = P.rl(g, b, f0, oracle.default_options(max_iter=1, init=oracle.INIT_USER, rl_linear=lam))
    fr, _ = P.rl(g, b, f0, oracle.default_options(max_iter=1, init=oracle.INIT_USER))
    assert np.abs(fl - np.maximum(0.0, (1 - lam) * f0 + lam * fr)).max() <= 1e-12 * np.abs(fr).max()
    assert np.abs(fl - fr).max() > 1e-3 * np.abs(fr).max()                    # and is not the RL step itself
    if p == 1 and not masked:
        # flux: sum f_RL = sum g f/(Af+b) A1 ... for b = 0 and a unit-volume PSF sum f_RL = sum g; the relaxed step keeps
        # (1 - lam) sum f0 + lam sum g
        g0 = [P.A(0, truth)]
        fz, _ = P.rl(g0, [np.zeros_like(truth)], f0, oracle.default_options(max_iter=1, init=oracle.INIT_USER, rl_linear=lam))
        if fz[f0 > 0].min() > 0:      # no pixel was projected
            assert abs(fz.sum() - ((1 - lam) * f0.sum() + lam * g0[0].sum())) <= 1e-11 * g0[0].sum()
        # a start point far above the data: the unprojected step (1 - lam) f + lam f_RL is negative there, the result is 0
        fbig = f0.copy(); fbig[3, 4] = 1e6
        fc, _ = P.rl(g, b, fbig, oracle.default_options(max_iter=1, init=oracle.INIT_USER, rl_linear=lam))
        assert fc[3, 4] == 0.0 and fc.min() == 0.0
    # fixed point: noiseless data g_j = A_j truth + b
    gq = [q + b[j] for j, q in enumerate(P.all_A(truth))]
    ft, _ = P.rl(gq, b, truth, oracle.default_options(max_iter=3, init=oracle.INIT_USER, rl_linear=lam))
    assert np.abs(ft - truth).max() <= 1e-11 * truth.max()
    _, ra = P.rl(g, b, f0, oracle.default_options(max_iter=12, init=oracle.INIT_USER, rl_linear=lam))
    _, rp = P.rl(g, b, f0, oracle.default_options(max_iter=12, init=oracle.INIT_USER))
    assert ra.J0_final < rp.J0_final
    with pytest.raises(oracle.OracleError):
        P.rl(g, b, f0, oracle.default_options(max_iter=1, init=oracle.INIT_USER, rl_linear=0.0))
    with pytest.raises(oracle.OracleError):                                   # Eq.3 and Eq.4 are alternatives
        P.rl(g, b, f0, oracle.default_options(max_iter=1, init=oracle.INIT_USER, rl_linear=1.2, rl_relax=1.2))


def test_entry_points_match_problem_api():
    w = synth.c3_boundary(24, 32, n_stars=30)
    o = oracle.default_options(max_iter=15)
    f, res = oracle.sgp_boundary(w["g"], w["psf"], w["b"], w["S"][0], w["S"][1], None, o)
    P = oracle.Problem(w["psf"], masked=True, S=w["S"], sigma_R=o.sigma_R)
    f2, res2 = P.sgp(P.embed(w["g"]), [np.full((32, 32), w["b"][0])], None, o)
    assert res.rc == 0 and np.array_equal(f, f2) and np.array_equal(res.J, res2.J)
    assert np.array_equal(res.maskR, P.info()["MR"])
    w1 = synth.c0_stars_gaussian(32)
    fa, ra = oracle.sgp_single(w1["g"][0], w1["psf"][0], w1["b"][0], None, o)
    fb, rb = oracle.sgp_multi(w1["g"], w1["psf"], w1["b"], None, o)
    assert np.array_equal(fa, fb) and ra.iterations == 15
    fr, rr = oracle.rl_single(w1["g"][0], w1["psf"][0], w1["b"][0], None, o)
    assert rr.iterations == 15 and np.all(np.diff(rr.J) < 0)      # RL decreases J0 monotonically
    # b given as an array is the same as the constant
    fc, rc_ = oracle.sgp_single(w1["g"][0], w1["psf"][0], np.full((32, 32), w1["b"][0]), None, o)
    assert np.array_equal(fa, fc)


def test_float_build_tracks_double_build():
    w = synth.c0_stars_gaussian(32)
    o = oracle.default_options(max_iter=10)
    f64, r64 = oracle.sgp_single(w["g"][0], w["psf"][0], w["b"][0], None, o, dtype=np.float64)
    f32, r32 = oracle.sgp_single(w["g"][0], w["psf"][0], w["b"][0], None, o, dtype=np.float32)
    assert f32.dtype == np.float32
    assert np.linalg.norm(f32 - f64) <= 1e-3 * np.linalg.norm(f64)
    assert abs(r32.J0_final - r64.J0_final) <= 1e-4 * r64.J0_final


def test_error_codes():
    w = synth.c0_stars_gaussian(16)
    o = oracle.default_options(max_iter=2)
    with pytest.raises(oracle.OracleError):
        oracle.Problem([np.zeros((8, 8))])                       # PSF with zero volume
    _, res = oracle.sgp_single(-np.ones((16, 16)), w["psf"][0], 1.0, None, oracle.default_options(max_iter=2, strict=1))
    assert res.rc == -3
    o_bad = oracle.default_options(max_iter=2, theta=1.5)
    _, res = oracle.sgp_single(w["g"][0], w["psf"][0], 10.0, None, o_bad)
    assert res.rc == -1
