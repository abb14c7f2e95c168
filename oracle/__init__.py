"""ctypes access to the CPU oracle (oracle/sgp_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports the CUDA
package and the CUDA package never imports it.

The wrappers below only marshal numpy arrays into the C calls; all arithmetic is in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sgp_oracle.c"
_HDR = _HERE / "sgp_oracle.h"
_LIBS = {np.dtype(np.float64): _HERE / "liboracle_f64.so", np.dtype(np.float32): _HERE / "liboracle_f32.so"}
_loaded: dict = {}

STOP_MAXIT, STOP_RELJ, STOP_DISCREPANCY, STOP_MINERR = 0, 1, 2, 3
INIT_USER, INIT_CONST, INIT_ZERO, INIT_G, INIT_CONST_SMOOTH = 0, 1, 2, 3, 4
PSF_CENTER, PSF_CORNER = 0, 1
REASON = {1: "maxit", 2: "relJ", 3: "discrepancy", 4: "minerr"}
ERR_LINESEARCH = -6


def build(force: bool = False) -> None:
    """Compile liboracle_f64.so and liboracle_f32.so with gcc (plain C99 + OpenMP)."""
    for dt, out in _LIBS.items():
        stale = force or not out.exists() or out.stat().st_mtime < max(_SRC.stat().st_mtime, _HDR.stat().st_mtime)
        if not stale:
            continue
        cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-Wno-unknown-pragmas", "-o", str(out), str(_SRC), "-lm"]
        if dt == np.dtype(np.float32):
            cmd.insert(1, "-DORACLE_FLOAT")
        subprocess.run(cmd, check=True)


class Options(C.Structure):
    """oracle_options of sgp_oracle.h (paper defaults via oracle_options_default)."""
    _fields_ = [
        ("beta", C.c_double), ("theta", C.c_double),
        ("alpha0", C.c_double), ("alpha_min", C.c_double), ("alpha_max", C.c_double), ("tau1", C.c_double),
        ("m_alpha", C.c_int), ("alt_start", C.c_int), ("armijo_memory", C.c_int),
        ("L1", C.c_double), ("L2", C.c_double), ("adaptive_L", C.c_int),
        ("max_iter", C.c_int), ("stop_rule", C.c_int), ("tol", C.c_double), ("disc_threshold", C.c_double),
        ("sigma_R", C.c_double), ("max_backtracks", C.c_int), ("psf_origin", C.c_int), ("init", C.c_int),
        ("refresh_every", C.c_int), ("strict", C.c_int), ("rl_relax", C.c_double), ("rl_linear", C.c_double),
        ("flux_constraint", C.c_int), ("flux_value", C.c_double), ("init_sigma", C.c_double),
    ]


class _Result(C.Structure):
    _fields_ = [
        ("iterations", C.c_int), ("stop_reason", C.c_int), ("J0_final", C.c_double),
        ("discrepancy_final", C.c_double), ("total_backtracks", C.c_int),
        ("L1_used", C.c_double), ("L2_used", C.c_double), ("n_fft2", C.c_long),
        ("trace_J", C.POINTER(C.c_double)), ("trace_alpha", C.POINTER(C.c_double)),
        ("trace_lambda", C.POINTER(C.c_double)), ("trace_rule", C.POINTER(C.c_int)),
        ("trace_backtracks", C.POINTER(C.c_int)),
        ("force_alpha", C.POINTER(C.c_double)), ("force_lambda", C.POINTER(C.c_double)),
        ("truth", C.c_void_p), ("trace_err", C.POINTER(C.c_double)), ("err_final", C.c_double),
    ]


class BBState(C.Structure):
    _fields_ = [("alpha_prev", C.c_double), ("tau", C.c_double), ("ring", C.c_double * 16),
                ("ring_len", C.c_int), ("ring_pos", C.c_int), ("m_alpha", C.c_int)]


def lib(dtype=np.float64) -> C.CDLL:
    dt = np.dtype(dtype)
    if dt not in _LIBS:
        raise TypeError(f"oracle has no build for dtype {dt}")
    if dt not in _loaded:
        build()
        L = C.CDLL(str(_LIBS[dt]))
        L.oracle_J0.restype = C.c_double
        L.oracle_bb_next.restype = C.c_double
        L.oracle_rel_error.restype = C.c_double
        L.oracle_problem_create.restype = C.c_void_p
        L.oracle_options_default.restype = None
        L.oracle_bb_init.restype = None
        L.oracle_problem_destroy.restype = None
        L.oracle_problem_destroy.argtypes = [C.c_void_p]
        _loaded[dt] = L
    return _loaded[dt]


def default_options(**kw) -> Options:
    o = Options()
    lib().oracle_options_default(C.byref(o))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise AttributeError(k)
        setattr(o, k, v)
    return o


def _arr(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _pp(arrs):
    """array of pointers (const oreal *const *)"""
    return (C.c_void_p * len(arrs))(*[a.ctypes.data for a in arrs])


def _check(rc, what):
    if rc != 0:
        raise OracleError(rc, what)


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"{what}: oracle error {code}")
        self.code = code


def fft2(x, sign=-1, dtype=np.float64):
    dt = np.dtype(dtype)
    x = np.asarray(x)
    re, im = _arr(x.real, dt), _arr(x.imag, dt)
    ny, nx = re.shape
    ore, oim = np.empty_like(re), np.empty_like(re)
    _check(lib(dt).oracle_fft2(ny, nx, int(sign), _ptr(re), _ptr(im), _ptr(ore), _ptr(oim)), "fft2")
    return ore + 1j * oim


def conv2_direct(K, x, dtype=np.float64):
    dt = np.dtype(dtype)
    K, x = _arr(K, dt), _arr(x, dt)
    out = np.empty_like(x)
    _check(lib(dt).oracle_conv2_direct(x.shape[0], x.shape[1], _ptr(K), _ptr(x), _ptr(out)), "conv2_direct")
    return out


def project(f, grad, D, alpha, dtype=np.float64):
    dt = np.dtype(dtype)
    f, grad, D = _arr(f, dt), _arr(grad, dt), _arr(D, dt)
    y = np.empty_like(f)
    _check(lib(dt).oracle_project(C.c_long(f.size), _ptr(f), _ptr(grad), _ptr(D), C.c_double(alpha), _ptr(y)), "project")
    return y


def adaptive_bounds(y, dtype=np.float64):
    dt = np.dtype(dtype)
    y = _arr(y, dt)
    L1, L2 = C.c_double(), C.c_double()
    _check(lib(dt).oracle_adaptive_bounds(C.c_long(y.size), _ptr(y), C.byref(L1), C.byref(L2)), "adaptive_bounds")
    return L1.value, L2.value


def project_flux(x, D, c, dtype=np.float64):
    """(y, mu): projection on {y >= 0, sum y = c} in the metric D^-1 (oracle_project_flux)"""
    dt = np.dtype(dtype)
    x, D = _arr(x, dt), _arr(D, dt)
    y = np.empty_like(x)
    mu = C.c_double()
    _check(lib(dt).oracle_project_flux(C.c_long(x.size), _ptr(x), _ptr(D), C.c_double(c), _ptr(y), C.byref(mu)), "project_flux")
    return y, mu.value


def rel_error(f, truth, dtype=np.float64):
    dt = np.dtype(dtype)
    f, truth = _arr(f, dt), _arr(truth, dt)
    return lib(dt).oracle_rel_error(C.c_long(f.size), _ptr(f), _ptr(truth))


class BB:
    """The step-length state machine of PAPER.md:130-155 (oracle_bb_init / oracle_bb_next)."""

    def __init__(self, opts: Options | None = None):
        self.o = opts or default_options()
        self.s = BBState()
        lib().oracle_bb_init(C.byref(self.s), C.byref(self.o))

    def next(self, k, a, c, e, h):
        rule, a1, a2 = C.c_int(), C.c_double(), C.c_double()
        alpha = lib().oracle_bb_next(C.byref(self.s), C.byref(self.o), int(k), C.c_double(a), C.c_double(c),
                                     C.c_double(e), C.c_double(h), C.byref(rule), C.byref(a1), C.byref(a2))
        return alpha, rule.value, a1.value, a2.value


class Result:
    def __init__(self, raw: _Result, traces: dict):
        self.iterations = raw.iterations
        self.stop_reason = raw.stop_reason
        self.J0_final = raw.J0_final
        self.discrepancy_final = raw.discrepancy_final
        self.total_backtracks = raw.total_backtracks
        self.L1_used, self.L2_used = raw.L1_used, raw.L2_used
        self.n_fft2 = raw.n_fft2
        k = self.iterations
        self.J = traces["J"][: k + 1].copy()
        self.alpha = traces["alpha"][:k].copy()
        self.lam = traces["lambda"][:k].copy()
        self.rule = traces["rule"][:k].copy()
        self.backtracks = traces["backtracks"][:k].copy()
        self.err_final = raw.err_final
        self.err = traces["err"][: k + 2].copy()      # rho(0..k) and, for a MINERR stop, the discarded rho(k+1)


def _make_result(max_iter, force_alpha=None, force_lambda=None, truth=None, dt=np.float64):
    n = max_iter + 1
    tr = {"J": np.zeros(n), "alpha": np.zeros(n), "lambda": np.zeros(n),
          "rule": np.zeros(n, np.int32), "backtracks": np.zeros(n, np.int32), "err": np.full(n + 1, np.nan)}
    raw = _Result()
    raw.trace_err = tr["err"].ctypes.data_as(C.POINTER(C.c_double))
    raw.trace_J = tr["J"].ctypes.data_as(C.POINTER(C.c_double))
    raw.trace_alpha = tr["alpha"].ctypes.data_as(C.POINTER(C.c_double))
    raw.trace_lambda = tr["lambda"].ctypes.data_as(C.POINTER(C.c_double))
    raw.trace_rule = tr["rule"].ctypes.data_as(C.POINTER(C.c_int))
    raw.trace_backtracks = tr["backtracks"].ctypes.data_as(C.POINTER(C.c_int))
    keep = []
    for name, arr in (("force_alpha", force_alpha), ("force_lambda", force_lambda)):
        if arr is not None:
            a = np.full(max(max_iter, 1), np.nan)
            a[: len(arr)] = np.asarray(arr, dtype=np.float64)[: len(a)]
            keep.append(a)
            setattr(raw, name, a.ctypes.data_as(C.POINTER(C.c_double)))
    if truth is not None:
        t = _arr(truth, dt)
        keep.append(t)
        raw.truth = t.ctypes.data
    return raw, tr, keep


class Problem:
    """oracle_problem: the grid, the masks and the transfer functions."""

    def __init__(self, psfs, masked=False, S=None, sigma_R=1e-2, psf_origin=PSF_CENTER, dtype=np.float64):
        self.dt = np.dtype(dtype)
        self.L = lib(self.dt)
        self.psfs = [_arr(k, self.dt) for k in psfs]
        self.p = len(self.psfs)
        self.ny, self.nx = self.psfs[0].shape
        oy, ox, sy, sx = S if S is not None else (0, 0, self.ny, self.nx)
        self.S = (oy, ox, sy, sx)
        err = C.c_int()
        self.h = self.L.oracle_problem_create(self.p, self.ny, self.nx, _pp(self.psfs), int(bool(masked)),
                                              oy, ox, sy, sx, C.c_double(sigma_R), int(psf_origin), C.byref(err))
        if not self.h:
            raise OracleError(err.value, "problem_create")
        self.h = C.c_void_p(self.h)

    def __del__(self):
        h = getattr(self, "h", None)
        if h:
            self.L.oracle_problem_destroy(h)
            self.h = None

    def _planes(self, arrs):
        out = [_arr(a, self.dt) for a in arrs]
        assert len(out) == self.p and all(a.shape == (self.ny, self.nx) for a in out)
        return out

    def embed(self, imgs, fill=0.0):
        """place sy x sx images on the S-bar grid (zero padding)"""
        oy, ox, sy, sx = self.S
        out = []
        for a in imgs:
            e = np.full((self.ny, self.nx), fill, self.dt)
            e[oy:oy + sy, ox:ox + sx] = a
            out.append(e)
        return out

    def info(self):
        alpha = np.empty((self.ny, self.nx), self.dt)
        W = np.empty_like(alpha)
        MR = np.empty((self.ny, self.nx), np.uint8)
        nS, nR = C.c_long(), C.c_long()
        _check(self.L.oracle_problem_get(self.h, _ptr(alpha), _ptr(W), _ptr(MR), C.byref(nS), C.byref(nR)), "get")
        return {"alpha": alpha, "W": W, "MR": MR, "nS": nS.value, "nR": nR.value}

    def A(self, j, x):
        x = _arr(x, self.dt); out = np.empty_like(x)
        _check(self.L.oracle_apply_A(self.h, j, _ptr(x), _ptr(out)), "apply_A")
        return out

    def AT(self, j, y):
        y = _arr(y, self.dt); out = np.empty_like(y)
        _check(self.L.oracle_apply_AT(self.h, j, _ptr(y), _ptr(out)), "apply_AT")
        return out

    def all_A(self, x):
        x = _arr(x, self.dt)
        outs = [np.empty_like(x) for _ in range(self.p)]
        _check(self.L.oracle_all_A(self.h, _ptr(x), _pp(outs)), "all_A")
        return outs

    def sum_AT(self, rs):
        rs = self._planes(rs); out = np.empty_like(rs[0])
        _check(self.L.oracle_sum_AT(self.h, _pp(rs), _ptr(out)), "sum_AT")
        return out

    def J0(self, q, g, b):
        q, g, b = self._planes(q), self._planes(g), self._planes(b)
        return self.L.oracle_J0(self.h, _pp(q), _pp(g), _pp(b))

    def J0_of_f(self, f, g, b):
        return self.J0(self.all_A(f), g, b)

    def gradient(self, f, g, b):
        f, g, b = _arr(f, self.dt), self._planes(g), self._planes(b)
        out = np.empty_like(f)
        _check(self.L.oracle_gradient(self.h, _ptr(f), _pp(g), _pp(b), _ptr(out)), "gradient")
        return out

    def rl_step(self, f, g, b):
        f, g, b = _arr(f, self.dt), self._planes(g), self._planes(b)
        out = np.empty_like(f)
        _check(self.L.oracle_rl_step(self.h, _ptr(f), _pp(g), _pp(b), _ptr(out)), "rl_step")
        return out

    def scaling(self, f, L1, L2):
        f = _arr(f, self.dt); out = np.empty_like(f)
        _check(self.L.oracle_scaling(self.h, _ptr(f), C.c_double(L1), C.c_double(L2), _ptr(out)), "scaling")
        return out

    def _run(self, fn, g, b, f0, opts, force_alpha=None, force_lambda=None, check=True, truth=None):
        g, b = self._planes(g), self._planes(b)
        f0a = _arr(f0, self.dt) if f0 is not None else None
        raw, tr, keep = _make_result(opts.max_iter, force_alpha, force_lambda, truth, self.dt)
        f_out = np.empty((self.ny, self.nx), self.dt)
        rc = fn(self.h, _pp(g), _pp(b), _ptr(f0a) if f0a is not None else None, C.byref(opts), C.byref(raw), _ptr(f_out))
        if check:
            _check(rc, "run")
        res = Result(raw, tr)
        res.rc = rc
        return f_out, res

    def sgp(self, g, b, f0=None, opts=None, **kw):
        return self._run(self.L.oracle_sgp_run, g, b, f0, opts or default_options(), **kw)

    def rl(self, g, b, f0=None, opts=None, **kw):
        return self._run(self.L.oracle_rl_run, g, b, f0, opts or default_options(), **kw)

    def osem(self, g, b, f0=None, opts=None, **kw):
        """Algorithm 2 (Eq.15 / Eq.22): max_iter cycles over the images; J0 only at the final iterate"""
        return self._run(self.L.oracle_osem_run, g, b, f0, opts or default_options(), **kw)


# ---- paper-level entry points (same argument lists as the CUDA library, host arrays) ----

def _entry(name, p, g, psf, b, f0, ny, nx, opts, dtype, boundary=None, single=False):
    dt = np.dtype(dtype)
    L = lib(dt)
    code = 1 if dt == np.dtype(np.float64) else 0
    g = [_arr(a, dt) for a in g]
    psf = [_arr(a, dt) for a in psf]
    b_arr, b_const = None, np.zeros(p)
    if np.ndim(b[0]) == 0:
        b_const = np.array([float(v) for v in b], dtype=np.float64)
    else:
        b_arr = [_arr(a, dt) for a in b]
    f0a = _arr(f0, dt) if f0 is not None else None
    raw, tr, _keep = _make_result(opts.max_iter)
    f_out = np.empty((ny, nx), dt)
    fn = getattr(L, name)
    f0p = _ptr(f0a) if f0a is not None else None
    maskR = None
    if single:
        rc = fn(_ptr(g[0]), _ptr(psf[0]), _ptr(b_arr[0]) if b_arr else None, C.c_double(b_const[0]), f0p,
                _ptr(f_out), ny, nx, code, C.byref(opts), C.byref(raw))
    elif boundary is None:
        rc = fn(p, _pp(g), _pp(psf), _pp(b_arr) if b_arr else None, _ptr(b_const), f0p, _ptr(f_out), ny, nx,
                code, C.byref(opts), C.byref(raw))
    else:
        oy, ox, sy, sx = boundary
        maskR = np.empty((ny, nx), np.uint8)
        rc = fn(p, _pp(g), _pp(psf), _pp(b_arr) if b_arr else None, _ptr(b_const), oy, ox, sy, sx, ny, nx, f0p,
                _ptr(f_out), _ptr(maskR), code, C.byref(opts), C.byref(raw))
    res = Result(raw, tr)
    res.rc = rc
    res.maskR = maskR
    return f_out, res


def sgp_single(g, psf, b, f0=None, opts=None, dtype=np.float64):
    ny, nx = np.shape(g)
    return _entry("oracle_sgp_single", 1, [g], [psf], [b], f0, ny, nx, opts or default_options(), dtype, single=True)


def rl_single(g, psf, b, f0=None, opts=None, dtype=np.float64):
    ny, nx = np.shape(g)
    return _entry("oracle_rl_single", 1, [g], [psf], [b], f0, ny, nx, opts or default_options(), dtype, single=True)


def sgp_multi(g, psf, b, f0=None, opts=None, dtype=np.float64):
    ny, nx = np.shape(g[0])
    return _entry("oracle_sgp_multi", len(g), g, psf, b, f0, ny, nx, opts or default_options(), dtype)


def rl_multi(g, psf, b, f0=None, opts=None, dtype=np.float64):
    ny, nx = np.shape(g[0])
    return _entry("oracle_rl_multi", len(g), g, psf, b, f0, ny, nx, opts or default_options(), dtype)


def osem_multi(g, psf, b, f0=None, opts=None, dtype=np.float64):
    ny, nx = np.shape(g[0])
    return _entry("oracle_osem_multi", len(g), g, psf, b, f0, ny, nx, opts or default_options(), dtype)


def osem_boundary(g, psf, b, oy, ox, f0=None, opts=None, dtype=np.float64):
    sy, sx = np.shape(g[0]); ny, nx = np.shape(psf[0])
    return _entry("oracle_osem_boundary", len(g), g, psf, b, f0, ny, nx, opts or default_options(), dtype,
                  boundary=(oy, ox, sy, sx))


def sgp_boundary(g, psf, b, oy, ox, f0=None, opts=None, dtype=np.float64):
    sy, sx = np.shape(g[0]); ny, nx = np.shape(psf[0])
    return _entry("oracle_sgp_boundary", len(g), g, psf, b, f0, ny, nx, opts or default_options(), dtype,
                  boundary=(oy, ox, sy, sx))


def rl_boundary(g, psf, b, oy, ox, f0=None, opts=None, dtype=np.float64):
    sy, sx = np.shape(g[0]); ny, nx = np.shape(psf[0])
    return _entry("oracle_rl_boundary", len(g), g, psf, b, f0, ny, nx, opts or default_options(), dtype,
                  boundary=(oy, ox, sy, sx))


def set_threads(n: int) -> None:
    """OpenMP thread count for the oracle's FFT loops (takes effect before the library is first loaded)."""
    os.environ["OMP_NUM_THREADS"] = str(int(n))


# ---- mosaic of sub-domain reconstructions with boundary-effect correction (pin P19) ----

def mosaic_layout(Ny, Nx, ty, tx, sy, sx, ny, nx):
    """The paper's procedure: the Ny x Nx image is partitioned into ty x tx partially overlapping
    sy x sx sub-images; each is merged by zero padding into an ny x nx array (S centred in S-bar: reading A29); from
    each reconstruction the (Ny/ty) x (Nx/tx) non-overlapping part is extracted.  Sub-image t starts at
    clamp(t*N/T - (s - N/T)/2, 0, N - s) (256 -> four 160^2 sub-images at offsets 0 and 96, 128^2 parts extracted).
    Returns one dict per tile: img = (y, x) offset of the sub-image in the image, S = (oy, ox, sy, sx) in S-bar,
    out = (y0, x0, hy, hx) the part of the mosaic it fills (image coordinates), src = (y, x) of that part in S-bar."""
    assert Ny % ty == 0 and Nx % tx == 0 and sy >= Ny // ty and sx >= Nx // tx and sy <= min(Ny, ny) and sx <= min(Nx, nx)
    hy, hx = Ny // ty, Nx // tx
    oy, ox = (ny - sy) // 2, (nx - sx) // 2
    tiles = []
    for iy in range(ty):
        y_img = min(max(iy * hy - (sy - hy) // 2, 0), Ny - sy)
        for ix in range(tx):
            x_img = min(max(ix * hx - (sx - hx) // 2, 0), Nx - sx)
            tiles.append({"img": (y_img, x_img), "S": (oy, ox, sy, sx), "out": (iy * hy, ix * hx, hy, hx),
                          "src": (iy * hy - y_img + oy, ix * hx - x_img + ox)})
    return tiles


def mosaic(alg, g, psf, b, ty, tx, sub, opts=None, dtype=np.float64):
    """alg in {"sgp", "rl", "osem"}; g: p images (Ny x Nx); psf: p PSFs (ny x nx, the S-bar grid of every sub-problem);
    b: p background constants.  Every sub-domain is reconstructed independently by the boundary-effect-corrected
    method (Eq.16-23) and the non-overlapping parts are put together.  Returns (mosaic Ny x Nx, [Result per tile])."""
    opts = opts or default_options()
    Ny, Nx = np.shape(g[0]); ny, nx = np.shape(psf[0])
    fn = {"sgp": sgp_boundary, "rl": rl_boundary, "osem": osem_boundary}[alg]
    out = np.zeros((Ny, Nx), np.dtype(dtype))
    results = []
    for t in mosaic_layout(Ny, Nx, ty, tx, sub[0], sub[1], ny, nx):
        yi, xi = t["img"]; oy, ox, sy, sx = t["S"]
        gs = [np.ascontiguousarray(a[yi:yi + sy, xi:xi + sx]) for a in g]
        f, r = fn(gs, psf, b, oy, ox, None, opts, dtype)
        if r.rc != 0:
            raise OracleError(r.rc, "mosaic tile")
        y0, x0, hy, hx = t["out"]; ys, xs = t["src"]
        out[y0:y0 + hy, x0:x0 + hx] = f[ys:ys + hy, xs:xs + hx]
        results.append(r)
    return out, results
