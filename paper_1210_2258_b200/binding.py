"""Thin ctypes binding of libsgp_b200.so (include/sgp.h): argument marshalling only.

Every step of the SGP / RL iteration runs in the CUDA kernels of the library.  torch is used for
device memory and the stream only.  There is no CPU fallback: if the library cannot be loaded,
importing the symbols raises.  This module never imports the CPU oracle.
"""
from __future__ import annotations

import ctypes as C
import subprocess
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
_CSRC = _PKG / "csrc"
import os as _os
# SGP_B200_LIB: developer override (e.g. the FAST=1 build of csrc/Makefile); the product library is libsgp_b200.so
LIB_PATH = Path(_os.environ["SGP_B200_LIB"]).resolve() if _os.environ.get("SGP_B200_LIB") else _PKG / "libsgp_b200.so"

F32, F64 = 0, 1
STOP_MAXIT, STOP_RELJ, STOP_DISCREPANCY, STOP_MINERR = 0, 1, 2, 3
INIT_USER, INIT_CONST, INIT_ZERO, INIT_G, INIT_CONST_SMOOTH = 0, 1, 2, 3, 4
PSF_CENTER, PSF_CORNER = 0, 1
KIND_SINGLE, KIND_MULTI, KIND_BOUNDARY = 0, 1, 2
ALG_SGP, ALG_RL, ALG_OSEM = 0, 1, 2
STATIC_MAX_ELEMS = 4096 * 4096     # SGP_STATIC_MAX_ELEMS of include/sgp.h
OK, ERR_ARG, ERR_PSF, ERR_DATA, ERR_ALLOC, ERR_CUDA, ERR_LINESEARCH, ERR_NONFINITE, ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5, -6, -7, -8
REASON = {0: "none", 1: "maxit", 2: "relJ", 3: "discrepancy", 4: "minerr"}

EXPORTS = [
    "sgp_options_default", "sgp_result_init", "sgp_strerror", "sgp_version", "sgp_last_cuda_error", "sgp_workspace_bytes", "sgp_plan_workspace_bytes",
    "sgp_release_cached_plans", "sgp_rel_error_static", "sgp_rel_error_static_max",
    "sgp_single", "sgp_multi", "sgp_boundary", "rl_single", "rl_multi", "rl_boundary",
    "osem_multi", "osem_boundary",
    "sgp_single_host", "sgp_multi_host", "sgp_boundary_host", "rl_single_host", "rl_multi_host", "rl_boundary_host",
    "osem_multi_host", "osem_boundary_host",
    "sgp_plan_create", "sgp_plan_create_batched", "sgp_plan_run_batched", "sgp_mosaic", "sgp_mosaic_host", "sgp_plan_set_psf", "sgp_plan_run", "sgp_plan_apply_A", "sgp_plan_apply_AT", "sgp_plan_get_mask",
    "sgp_plan_rfft2", "sgp_plan_irfft2", "sgp_plan_set_profiling", "sgp_plan_get_kernel_ms", "sgp_plan_destroy",
]
PROF_SLOTS = ["K1_ratio_rowfft", "K2_col_conjsum", "K3_rowifft_grad_bb", "K4_project_rowfft", "K5_col_mult", "K6_rowifft_linesearch",
              "K7_backtrack", "R1_rowfft", "R2_col_mult", "R3_rowifft_q_J", "R4_ratio_rowfft", "R5_col_conjsum", "R6_rowifft_update"]


class Options(C.Structure):
    """sgp_options of include/sgp.h"""
    _fields_ = [
        ("beta", C.c_double), ("theta", C.c_double),
        ("alpha0", C.c_double), ("alpha_min", C.c_double), ("alpha_max", C.c_double), ("tau1", C.c_double),
        ("m_alpha", C.c_int), ("alt_start", C.c_int), ("armijo_memory", C.c_int),
        ("L1", C.c_double), ("L2", C.c_double), ("adaptive_L", C.c_int),
        ("max_iter", C.c_int), ("stop_rule", C.c_int), ("tol", C.c_double), ("disc_threshold", C.c_double),
        ("sigma_R", C.c_double), ("max_backtracks", C.c_int), ("psf_origin", C.c_int), ("init", C.c_int),
        ("refresh_every", C.c_int), ("strict", C.c_int), ("check_every", C.c_int),
        ("tile_cols", C.c_int), ("rows_per_block", C.c_int), ("use_graph", C.c_int), ("rl_relax", C.c_double), ("rl_linear", C.c_double),
        ("flux_constraint", C.c_int), ("flux_value", C.c_double), ("init_sigma", C.c_double),
    ]


class _Result(C.Structure):
    _fields_ = [
        ("iterations", C.c_int), ("stop_reason", C.c_int), ("J0_final", C.c_double),
        ("discrepancy_final", C.c_double), ("total_backtracks", C.c_int),
        ("L1_used", C.c_double), ("L2_used", C.c_double), ("n_fft2", C.c_long),
        ("setup_ms", C.c_double), ("loop_ms", C.c_double), ("kernel_launches", C.c_long),
        ("fused_linesearch", C.c_int), ("status", C.c_int),
        ("trace_J", C.POINTER(C.c_double)), ("trace_alpha", C.POINTER(C.c_double)),
        ("trace_lambda", C.POINTER(C.c_double)), ("trace_rule", C.POINTER(C.c_int)),
        ("trace_backtracks", C.POINTER(C.c_int)),
        ("force_alpha", C.POINTER(C.c_double)), ("force_lambda", C.POINTER(C.c_double)),
        ("truth", C.c_void_p), ("trace_err", C.POINTER(C.c_double)), ("err_final", C.c_double),
    ]


class SgpError(RuntimeError):
    def __init__(self, code, what):
        msg = lib().sgp_strerror(code).decode()
        extra = lib().sgp_last_cuda_error().decode() if code == ERR_CUDA else ""
        super().__init__(f"{what}: {msg} ({code}) {extra}")
        self.code = code


def build(force: bool = False, jobs: int = 8) -> None:
    """Compile libsgp_b200.so for sm_100a with nvcc (make -C csrc)."""
    if force:
        subprocess.run(["make", "-C", str(_CSRC), "clean"], check=True, capture_output=True)
    r = subprocess.run(["make", "-C", str(_CSRC), f"-j{jobs}"], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("building libsgp_b200.so failed:\n" + r.stdout[-4000:] + r.stderr[-4000:])


_lib = None


def lib() -> C.CDLL:
    """The loaded C-ABI library.  Raises if it is missing -- there is no fallback path."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} is missing: build it with paper_1210_2258_b200.binding.build() "
                               "(or `make -C paper_1210_2258_b200/csrc`); there is no CPU fallback")
        L = C.CDLL(str(LIB_PATH))
        L.sgp_strerror.restype = C.c_char_p
        L.sgp_version.restype = C.c_char_p
        L.sgp_last_cuda_error.restype = C.c_char_p
        L.sgp_workspace_bytes.restype = C.c_size_t
        L.sgp_plan_workspace_bytes.restype = C.c_size_t
        L.sgp_plan_workspace_bytes.argtypes = [C.c_void_p]
        L.sgp_options_default.restype = None
        L.sgp_release_cached_plans.restype = None
        L.sgp_rel_error_static.restype = C.c_int
        L.sgp_rel_error_static.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_int, C.c_void_p, C.c_void_p]
        L.sgp_rel_error_static_max.restype = C.c_size_t
        L.sgp_rel_error_static_max.argtypes = []
        L.sgp_release_cached_plans.argtypes = []
        L.sgp_result_init.restype = None
        L.sgp_plan_destroy.restype = None
        L.sgp_plan_destroy.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def default_options(**kw) -> Options:
    o = Options()
    lib().sgp_options_default(C.byref(o))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise AttributeError(k)
        setattr(o, k, v)
    return o


def _dtype_code(dt) -> int:
    dt = np.dtype(dt)
    if dt == np.float32:
        return F32
    if dt == np.float64:
        return F64
    raise TypeError(f"unsupported dtype {dt}")


class Result:
    """Python view of sgp_result (traces copied out)."""

    def __init__(self, raw: _Result, tr: dict, rc: int):
        self.rc = rc
        self.iterations = raw.iterations
        self.stop_reason = raw.stop_reason
        self.J0_final = raw.J0_final
        self.discrepancy_final = raw.discrepancy_final
        self.total_backtracks = raw.total_backtracks
        self.L1_used, self.L2_used = raw.L1_used, raw.L2_used
        self.n_fft2 = raw.n_fft2
        self.setup_ms, self.loop_ms = raw.setup_ms, raw.loop_ms
        self.kernel_launches = raw.kernel_launches
        self.fused_linesearch = raw.fused_linesearch
        k = self.iterations
        self.J = tr["J"][: k + 1].copy()
        self.alpha = tr["alpha"][:k].copy()
        self.lam = tr["lambda"][:k].copy()
        self.rule = tr["rule"][:k].copy()
        self.backtracks = tr["backtracks"][:k].copy()
        self.err = tr["err"][: k + 2].copy()
        self.err_final = raw.err_final
        self.maskR = None


def _make_result(max_iter, force_alpha=None, force_lambda=None, traces=True, truth=None):
    n = max_iter + 1
    tr = {"J": np.zeros(n), "alpha": np.zeros(n), "lambda": np.zeros(n),
          "rule": np.zeros(n, np.int32), "backtracks": np.zeros(n, np.int32), "err": np.full(n + 1, np.nan)}
    raw = _Result()
    lib().sgp_result_init(C.byref(raw))
    if traces:
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
    if truth is not None:          # Eq.25: a CUDA tensor holding the true object
        raw.truth = truth.data_ptr()
        raw.trace_err = tr["err"].ctypes.data_as(C.POINTER(C.c_double))
        keep.append(truth)
    return raw, tr, keep


def _torch():
    import torch
    return torch


def _stream_ptr():
    return C.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _dev_ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _pp(tensors):
    """HOST array of device pointers"""
    return (C.c_void_p * len(tensors))(*[t.data_ptr() if t is not None else None for t in tensors])


def _check_dev(t, shape, tdt, name):
    if t is None:
        return
    if not t.is_cuda or not t.is_contiguous() or tuple(t.shape) != tuple(shape) or t.dtype != tdt:
        raise ValueError(f"{name}: expected a contiguous CUDA tensor of shape {tuple(shape)} and dtype {tdt}")


class Plan:
    """sgp_plan: workspace, twiddles, transfer functions and boundary weights for one problem shape.

    psfs: list of p CUDA tensors (ny x nx).  S = (oy, ox, sy, sx) selects a boundary-effect problem
    (PAPER.md:216-238); None = periodic problem on the whole grid.
    """

    def __init__(self, psfs, S=None, opts: Options | None = None, dtype=None):
        torch = _torch()
        self.p = len(psfs)
        self.ny, self.nx = psfs[0].shape
        self.tdt = psfs[0].dtype if dtype is None else dtype
        self.code = F32 if self.tdt == torch.float32 else F64
        self.opts = opts or default_options()
        self.S = S
        kind = KIND_BOUNDARY if S is not None else (KIND_SINGLE if self.p == 1 else KIND_MULTI)
        oy, ox, sy, sx = S if S is not None else (0, 0, self.ny, self.nx)
        self.sy, self.sx = sy, sx
        self.h = C.c_void_p()
        rc = lib().sgp_plan_create(C.byref(self.h), kind, self.p, self.ny, self.nx, oy, ox, sy, sx, self.code, C.byref(self.opts))
        if rc != OK:
            self.h = None
            raise SgpError(rc, "sgp_plan_create")
        for k in psfs:
            _check_dev(k, (self.ny, self.nx), self.tdt, "psf")
        self._psfs = psfs
        rc = lib().sgp_plan_set_psf(self.h, _pp(psfs), _stream_ptr())
        if rc != OK:
            raise SgpError(rc, "sgp_plan_set_psf")

    def close(self):
        if getattr(self, "h", None):
            lib().sgp_plan_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def run(self, algorithm, g, b, f0=None, opts: Options | None = None, f_out=None, force_alpha=None, force_lambda=None,
            traces=True, check=True, truth=None):
        """g: list of p CUDA tensors (sy x sx); b: list of p scalars or p CUDA tensors."""
        torch = _torch()
        o = opts or self.opts
        for t in g:
            _check_dev(t, (self.sy, self.sx), self.tdt, "g")
        b_arr, b_const = None, (C.c_double * self.p)()
        if torch.is_tensor(b[0]):
            for t in b:
                _check_dev(t, (self.sy, self.sx), self.tdt, "b")
            b_arr = _pp(b)
        else:
            for j, v in enumerate(b):
                b_const[j] = float(v)
        _check_dev(f0, (self.ny, self.nx), self.tdt, "f0")
        if f_out is None:
            f_out = torch.empty((self.ny, self.nx), dtype=self.tdt, device=g[0].device)
        _check_dev(truth, (self.ny, self.nx), self.tdt, "truth")
        raw, tr, keep = _make_result(o.max_iter, force_alpha, force_lambda, traces, truth)
        rc = lib().sgp_plan_run(self.h, int(algorithm), _pp(g), b_arr, b_const, _dev_ptr(f0), _dev_ptr(f_out), C.byref(o),
                                C.byref(raw), _stream_ptr())
        res = Result(raw, tr, rc)
        if check and rc != OK:
            raise SgpError(rc, "sgp_plan_run")
        return f_out, res

    def sgp(self, g, b, **kw):
        return self.run(ALG_SGP, g, b, **kw)

    def rl(self, g, b, **kw):
        return self.run(ALG_RL, g, b, **kw)

    def osem(self, g, b, **kw):
        return self.run(ALG_OSEM, g, b, **kw)

    def workspace_bytes(self) -> int:
        return int(lib().sgp_plan_workspace_bytes(self.h))

    def set_profiling(self, on: bool):
        rc = lib().sgp_plan_set_profiling(self.h, int(bool(on)))
        if rc != OK:
            raise SgpError(rc, "sgp_plan_set_profiling")

    def kernel_ms(self):
        """{slot name: (summed ms, launches)} of the last profiled run"""
        n = len(PROF_SLOTS)
        ms, cnt = (C.c_double * n)(), (C.c_long * n)()
        rc = lib().sgp_plan_get_kernel_ms(self.h, ms, cnt)
        if rc != OK:
            raise SgpError(rc, "sgp_plan_get_kernel_ms")
        return {PROF_SLOTS[i]: (ms[i], cnt[i]) for i in range(n) if cnt[i] > 0}

    def apply_A(self, j, x):
        out = _torch().empty_like(x)
        rc = lib().sgp_plan_apply_A(self.h, int(j), _dev_ptr(x), _dev_ptr(out), _stream_ptr())
        if rc != OK:
            raise SgpError(rc, "sgp_plan_apply_A")
        return out

    def apply_AT(self, j, y):
        out = _torch().empty_like(y)
        rc = lib().sgp_plan_apply_AT(self.h, int(j), _dev_ptr(y), _dev_ptr(out), _stream_ptr())
        if rc != OK:
            raise SgpError(rc, "sgp_plan_apply_AT")
        return out

    def mask(self):
        torch = _torch()
        dev = self._psfs[0].device
        m = torch.empty((self.ny, self.nx), dtype=torch.uint8, device=dev)
        a = torch.empty((self.ny, self.nx), dtype=self.tdt, device=dev)
        nR = C.c_long()
        rc = lib().sgp_plan_get_mask(self.h, _dev_ptr(m), _dev_ptr(a), C.byref(nR), _stream_ptr())
        if rc != OK:
            raise SgpError(rc, "sgp_plan_get_mask")
        return m, a, nR.value

    def rfft2(self, x):
        torch = _torch()
        cdt = torch.complex64 if self.tdt == torch.float32 else torch.complex128
        out = torch.empty((self.ny, self.nx // 2 + 1), dtype=cdt, device=x.device)
        rc = lib().sgp_plan_rfft2(self.h, _dev_ptr(x), _dev_ptr(out), _stream_ptr())
        if rc != OK:
            raise SgpError(rc, "sgp_plan_rfft2")
        return out

    def irfft2(self, spec):
        torch = _torch()
        out = torch.empty((self.ny, self.nx), dtype=self.tdt, device=spec.device)
        rc = lib().sgp_plan_irfft2(self.h, _dev_ptr(spec.contiguous()), _dev_ptr(out), _stream_ptr())
        if rc != OK:
            raise SgpError(rc, "sgp_plan_irfft2")
        return out


# ---- one-shot entry points with the names of include/sgp.h ----------------------------------------

def _one_shot(name, g, psf, b, f0, opts, boundary=None, single=False, host=False, check=True, f_out=None):
    """g, psf: lists of arrays (CUDA tensors, or numpy arrays when host=True); b: scalars or arrays."""
    torch = _torch() if not host else None
    p = len(g)
    o = opts or default_options()
    if host:
        dt = np.dtype(g[0].dtype)
        code = _dtype_code(dt)
        g = [np.ascontiguousarray(a, dtype=dt) for a in g]
        psf = [np.ascontiguousarray(a, dtype=dt) for a in psf]
        ny, nx = psf[0].shape
        ptr = lambda a: C.c_void_p(a.ctypes.data) if a is not None else None
        pp = lambda arrs: (C.c_void_p * len(arrs))(*[a.ctypes.data for a in arrs])
        b_is_arr = np.ndim(b[0]) != 0
        b = [np.ascontiguousarray(a, dtype=dt) for a in b] if b_is_arr else b
        f0 = np.ascontiguousarray(f0, dtype=dt) if f0 is not None else None
        if f_out is None:
            f_out = np.empty((ny, nx), dt)
        assert f_out.dtype == dt and f_out.shape == (ny, nx) and f_out.flags.c_contiguous
        maskR = np.empty((ny, nx), np.uint8) if boundary is not None else None
        stream = None
    else:
        tdt = g[0].dtype
        code = F32 if tdt == torch.float32 else F64
        ny, nx = psf[0].shape
        ptr, pp = _dev_ptr, _pp
        b_is_arr = torch.is_tensor(b[0])
        if f_out is None:
            f_out = torch.empty((ny, nx), dtype=tdt, device=g[0].device)
        _check_dev(f_out, (ny, nx), tdt, "f_out")
        maskR = torch.empty((ny, nx), dtype=torch.uint8, device=g[0].device) if boundary is not None else None
        stream = _stream_ptr()
    b_const = (C.c_double * p)(*([0.0] * p if b_is_arr else [float(v) for v in b]))
    raw, tr, _keep = _make_result(o.max_iter)
    fn = getattr(lib(), name + ("_host" if host else ""))
    if single:
        rc = fn(ptr(g[0]), ptr(psf[0]), ptr(b[0]) if b_is_arr else None, C.c_double(b_const[0]), ptr(f0), ptr(f_out), ny, nx, code,
                C.byref(o), C.byref(raw), stream)
    elif boundary is None:
        rc = fn(p, pp(g), pp(psf), pp(b) if b_is_arr else None, b_const, ptr(f0), ptr(f_out), ny, nx, code, C.byref(o), C.byref(raw), stream)
    else:
        oy, ox = boundary
        sy, sx = g[0].shape
        rc = fn(p, pp(g), pp(psf), pp(b) if b_is_arr else None, b_const, oy, ox, sy, sx, ny, nx, ptr(f0), ptr(f_out), ptr(maskR), code,
                C.byref(o), C.byref(raw), stream)
    res = Result(raw, tr, rc)
    res.maskR = maskR
    if check and rc != OK:
        raise SgpError(rc, name)
    return f_out, res


def release_cached_plans() -> None:
    """Free the plan and staging buffer the one-shot calls of this thread keep (include/sgp.h)."""
    lib().sgp_release_cached_plans()


def rel_error_static(f, truth, rho_out, check=True) -> int:
    """sgp_rel_error_static (include/sgp.h): || f - truth || / || truth || (Eq.25) into the one-element float64 DEVICE tensor
    `rho_out`, on torch's current stream, through the entry point that allocates nothing (scratch in a static device array;
    at most STATIC_MAX_ELEMS elements; calls that overlap on the GPU race).  Returns the status code."""
    torch = _torch()
    if f.shape != truth.shape or f.dtype != truth.dtype or not (f.is_cuda and truth.is_cuda and rho_out.is_cuda):
        raise ValueError("f and truth: device tensors of one shape and dtype; rho_out: a device tensor")
    if rho_out.dtype != torch.float64 or rho_out.numel() != 1 or not (f.is_contiguous() and truth.is_contiguous()):
        raise ValueError("rho_out: one float64; f and truth contiguous")
    if f.dtype not in (torch.float32, torch.float64):
        raise TypeError(f"unsupported dtype {f.dtype}")
    code = F32 if f.dtype == torch.float32 else F64
    rc = lib().sgp_rel_error_static(_dev_ptr(f), _dev_ptr(truth), f.numel(), code, _dev_ptr(rho_out), _stream_ptr())
    if rc and check:
        raise SgpError(rc, lib().sgp_last_cuda_error().decode() or "sgp_rel_error_static")
    return rc


def sgp_single(g, psf, b, f0=None, opts=None, host=False, check=True, f_out=None):
    return _one_shot("sgp_single", [g], [psf], [b], f0, opts, single=True, host=host, check=check, f_out=f_out)


def rl_single(g, psf, b, f0=None, opts=None, host=False, check=True, f_out=None):
    return _one_shot("rl_single", [g], [psf], [b], f0, opts, single=True, host=host, check=check, f_out=f_out)


def sgp_multi(g, psf, b, f0=None, opts=None, host=False, check=True, f_out=None):
    return _one_shot("sgp_multi", g, psf, b, f0, opts, host=host, check=check, f_out=f_out)


def rl_multi(g, psf, b, f0=None, opts=None, host=False, check=True, f_out=None):
    return _one_shot("rl_multi", g, psf, b, f0, opts, host=host, check=check, f_out=f_out)


def sgp_boundary(g, psf, b, oy, ox, f0=None, opts=None, host=False, check=True, f_out=None):
    return _one_shot("sgp_boundary", g, psf, b, f0, opts, boundary=(oy, ox), host=host, check=check, f_out=f_out)


def rl_boundary(g, psf, b, oy, ox, f0=None, opts=None, host=False, check=True, f_out=None):
    return _one_shot("rl_boundary", g, psf, b, f0, opts, boundary=(oy, ox), host=host, check=check, f_out=f_out)


def osem_multi(g, psf, b, f0=None, opts=None, host=False, check=True, f_out=None):
    return _one_shot("osem_multi", g, psf, b, f0, opts, host=host, check=check, f_out=f_out)


def osem_boundary(g, psf, b, oy, ox, f0=None, opts=None, host=False, check=True, f_out=None):
    return _one_shot("osem_boundary", g, psf, b, f0, opts, boundary=(oy, ox), host=host, check=check, f_out=f_out)


# ---- batched plans and the mosaic driver ------------------------------------

class BatchedPlan(Plan):
    """sgp_plan_create_batched: nb problems of one geometry and one set of PSFs, every kernel launched once for all of them"""

    def __init__(self, nb, psfs, S=None, opts: Options | None = None):
        torch = _torch()
        self.nb = int(nb)
        self.p = len(psfs)
        self.ny, self.nx = psfs[0].shape
        self.tdt = psfs[0].dtype
        self.code = F32 if self.tdt == torch.float32 else F64
        self.opts = opts or default_options()
        self.S = S
        kind = KIND_BOUNDARY if S is not None else (KIND_SINGLE if self.p == 1 else KIND_MULTI)
        oy, ox, sy, sx = S if S is not None else (0, 0, self.ny, self.nx)
        self.sy, self.sx = sy, sx
        self.h = C.c_void_p()
        rc = lib().sgp_plan_create_batched(C.byref(self.h), self.nb, kind, self.p, self.ny, self.nx, oy, ox, sy, sx, self.code, C.byref(self.opts))
        if rc != OK:
            self.h = None
            raise SgpError(rc, "sgp_plan_create_batched")
        for k in psfs:
            _check_dev(k, (self.ny, self.nx), self.tdt, "psf")
        self._psfs = psfs
        rc = lib().sgp_plan_set_psf(self.h, _pp(psfs), _stream_ptr())
        if rc != OK:
            raise SgpError(rc, "sgp_plan_set_psf")

    def run_batched(self, algorithm, g, b, f0=None, opts: Options | None = None, check=True):
        """g: nb lists of p CUDA tensors; b: nb lists of p scalars.  Returns ([f_out per problem], [Result per problem])."""
        torch = _torch()
        o = opts or self.opts
        flat_g = [t for prob in g for t in prob]
        for t in flat_g:
            _check_dev(t, (self.sy, self.sx), self.tdt, "g")
        n = self.nb * self.p
        b_const = (C.c_double * n)(*[float(v) for prob in b for v in prob])
        f_out = [torch.empty((self.ny, self.nx), dtype=self.tdt, device=flat_g[0].device) for _ in range(self.nb)]
        raws = (_Result * self.nb)()
        trs = []
        for i in range(self.nb):
            lib().sgp_result_init(C.byref(raws[i]))
            tr = {"J": np.zeros(o.max_iter + 1), "alpha": np.zeros(o.max_iter + 1), "lambda": np.zeros(o.max_iter + 1),
                  "rule": np.zeros(o.max_iter + 1, np.int32), "backtracks": np.zeros(o.max_iter + 1, np.int32), "err": np.full(o.max_iter + 2, np.nan)}
            raws[i].trace_J = tr["J"].ctypes.data_as(C.POINTER(C.c_double))
            raws[i].trace_alpha = tr["alpha"].ctypes.data_as(C.POINTER(C.c_double))
            raws[i].trace_lambda = tr["lambda"].ctypes.data_as(C.POINTER(C.c_double))
            raws[i].trace_rule = tr["rule"].ctypes.data_as(C.POINTER(C.c_int))
            raws[i].trace_backtracks = tr["backtracks"].ctypes.data_as(C.POINTER(C.c_int))
            trs.append(tr)
        rc = lib().sgp_plan_run_batched(self.h, int(algorithm), _pp(flat_g), None, b_const, _pp(f0) if f0 is not None else None,
                                        _pp(f_out), C.byref(o), raws, _stream_ptr())
        res = [Result(raws[i], trs[i], raws[i].status) for i in range(self.nb)]
        if check and rc != OK:
            raise SgpError(rc, "sgp_plan_run_batched")
        return f_out, res


def mosaic(algorithm, g, psf, b, ty, tx, sub, opts=None, host=False, check=True):
    """sgp_mosaic / sgp_mosaic_host: g: p images (Ny x Nx); psf: p PSFs (ny x nx); b: p constants; sub = (sy, sx).
    Returns (mosaic Ny x Nx, [Result per tile])."""
    o = opts or default_options()
    p = len(g)
    nb = ty * tx
    if host:
        dt = np.dtype(g[0].dtype)
        code = _dtype_code(dt)
        g = [np.ascontiguousarray(a, dtype=dt) for a in g]; psf = [np.ascontiguousarray(a, dtype=dt) for a in psf]
        Ny, Nx = g[0].shape; ny, nx = psf[0].shape
        f_out = np.empty((Ny, Nx), dt)
        pp = lambda arrs: (C.c_void_p * len(arrs))(*[a.ctypes.data for a in arrs])
        fptr, stream, fn = C.c_void_p(f_out.ctypes.data), None, lib().sgp_mosaic_host
    else:
        torch = _torch()
        tdt = g[0].dtype
        code = F32 if tdt == torch.float32 else F64
        Ny, Nx = g[0].shape; ny, nx = psf[0].shape
        f_out = torch.empty((Ny, Nx), dtype=tdt, device=g[0].device)
        pp, fptr, stream, fn = _pp, _dev_ptr(f_out), _stream_ptr(), lib().sgp_mosaic
    b_const = (C.c_double * p)(*[float(v) for v in b])
    raws = (_Result * nb)()
    trs = []
    for i in range(nb):
        lib().sgp_result_init(C.byref(raws[i]))
        tr = {"J": np.zeros(o.max_iter + 1), "alpha": np.zeros(o.max_iter + 1), "lambda": np.zeros(o.max_iter + 1),
              "rule": np.zeros(o.max_iter + 1, np.int32), "backtracks": np.zeros(o.max_iter + 1, np.int32), "err": np.full(o.max_iter + 2, np.nan)}
        raws[i].trace_J = tr["J"].ctypes.data_as(C.POINTER(C.c_double))
        trs.append(tr)
    rc = fn(int(algorithm), p, pp(g), pp(psf), b_const, Ny, Nx, int(ty), int(tx), int(sub[0]), int(sub[1]), ny, nx, fptr, code,
            C.byref(o), raws, stream)
    res = [Result(raws[i], trs[i], raws[i].status) for i in range(nb)]
    if check and rc != OK:
        raise SgpError(rc, "sgp_mosaic")
    return f_out, res
