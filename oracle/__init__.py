"""CPU oracle for AMP-PCG (arXiv 2505.04155) — TEST INFRASTRUCTURE, not product code.

Thin ctypes wrapper over ``oracle/amp_pcg_oracle.cpp`` (plain C++, g++ -O2 -fopenmp).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import this package; the CUDA library never does, and this package never
imports ``paper_2505_04155_b200``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Callable, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "amp_pcg_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_amp_pcg.so")

FP64, FP32, FP16 = 0, 1, 2
ETA_DELAY, ETA_LINEAR, ETA_NEVER = 0, 1, 2
SCALE_NORM2, SCALE_RMS, SCALE_POW2, SCALE_NONE, SCALE_LAGGED = 0, 1, 2, 3, 4
PRECOND_NONE, PRECOND_JACOBI, PRECOND_CHEBJACOBI = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile the oracle shared library in-tree (building the checker is not using it)."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    flags = ["-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-std=c++17"]
    has_fma = False
    try:
        with open("/proc/cpuinfo") as f:
            has_fma = " fma " in f.read().replace("\n", " ")
    except OSError:
        pass
    if has_fma:
        flags.append("-mfma")  # std::fma -> one instruction instead of a libm call
    subprocess.check_call(["g++", *flags, _SRC, "-o", _LIB])
    return _LIB


class _Policy(C.Structure):
    _fields_ = [
        ("amp", C.c_int32), ("u0", C.c_int32), ("eta_rule", C.c_int32), ("d", C.c_int32), ("ell", C.c_int32),
        ("scale_mode", C.c_int32), ("no_stop", C.c_int32), ("strict_rounding", C.c_int32),
        ("accumulate64", C.c_int32), ("precond", C.c_int32), ("cheb_degree", C.c_int32), ("pad0", C.c_int32),
        ("cheb_lmin", C.c_double), ("cheb_lmax", C.c_double),
        ("C", C.c_double), ("tau_zs", C.c_double), ("tau_zh", C.c_double), ("eps32", C.c_double),
        ("eta_safety", C.c_double), ("stop_safety", C.c_double),
    ]


class _Stats(C.Structure):
    _fields_ = [
        ("status", C.c_int32), ("iters", C.c_int32), ("it_ur32", C.c_int32), ("it_uz32", C.c_int32),
        ("it_uz16", C.c_int32),
        ("bnorm", C.c_double), ("relres_updated", C.c_double), ("relres_true", C.c_double),
        ("fp16_subnormal", C.c_int64), ("fp16_flushed", C.c_int64), ("fp16_inf", C.c_int64),
        ("fp16_stored", C.c_int64),
    ]


_TRACE = C.CFUNCTYPE(None, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                     C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p)

_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_round_fp32.restype = C.c_double
        L.orc_round_fp32.argtypes = [C.c_double]
        L.orc_round_fp16.restype = C.c_double
        L.orc_round_fp16.argtypes = [C.c_double]
        L.orc_round_array.restype = None
        L.orc_round_array.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_int]
        L.orc_dot.restype = C.c_double
        L.orc_dot.argtypes = [C.c_int64, C.c_void_p, C.c_void_p]
        L.orc_spmv_fp64.restype = None
        L.orc_spmv_fp64.argtypes = [C.c_int64] + [C.c_void_p] * 5
        L.orc_spmv_fp32.restype = None
        L.orc_spmv_fp32.argtypes = [C.c_int64] + [C.c_void_p] * 5 + [C.c_int]
        L.orc_eta.restype = C.c_double
        L.orc_eta.argtypes = [C.POINTER(_Policy), C.c_void_p, C.c_int32]
        L.orc_eta_posteriori.restype = C.c_double
        L.orc_eta_posteriori.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double]
        L.orc_select_uz.restype = C.c_int32
        L.orc_select_uz.argtypes = [C.POINTER(_Policy), C.c_double]
        L.orc_step_z.restype = None
        L.orc_step_z.argtypes = [C.c_int64, C.c_void_p, C.c_double, C.c_void_p, C.c_int32, C.c_int32, C.c_int32,
                                 C.c_void_p, C.c_void_p]
        L.orc_step_p.restype = None
        L.orc_step_p.argtypes = [C.c_int64, C.c_double, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
        L.orc_step_xr.restype = None
        L.orc_step_xr.argtypes = [C.c_int64, C.c_double, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
        L.orc_classify_fp16.restype = C.c_int32
        L.orc_classify_fp16.argtypes = [C.c_double, C.c_double]
        L.orc_cheb_default_bounds.restype = None
        L.orc_cheb_default_bounds.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_cheb_coeffs.restype = None
        L.orc_cheb_coeffs.argtypes = [C.c_int32, C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_cheb_first.restype = None
        L.orc_cheb_first.argtypes = [C.c_int64, C.c_void_p, C.c_double, C.c_void_p, C.c_double, C.c_int32, C.c_void_p, C.c_void_p]
        L.orc_cheb_step.restype = None
        L.orc_cheb_step.argtypes = [C.c_int64, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                    C.c_int32, C.c_void_p, C.c_void_p]
        L.orc_cheb_apply.restype = None
        L.orc_cheb_apply.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                     C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_int32, C.c_int32, C.c_void_p,
                                     C.c_void_p, C.c_void_p]
        L.orc_amp_pcg.restype = C.c_int32
        L.orc_amp_pcg.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.c_double, C.c_int32, C.POINTER(_Policy), C.POINTER(_Stats), C.c_void_p,
                                  C.c_void_p, C.c_void_p]
        assert L.orc_sizeof_policy() == C.sizeof(_Policy)
        assert L.orc_sizeof_stats() == C.sizeof(_Stats)
        _lib = L
    return _lib


def make_policy(amp: int = 1, u0: int = FP64, eta_rule: int = ETA_DELAY, d: int = 10, ell: int = 5, C_: float = 1.0,
                tau_zs: float = 1e-4, tau_zh: float = 1e-6, eps32: float = 2.0 ** -24, eta_safety: float = 1.0,
                stop_safety: float = 1.0, scale_mode: int = SCALE_NORM2, no_stop: int = 0,
                strict_rounding: int = 0, accumulate64: int = 0, precond: int = PRECOND_JACOBI, cheb_degree: int = 2,
                cheb_lmin: float = 0.0, cheb_lmax: float = 0.0) -> _Policy:
    """Paper defaults: d=10, C=1, ell=5 (:400), tau (5.1) (:404-405), eps32 = 2^-24 (:354)."""
    return _Policy(amp=amp, u0=u0, eta_rule=eta_rule, d=d, ell=ell, scale_mode=scale_mode, no_stop=no_stop,
                   strict_rounding=strict_rounding, accumulate64=accumulate64, precond=precond, cheb_degree=cheb_degree,
                   cheb_lmin=cheb_lmin, cheb_lmax=cheb_lmax, C=C_,
                   tau_zs=tau_zs, tau_zh=tau_zh, eps32=eps32, eta_safety=eta_safety, stop_safety=stop_safety)


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _round(v, prec: int) -> np.ndarray:
    a = np.ascontiguousarray(np.atleast_1d(np.asarray(v, dtype=np.float64)))
    out = np.empty_like(a)
    lib().orc_round_array(a.size, _ptr(a), _ptr(out), prec)
    return out


def round_fp16(v) -> np.ndarray:
    """IEEE binary16 round-to-nearest-even of doubles, returned as doubles."""
    return _round(v, FP16)


def round_fp32(v) -> np.ndarray:
    """IEEE binary32 round-to-nearest-even of doubles, returned as doubles."""
    return _round(v, FP32)


def dot(a: np.ndarray, b: np.ndarray) -> float:
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    return float(lib().orc_dot(len(a), _ptr(a), _ptr(b)))


def spmv_fp64(rowptr, colidx, vals, p) -> np.ndarray:
    n = len(rowptr) - 1
    p = np.ascontiguousarray(p, dtype=np.float64)
    q = np.empty(n, dtype=np.float64)
    lib().orc_spmv_fp64(n, _ptr(rowptr), _ptr(colidx), _ptr(vals), _ptr(p), _ptr(q))
    return q


def spmv_fp32(rowptr, colidx, vals, p, accumulate64: int = 0) -> np.ndarray:
    """u_r = FP32 mat-vec: values rounded to FP32 once, float fma chain; p holds the stored values."""
    n = len(rowptr) - 1
    p = np.ascontiguousarray(p, dtype=np.float64)
    v32 = np.ascontiguousarray(vals, dtype=np.float64).astype(np.float32)
    q = np.empty(n, dtype=np.float64)
    lib().orc_spmv_fp32(n, _ptr(rowptr), _ptr(colidx), _ptr(v32), _ptr(p), _ptr(q), int(accumulate64))
    return q


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def step_z(r, omega: float, dinv, ur: int, uz: int, strict: int = 0):
    """O2: z = RN_{u_z}((r omega) dinv) (Alg 4.1 lines 4-5).  Returns (z, counts[inf, flushed, subnormal])."""
    r, dinv = _f64(r), _f64(dinv)
    z = np.empty_like(r)
    counts = np.zeros(3, dtype=np.int64)
    lib().orc_step_z(r.size, _ptr(r), float(omega), _ptr(dinv), int(ur), int(uz), int(strict), _ptr(z), _ptr(counts))
    return z, counts


def step_p(beta: float, p, z, uz: int):
    """O5: p = RN_{u_z}(fma(beta, p, z)) (Alg 4.1 line 10).  Returns (p_new, counts)."""
    z = _f64(z)
    p = np.array(p, dtype=np.float64, copy=True)
    counts = np.zeros(3, dtype=np.int64)
    lib().orc_step_p(z.size, float(beta), _ptr(z), int(uz), _ptr(p), _ptr(counts))
    return p, counts


def step_xr(alpha: float, p, q, x, r, ur: int):
    """O9, O10: x = fma(alpha, p, x) (FP64); r = RN_{u_r}(fma(-alpha, q, r)) (Alg 4.1 lines 15-16).  Returns (x, r)."""
    p, q = _f64(p), _f64(q)
    x = np.array(x, dtype=np.float64, copy=True)
    r = np.array(r, dtype=np.float64, copy=True)
    lib().orc_step_xr(p.size, float(alpha), _ptr(p), _ptr(q), int(ur), _ptr(x), _ptr(r))
    return x, r


def classify_fp16(unrounded: float, stored: float) -> int:
    """1 = became inf, 2 = flushed to zero, 3 = subnormal, 0 = anything else."""
    return int(lib().orc_classify_fp16(float(unrounded), float(stored)))


def cheb_default_bounds(rowptr, colidx, vals, ratio: float = 30.0):
    """(lmin, lmax): Gershgorin bound of D^-1 A and lmax / ratio (the defaults of the Chebyshev-Jacobi preconditioner)."""
    lo, hi = C.c_double(), C.c_double()
    lib().orc_cheb_default_bounds(len(rowptr) - 1, _ptr(rowptr), _ptr(colidx), _ptr(vals), float(ratio), C.byref(lo), C.byref(hi))
    return lo.value, hi.value


def cheb_coeffs(s: int, lmin: float, lmax: float):
    """(1/theta, c1[0..s-1], c2[0..s-1]) of the Chebyshev recurrence (index 0 unused)."""
    it = C.c_double()
    c1 = np.zeros(s + 1); c2 = np.zeros(s + 1)
    lib().orc_cheb_coeffs(int(s), float(lmin), float(lmax), C.byref(it), _ptr(c1), _ptr(c2))
    return it.value, c1[:s], c2[:s]


def cheb_first(r, omega: float, dinv, inv_theta: float, uz: int):
    r, dinv = _f64(r), _f64(dinv)
    d = np.empty_like(r); z = np.empty_like(r)
    lib().orc_cheb_first(r.size, _ptr(r), float(omega), _ptr(dinv), float(inv_theta), int(uz), _ptr(d), _ptr(z))
    return d, z


def cheb_step(r, omega: float, w, dinv, c1: float, c2: float, uz: int, d, z):
    r, w, dinv = _f64(r), _f64(w), _f64(dinv)
    d = np.array(d, dtype=np.float64, copy=True); z = np.array(z, dtype=np.float64, copy=True)
    lib().orc_cheb_step(r.size, _ptr(r), float(omega), _ptr(w), _ptr(dinv), float(c1), float(c2), int(uz), _ptr(d), _ptr(z))
    return d, z


def cheb_apply(rowptr, colidx, vals, r, omega: float, dinv, s: int, lmin: float, lmax: float, uz: int = FP64, ur: int = FP64):
    """z = M^-1 (omega r): s sweeps of Chebyshev-accelerated Jacobi in precisions (u_z, u_r)."""
    rowptr = np.ascontiguousarray(rowptr, dtype=np.int32); colidx = np.ascontiguousarray(colidx, dtype=np.int32)
    vals = _f64(vals); r = _f64(r); dinv = _f64(dinv)
    v32 = vals.astype(np.float32)
    n = r.size
    z = np.empty(n); d = np.empty(n); w = np.empty(n)
    lib().orc_cheb_apply(n, _ptr(rowptr), _ptr(colidx), _ptr(vals), _ptr(v32), _ptr(r), float(omega), _ptr(dinv), int(s),
                         float(lmin), float(lmax), int(uz), int(ur), _ptr(z), _ptr(d), _ptr(w))
    return z


def eta(policy: _Policy, hist: np.ndarray, k: int) -> float:
    hist = np.ascontiguousarray(hist, dtype=np.float64)
    return float(lib().orc_eta(C.byref(policy), _ptr(hist), int(k)))


def eta_posteriori(hist: np.ndarray, k: int, C_: float = 1.0, eps32: float = 2.0 ** -24, eps64: float = 2.0 ** -53) -> float:
    """eta_hat_m(k) of (4.7), with m = len(hist) - 1 (the whole history of a finished run)."""
    hist = np.ascontiguousarray(hist, dtype=np.float64)
    return float(lib().orc_eta_posteriori(_ptr(hist), len(hist) - 1, int(k), float(C_), float(eps32), float(eps64)))


def select_uz(policy: _Policy, nu: float) -> int:
    return int(lib().orc_select_uz(C.byref(policy), float(nu)))


@dataclass
class Result:
    status: int
    iters: int
    it_ur32: int
    it_uz32: int
    it_uz16: int
    bnorm: float
    relres_updated: float
    relres_true: float
    fp16_subnormal: int
    fp16_flushed: int
    fp16_inf: int
    fp16_stored: int
    x: np.ndarray
    hist: np.ndarray


def amp_pcg(rowptr, colidx, vals, b, tol: float, maxit: int, policy: Optional[_Policy] = None,
            x0: Optional[np.ndarray] = None,
            trace: Optional[Callable[[int, dict], None]] = None) -> Result:
    """Run Algorithm 4.1 (policy.amp=1) or Algorithm 3.1 (policy.amp=0) of the paper on the CPU."""
    L = lib()
    policy = policy if policy is not None else make_policy()
    rowptr = np.ascontiguousarray(rowptr, dtype=np.int32)
    colidx = np.ascontiguousarray(colidx, dtype=np.int32)
    vals = np.ascontiguousarray(vals, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    n = len(rowptr) - 1
    x = np.zeros(n, dtype=np.float64) if x0 is None else np.array(x0, dtype=np.float64, copy=True)
    hist = np.zeros(maxit + 2, dtype=np.float64)
    st = _Stats()
    cb = None
    if trace is not None:
        names = ("rho", "beta", "gamma", "alpha", "delta_k", "delta_next", "omega", "eta", "ur", "uz")

        def _cb(k, px, pr, pz, pp, pq, ps, _user):
            vec = lambda ptr: np.ctypeslib.as_array(ptr, shape=(n,)).copy()
            sc = np.ctypeslib.as_array(ps, shape=(10,))
            trace(int(k), dict(x=vec(px), r=vec(pr), z=vec(pz), p=vec(pp), q=vec(pq),
                               **{nm: float(sc[i]) for i, nm in enumerate(names)}))

        cb = _TRACE(_cb)
    L.orc_amp_pcg(n, _ptr(rowptr), _ptr(colidx), _ptr(vals), _ptr(b), _ptr(x), float(tol), int(maxit),
                  C.byref(policy), C.byref(st), _ptr(hist), C.cast(cb, C.c_void_p) if cb else None, None)
    return Result(st.status, st.iters, st.it_ur32, st.it_uz32, st.it_uz16, st.bnorm, st.relres_updated,
                  st.relres_true, st.fp16_subnormal, st.fp16_flushed, st.fp16_inf, st.fp16_stored, x,
                  hist[: st.iters + 1].copy())


def pcg_fp64(rowptr, colidx, vals, b, tol: float, maxit: int, precond: int = PRECOND_JACOBI, **kw) -> Result:
    """PCG(FP64): Algorithm 3.1 literally."""
    return amp_pcg(rowptr, colidx, vals, b, tol, maxit, make_policy(amp=0, precond=precond), **kw)
