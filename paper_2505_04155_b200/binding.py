"""ctypes binding of include/amp_pcg.h — argument marshalling only.

The names mirror the C ABI: ``AmpPcg(rowptr, colidx, vals, precond)`` = ``amp_pcg_create``,
``.solve`` = ``amp_pcg_solve``, ``.solve_host`` = ``amp_pcg_solve_host``, ``.spmv`` =
``amp_spmv``, ``.close`` = ``amp_pcg_destroy``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

FP64, FP32, FP16 = 0, 1, 2
ETA_DELAY, ETA_LINEAR, ETA_NEVER = 0, 1, 2
SCALE_NORM2, SCALE_RMS, SCALE_POW2, SCALE_NONE, SCALE_LAGGED = 0, 1, 2, 3, 4
LOOP_AUTO, LOOP_STREAM, LOOP_GRAPH, LOOP_PERSISTENT = 0, 1, 2, 3
PRECOND_NONE, PRECOND_JACOBI, PRECOND_CHEBJACOBI = 0, 1, 2
INDEX_AUTO, INDEX_NO_ALIGN, INDEX_FORCE32 = 0, 1, 2
SPMV_AUTO, SPMV_DIRECT, SPMV_PIPELINED = 0, 1, 2
VEC_AUTO, VEC_DIRECT, VEC_STAGED = 0, 1, 2
FUSE_AUTO, FUSE_OFF, FUSE_ON = 0, 1, 2
K_Z, K_P, K_SPMV, K_XR, K_XRZ, K_CHEB0, K_CHEBSTEP, K_VEC_FUSED = 0, 1, 2, 3, 4, 5, 6, 7
KERNEL_NAMES = {K_Z: "k_z", K_P: "k_p", K_SPMV: "k_spmv", K_XR: "k_xr", K_XRZ: "k_xrz", K_CHEB0: "k_cheb0",
                K_CHEBSTEP: "k_cheb_step", K_VEC_FUSED: "k_vec_fused"}
VEC_R, VEC_Q, VEC_Z, VEC_P, VEC_DINV, VEC_D = 0, 1, 2, 3, 4, 5
STEP_Z, STEP_P, STEP_SPMV, STEP_XR, STEP_XRZ, STEP_CHEB0, STEP_SPMV_Z, STEP_CHEBSTEP = 0, 1, 2, 3, 4, 5, 6, 7

EXPORTED_SYMBOLS = (
    "amp_policy_default", "amp_create_opts_default", "amp_pcg_create", "amp_pcg_create_ex", "amp_pcg_solve",
    "amp_pcg_solve_host", "amp_spmv",
    "amp_pcg_residual_history", "amp_pcg_set_stream", "amp_pcg_last_launch_count", "amp_pcg_destroy",
    "amp_pcg_last_error", "amp_pcg_bytes_per_row", "amp_pcg_spmv_bytes", "amp_pcg_iteration_bytes",
    "amp_pcg_eta_posteriori", "amp_pcg_kernel_times",
    "amp_pcg_debug_set_vector", "amp_pcg_debug_get_vector", "amp_pcg_debug_step",
    "amp_pcg_format_info", "amp_shard_plan", "amp_shard_extract", "amp_pcg_shard_export", "amp_pcg_shard_attach", "amp_pcg_shard_attach_local",
    "amp_pcg_solve_sharded", "amp_spmv_sharded", "amp_xr_update_static",
)
XR_STATIC_MAX_N = 67108864  # AMP_XR_STATIC_MAX_N
SHARD_MAX_WORLD = 16

_HERE = os.path.dirname(os.path.abspath(__file__))


class AmpPcgError(RuntimeError):
    pass


class Policy(C.Structure):
    """amp_policy_t (include/amp_pcg.h)."""

    _fields_ = [
        ("amp", C.c_int32), ("u0", C.c_int32), ("eta_rule", C.c_int32), ("d", C.c_int32), ("ell", C.c_int32),
        ("scale_mode", C.c_int32), ("no_stop", C.c_int32), ("x0_zero", C.c_int32), ("true_residual", C.c_int32),
        ("loop_mode", C.c_int32), ("profile_kernels", C.c_int32), ("reserved0", C.c_int32),
        ("C", C.c_double), ("tau_zs", C.c_double), ("tau_zh", C.c_double), ("eps32", C.c_double),
        ("eta_safety", C.c_double), ("stop_safety", C.c_double),
    ]

    @classmethod
    def default(cls, **overrides) -> "Policy":
        p = cls()
        load_library().amp_policy_default(C.byref(p))
        for k, v in overrides.items():
            if not hasattr(p, k):
                raise AttributeError(k)
            setattr(p, k, v)
        return p


class CreateOpts(C.Structure):
    """amp_create_opts_t (include/amp_pcg.h)."""

    _fields_ = [
        ("struct_bytes", C.c_int32), ("precond", C.c_int32), ("index_format", C.c_int32), ("spmv_kernel", C.c_int32),
        ("spmv_grid_mult", C.c_int32), ("pdl", C.c_int32), ("cheb_degree", C.c_int32), ("reserved0", C.c_int32),
        ("cheb_lmin", C.c_double), ("cheb_lmax", C.c_double), ("stream", C.c_void_p),
        ("halo_lo", C.c_int64), ("halo_hi", C.c_int64), ("vec_kernel", C.c_int32), ("fuse_vec", C.c_int32),
    ]

    @classmethod
    def default(cls, **overrides) -> "CreateOpts":
        o = cls()
        load_library().amp_create_opts_default(C.byref(o))
        for k, v in overrides.items():
            if not hasattr(o, k):
                raise AttributeError(k)
            setattr(o, k, v)
        return o


class Shard(C.Structure):
    """amp_shard_t (include/amp_pcg.h): one rank's block row of the partition."""

    _fields_ = [("row0", C.c_int64), ("row1", C.c_int64), ("halo_lo", C.c_int64), ("halo_hi", C.c_int64), ("nnz", C.c_int64)]


class ShardExport(C.Structure):
    """amp_shard_export_t (include/amp_pcg.h): what a rank publishes to its peers (CUDA IPC handles + geometry)."""

    _fields_ = [("n", C.c_int64), ("halo_lo", C.c_int64), ("halo_hi", C.c_int64), ("guard", C.c_int64),
                ("mem", (C.c_ubyte * 64) * 4), ("off", C.c_int64 * 4)]


class FormatInfo(C.Structure):
    """amp_format_info_t (include/amp_pcg.h)."""

    _fields_ = [("slices", C.c_int64), ("aligned_slices", C.c_int64), ("uniform_slices", C.c_int64),
                ("stored_entries", C.c_int64), ("long_rows", C.c_int64), ("guard", C.c_int64),
                ("index_bits", C.c_int32), ("rows_sorted", C.c_int32), ("spmv_pipelined", C.c_int32),
                ("vec_staged", C.c_int32), ("uniform_width", C.c_int32), ("reserved0", C.c_int32)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved0"}


class KernelTime(C.Structure):
    """amp_kernel_time_t (include/amp_pcg.h)."""

    _fields_ = [("kernel", C.c_int32), ("uz", C.c_int32), ("ur", C.c_int32), ("launches", C.c_int32),
                ("total_ms", C.c_double), ("bytes_per_launch", C.c_double)]


class DebugStep(C.Structure):
    """amp_debug_step_t (include/amp_pcg.h)."""

    _fields_ = [("step", C.c_int32), ("rs", C.c_int32), ("ur", C.c_int32), ("uz", C.c_int32), ("ps", C.c_int32),
                ("ur_n", C.c_int32), ("uz_n", C.c_int32), ("first", C.c_int32),
                ("omega", C.c_double), ("beta", C.c_double), ("alpha", C.c_double), ("omega_n", C.c_double),
                ("sum0", C.c_double), ("sum1", C.c_double)]


class Stats(C.Structure):
    """amp_stats_t (include/amp_pcg.h)."""

    _fields_ = [
        ("status", C.c_int32), ("iters", C.c_int32), ("it_ur32", C.c_int32), ("it_uz32", C.c_int32),
        ("it_uz16", C.c_int32), ("loop_mode", C.c_int32),
        ("bnorm", C.c_double), ("relres_updated", C.c_double), ("relres_true", C.c_double),
        ("solve_ms", C.c_double), ("algorithmic_bytes", C.c_double),
        ("fp16_subnormal", C.c_uint64), ("fp16_flushed", C.c_uint64), ("fp16_inf", C.c_uint64),
    ]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_libs = {}


def library_path(variant: str = "") -> str:
    """In-tree CUDA library; variant "count" = the -DAMP_COUNT_FP16 build (FP16 store counters filled)."""
    return os.path.join(_HERE, "libamp_pcg.so" if not variant else f"libamp_pcg_{variant}.so")


def load_library(variant: str = ""):
    """dlopen the in-tree CUDA library (no build here: see build.py / __graft_entry__.build)."""
    if variant in _libs:
        return _libs[variant]
    path = library_path(variant)
    if not os.path.exists(path):
        raise AmpPcgError(f"{path} is missing: build it with `python -m paper_2505_04155_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.amp_policy_default.restype = None
    L.amp_policy_default.argtypes = [C.POINTER(Policy)]
    L.amp_create_opts_default.restype = None
    L.amp_create_opts_default.argtypes = [C.POINTER(CreateOpts)]
    L.amp_pcg_create.restype = vp
    L.amp_pcg_create.argtypes = [i64, i64, vp, vp, vp, C.c_int]
    L.amp_pcg_create_ex.restype = vp
    L.amp_pcg_create_ex.argtypes = [i64, i64, vp, vp, vp, C.POINTER(CreateOpts)]
    L.amp_pcg_solve.restype = C.c_int
    L.amp_pcg_solve.argtypes = [vp, vp, vp, dbl, i32, C.POINTER(Policy), C.POINTER(Stats)]
    L.amp_pcg_solve_host.restype = C.c_int
    L.amp_pcg_solve_host.argtypes = [vp, vp, vp, dbl, i32, C.POINTER(Policy), C.POINTER(Stats)]
    L.amp_spmv.restype = C.c_int
    L.amp_spmv.argtypes = [vp, C.c_int, C.c_int, vp, vp]
    L.amp_pcg_residual_history.restype = i32
    L.amp_pcg_residual_history.argtypes = [vp, vp, i32]
    L.amp_pcg_set_stream.restype = C.c_int
    L.amp_pcg_set_stream.argtypes = [vp, vp]
    L.amp_pcg_last_launch_count.restype = i64
    L.amp_pcg_last_launch_count.argtypes = [vp]
    L.amp_pcg_destroy.restype = None
    L.amp_pcg_destroy.argtypes = [vp]
    L.amp_pcg_last_error.restype = C.c_char_p
    L.amp_pcg_last_error.argtypes = []
    L.amp_pcg_bytes_per_row.restype = dbl
    L.amp_pcg_bytes_per_row.argtypes = [dbl, C.c_int, C.c_int]
    L.amp_pcg_eta_posteriori.restype = i32
    L.amp_pcg_eta_posteriori.argtypes = [vp, dbl, dbl, vp, i32]
    L.amp_pcg_spmv_bytes.restype = dbl
    L.amp_pcg_spmv_bytes.argtypes = [vp, C.c_int, C.c_int]
    L.amp_pcg_iteration_bytes.restype = dbl
    L.amp_pcg_iteration_bytes.argtypes = [vp, C.c_int, C.c_int]
    L.amp_pcg_kernel_times.restype = i32
    L.amp_pcg_kernel_times.argtypes = [vp, C.POINTER(KernelTime), i32]
    L.amp_pcg_debug_set_vector.restype = C.c_int
    L.amp_pcg_debug_set_vector.argtypes = [vp, C.c_int, C.c_int, vp]
    L.amp_pcg_debug_get_vector.restype = C.c_int
    L.amp_pcg_debug_get_vector.argtypes = [vp, C.c_int, C.c_int, vp]
    L.amp_pcg_debug_step.restype = C.c_int
    L.amp_pcg_debug_step.argtypes = [vp, C.POINTER(DebugStep), vp]
    L.amp_pcg_format_info.restype = C.c_int
    L.amp_pcg_format_info.argtypes = [vp, C.POINTER(FormatInfo)]
    L.amp_shard_plan.restype = C.c_int
    L.amp_shard_plan.argtypes = [i64, vp, vp, i32, C.POINTER(Shard)]
    L.amp_shard_extract.restype = C.c_int
    L.amp_shard_extract.argtypes = [i64, vp, vp, vp, C.POINTER(Shard), vp, vp, vp]
    L.amp_pcg_shard_export.restype = C.c_int
    L.amp_pcg_shard_export.argtypes = [vp, C.POINTER(ShardExport)]
    L.amp_pcg_shard_attach.restype = C.c_int
    L.amp_pcg_shard_attach.argtypes = [vp, i32, i32, C.POINTER(ShardExport)]
    L.amp_pcg_shard_attach_local.restype = C.c_int
    L.amp_pcg_shard_attach_local.argtypes = [C.POINTER(vp), i32]
    L.amp_pcg_solve_sharded.restype = C.c_int
    L.amp_pcg_solve_sharded.argtypes = [C.POINTER(vp), i32, C.POINTER(vp), C.POINTER(vp), dbl, i32, C.POINTER(Policy),
                                        C.POINTER(Stats)]
    L.amp_spmv_sharded.restype = C.c_int
    L.amp_spmv_sharded.argtypes = [C.POINTER(vp), i32, C.c_int, C.c_int, C.POINTER(vp), C.POINTER(vp)]
    L.amp_xr_update_static.restype = C.c_int
    L.amp_xr_update_static.argtypes = [i64, dbl, vp, vp, vp, vp, vp, vp]
    _libs[variant] = L
    return L


def bytes_per_row(m: float, uz: int, ur: int) -> float:
    return float(load_library().amp_pcg_bytes_per_row(float(m), int(uz), int(ur)))


def _last_error(L=None) -> str:
    return (L or load_library()).amp_pcg_last_error().decode("utf-8", "replace")


def xr_update_static(alpha: float, p, q, x, r, delta_out, n: Optional[int] = None) -> None:
    """amp_xr_update_static: x += alpha p, r -= alpha q, delta_out[0] = ||r|| (FP64 torch CUDA tensors, x and r updated
    in place) on torch's current stream, without a handle and without any device allocation by the library — for
    callers whose process can't cudaMalloc any more (all device memory already in their own pool) or can't afford its
    device-wide synchronisation.  n <= XR_STATIC_MAX_N; calls that may overlap on one GPU must be ordered by the caller
    (they share one static scratch array); make the first call on a device outside stream capture.  Asynchronous."""
    import torch

    L = load_library()
    n = int(p.numel() if n is None else n)
    for t in (p, q, x, r, delta_out):
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.device == x.device):
            raise AmpPcgError("xr_update_static: contiguous float64 CUDA tensors on one device expected")
    if min(p.numel(), q.numel(), x.numel(), r.numel()) < n or delta_out.numel() < 1:
        raise AmpPcgError("xr_update_static: a tensor is shorter than n")
    with torch.cuda.device(x.device):
        rc = L.amp_xr_update_static(n, float(alpha), p.data_ptr(), q.data_ptr(), x.data_ptr(), r.data_ptr(),
                                    delta_out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise AmpPcgError(f"amp_xr_update_static failed ({rc}): {_last_error(L)}")


class AmpPcg:
    """One SPD matrix in CSR on the current CUDA device (amp_pcg_create_ex ... amp_pcg_destroy).

    ``rowptr`` (int32[n+1]), ``colidx`` (int32[nnz]) and ``vals`` (float64[nnz]) are CUDA torch
    tensors; they are borrowed by the library, so this object keeps references to them.
    ``opts``: keyword overrides of amp_create_opts_t (index_format, spmv_kernel, spmv_grid_mult, pdl);
    the create() kernels run on torch's current stream.  ``variant="count"`` loads the counting build.
    """

    def __init__(self, rowptr, colidx, vals, precond: int = PRECOND_JACOBI, variant: str = "", **opts):
        import torch

        if not (rowptr.is_cuda and colidx.is_cuda and vals.is_cuda):
            raise AmpPcgError("AmpPcg needs CUDA tensors (there is no CPU fallback)")
        if rowptr.dtype != torch.int32 or colidx.dtype != torch.int32 or vals.dtype != torch.float64:
            raise AmpPcgError("rowptr/colidx must be int32 and vals float64")
        self._keep = (rowptr.contiguous(), colidx.contiguous(), vals.contiguous())
        self.n = int(rowptr.numel() - 1)
        self.nnz = int(colidx.numel())
        self.device = vals.device
        self._torch = torch
        self._L = L = load_library(variant)
        o = CreateOpts()
        L.amp_create_opts_default(C.byref(o))
        o.precond = int(precond)
        for k, v in opts.items():
            if not hasattr(o, k) or k in ("struct_bytes", "stream"):
                raise AttributeError(k)
            setattr(o, k, v)
        with torch.cuda.device(self.device):
            o.stream = torch.cuda.current_stream(self.device).cuda_stream
            self._h = L.amp_pcg_create_ex(self.n, self.nnz, self._keep[0].data_ptr(), self._keep[1].data_ptr(),
                                          self._keep[2].data_ptr(), C.byref(o))
        if not self._h:
            raise AmpPcgError(_last_error(L))

    # -- helpers --------------------------------------------------------------------------
    def _sync_stream(self):
        s = self._torch.cuda.current_stream(self.device).cuda_stream
        self._L.amp_pcg_set_stream(self._h, C.c_void_p(s))

    def _check(self, rc: int, allow=(0, 1, -2)):
        if rc not in allow:
            raise AmpPcgError(f"amp_pcg error {rc}: {_last_error(self._L)}")

    # -- C ABI ----------------------------------------------------------------------------
    def solve(self, b, x, tol: float, maxit: int, policy: Optional[Policy] = None) -> Stats:
        """amp_pcg_solve: b, x float64 CUDA tensors of length n; x is x0 on entry, x_m on exit."""
        torch = self._torch
        if b.dtype != torch.float64 or x.dtype != torch.float64 or not b.is_cuda or not x.is_cuda:
            raise AmpPcgError("b and x must be float64 CUDA tensors")
        if b.numel() != self.n or x.numel() != self.n or not b.is_contiguous() or not x.is_contiguous():
            raise AmpPcgError("b and x must be contiguous with n elements")
        st = Stats()
        with torch.cuda.device(self.device):
            self._sync_stream()
            rc = self._L.amp_pcg_solve(self._h, b.data_ptr(), x.data_ptr(), float(tol), int(maxit),
                                       C.byref(policy) if policy is not None else None, C.byref(st))
        self._check(rc)
        self._last_iters = int(st.iters)
        return st

    def solve_host(self, b_host, x_host, tol: float, maxit: int, policy: Optional[Policy] = None) -> Stats:
        """amp_pcg_solve_host: b, x are HOST float64 buffers (pinned torch tensors or numpy arrays)."""
        st = Stats()
        bp = b_host.data_ptr() if hasattr(b_host, "data_ptr") else b_host.ctypes.data
        xp = x_host.data_ptr() if hasattr(x_host, "data_ptr") else x_host.ctypes.data
        with self._torch.cuda.device(self.device):
            self._sync_stream()
            rc = self._L.amp_pcg_solve_host(self._h, bp, xp, float(tol), int(maxit),
                                            C.byref(policy) if policy is not None else None, C.byref(st))
        self._check(rc)
        self._last_iters = int(st.iters)
        return st

    def spmv(self, p, mat_prec: int = FP64, out=None):
        """amp_spmv: q = A p.  p: float64/float32/float16 CUDA tensor (float16: length padded to 8)."""
        torch = self._torch
        vec_prec = {torch.float64: FP64, torch.float32: FP32, torch.float16: FP16}[p.dtype]
        if p.numel() < self.n or not p.is_contiguous():
            raise AmpPcgError("p must be contiguous with at least n elements")
        qdt = torch.float64 if mat_prec == FP64 else torch.float32
        q = out if out is not None else torch.empty(self.n, dtype=qdt, device=self.device)
        if q.dtype != qdt or q.numel() < self.n:
            raise AmpPcgError("out has the wrong dtype/size")
        with torch.cuda.device(self.device):
            self._sync_stream()
            rc = self._L.amp_spmv(self._h, int(mat_prec), vec_prec, p.data_ptr(), q.data_ptr())
        self._check(rc, allow=(0,))
        return q

    def residual_history(self) -> np.ndarray:
        """amp_pcg_residual_history: ||r_t||, t = 0..iters of the last solve (host numpy array)."""
        buf = np.empty(self._last_iters + 1, dtype=np.float64)
        m = self._L.amp_pcg_residual_history(self._h, buf.ctypes.data, buf.size)
        if m < 0:
            raise AmpPcgError(_last_error(self._L))
        return buf[:m]

    _last_iters = -1

    def last_launch_count(self) -> int:
        return int(self._L.amp_pcg_last_launch_count(self._h))

    def eta_posteriori(self, C_: float = 1.0, eps32: float = 0.0) -> np.ndarray:
        """amp_pcg_eta_posteriori: eta_hat_m(k), k = 0..iters, of the last solve (host numpy array)."""
        buf = np.empty(max(self._last_iters + 1, 1), dtype=np.float64)
        m = self._L.amp_pcg_eta_posteriori(self._h, float(C_), float(eps32), buf.ctypes.data, buf.size)
        if m < 0:
            raise AmpPcgError(_last_error(self._L))
        return buf[:m]

    def spmv_bytes(self, mat_prec: int, vec_prec: int) -> float:
        """amp_pcg_spmv_bytes: compulsory bytes of one mat-vec with the matrix format this handle built."""
        return float(self._L.amp_pcg_spmv_bytes(self._h, int(mat_prec), int(vec_prec)))

    def iteration_bytes(self, uz: int, ur: int) -> float:
        """amp_pcg_iteration_bytes: compulsory bytes of one iteration in phase (u_z, u_r)."""
        return float(self._L.amp_pcg_iteration_bytes(self._h, int(uz), int(ur)))

    def format_info(self) -> FormatInfo:
        """amp_pcg_format_info: what create() built for this matrix."""
        fi = FormatInfo()
        self._check(self._L.amp_pcg_format_info(self._h, C.byref(fi)), allow=(0,))
        return fi

    def kernel_times(self):
        """amp_pcg_kernel_times: per (kernel, u_z, u_r) records of the last solve made with profile_kernels=1."""
        buf = (KernelTime * 64)()
        m = self._L.amp_pcg_kernel_times(self._h, buf, 64)
        if m < 0:
            raise AmpPcgError(_last_error(self._L))
        return [dict(kernel=KERNEL_NAMES[r.kernel], uz=r.uz, ur=r.ur, launches=r.launches, total_ms=r.total_ms,
                     bytes_per_launch=r.bytes_per_launch) for r in buf[:m]]

    # -- diagnostic entry points (parity tests) -------------------------------------------
    _TORCH_DT = None

    def _dtype(self, prec: int):
        torch = self._torch
        return {FP64: torch.float64, FP32: torch.float32, FP16: torch.float16}[prec]

    def debug_set_vector(self, which: int, t):
        """amp_pcg_debug_set_vector: copy a CUDA tensor of n elements into the work vector stored in t.dtype."""
        torch = self._torch
        prec = {torch.float64: FP64, torch.float32: FP32, torch.float16: FP16}[t.dtype]
        if t.numel() != self.n or not t.is_cuda or not t.is_contiguous():
            raise AmpPcgError("debug_set_vector needs a contiguous CUDA tensor of n elements")
        with torch.cuda.device(self.device):
            self._sync_stream()
            self._check(self._L.amp_pcg_debug_set_vector(self._h, int(which), prec, t.data_ptr()), allow=(0,))

    def debug_get_vector(self, which: int, prec: int):
        torch = self._torch
        out = torch.empty(self.n, dtype=self._dtype(prec), device=self.device)
        with torch.cuda.device(self.device):
            self._sync_stream()
            self._check(self._L.amp_pcg_debug_get_vector(self._h, int(which), int(prec), out.data_ptr()), allow=(0,))
        return out

    def debug_step(self, step: int, x=None, **kw) -> DebugStep:
        """amp_pcg_debug_step: one step of the loop with caller-given scalars / precisions (see the header)."""
        io = DebugStep(step=int(step), omega=1.0, beta=0.0, alpha=0.0, omega_n=1.0)
        for k, v in kw.items():
            if not hasattr(io, k):
                raise AttributeError(k)
            setattr(io, k, v)
        with self._torch.cuda.device(self.device):
            self._sync_stream()
            rc = self._L.amp_pcg_debug_step(self._h, C.byref(io), x.data_ptr() if x is not None else None)
        self._check(rc, allow=(0,))
        return io

    def close(self):
        if getattr(self, "_h", None):
            self._L.amp_pcg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


# ---- row-sharded solve (include/amp_pcg.h "row-sharded solve") ------------------------------------------------------
def shard_plan(rowptr: np.ndarray, colidx: np.ndarray, world: int):
    """amp_shard_plan: block-row partition of a HOST CSR pattern over `world` ranks; returns a list of Shard."""
    L = load_library()
    rowptr = np.ascontiguousarray(rowptr, dtype=np.int32)
    colidx = np.ascontiguousarray(colidx, dtype=np.int32)
    out = (Shard * int(world))()
    rc = L.amp_shard_plan(len(rowptr) - 1, rowptr.ctypes.data, colidx.ctypes.data, int(world), out)
    if rc != 0:
        raise AmpPcgError(f"amp_shard_plan error {rc}: {_last_error(L)}")
    return list(out)


def shard_extract(rowptr: np.ndarray, colidx: np.ndarray, vals: np.ndarray, shard: Shard):
    """amp_shard_extract: the block row of `shard` as HOST CSR arrays with columns shifted to [halo_lo | owned | halo_hi]."""
    L = load_library()
    rowptr = np.ascontiguousarray(rowptr, dtype=np.int32)
    colidx = np.ascontiguousarray(colidx, dtype=np.int32)
    vals = np.ascontiguousarray(vals, dtype=np.float64)
    rows = int(shard.row1 - shard.row0)
    rp = np.empty(rows + 1, dtype=np.int32)
    ci = np.empty(max(int(shard.nnz), 1), dtype=np.int32)
    va = np.empty(max(int(shard.nnz), 1), dtype=np.float64)
    rc = L.amp_shard_extract(len(rowptr) - 1, rowptr.ctypes.data, colidx.ctypes.data, vals.ctypes.data, C.byref(shard),
                             rp.ctypes.data, ci.ctypes.data, va.ctypes.data)
    if rc != 0:
        raise AmpPcgError(f"amp_shard_extract error {rc}: {_last_error(L)}")
    return rp, ci[:int(shard.nnz)], va[:int(shard.nnz)]


def _vp_array(ptrs):
    return (C.c_void_p * len(ptrs))(*[C.c_void_p(int(p)) for p in ptrs])


class ShardGroup:
    """The ranks of a sharded system that THIS process drives: all of them (``attach_local``: handles on one device or
    on peer-accessible devices) or one (``attach_ipc``: one process per GPU; the export blobs are all-gathered by the
    caller, e.g. with torch.distributed).  Argument marshalling only."""

    def __init__(self, handles):
        self.handles = list(handles)
        self._L = self.handles[0]._L
        self._torch = self.handles[0]._torch

    @classmethod
    def attach_local(cls, handles) -> "ShardGroup":
        g = cls(handles)
        arr = _vp_array([h._h for h in g.handles])
        rc = g._L.amp_pcg_shard_attach_local(arr, len(g.handles))
        if rc != 0:
            raise AmpPcgError(f"amp_pcg_shard_attach_local error {rc}: {_last_error(g._L)}")
        return g

    @staticmethod
    def export(handle) -> bytes:
        """amp_pcg_shard_export: this rank's blob (bytes) for the all-gather."""
        e = ShardExport()
        rc = handle._L.amp_pcg_shard_export(handle._h, C.byref(e))
        if rc != 0:
            raise AmpPcgError(f"amp_pcg_shard_export error {rc}: {_last_error(handle._L)}")
        return bytes(e)

    @classmethod
    def attach_ipc(cls, handle, rank: int, blobs) -> "ShardGroup":
        """amp_pcg_shard_attach: blobs[r] = export() of rank r, for every rank of the group."""
        g = cls([handle])
        arr = (ShardExport * len(blobs))(*[ShardExport.from_buffer_copy(b) for b in blobs])
        rc = g._L.amp_pcg_shard_attach(handle._h, int(rank), len(blobs), arr)
        if rc != 0:
            raise AmpPcgError(f"amp_pcg_shard_attach error {rc}: {_last_error(g._L)}")
        return g

    def _streams(self):
        for h in self.handles:
            with self._torch.cuda.device(h.device):
                h._sync_stream()

    def solve(self, b, x, tol: float, maxit: int, policy: Optional[Policy] = None):
        """amp_pcg_solve_sharded: b[i], x[i] = float64 CUDA block rows of the local ranks; returns a list of Stats."""
        torch = self._torch
        for h, bi, xi in zip(self.handles, b, x):
            if bi.dtype != torch.float64 or xi.dtype != torch.float64 or bi.numel() != h.n or xi.numel() != h.n or \
                    not (bi.is_cuda and xi.is_cuda and bi.is_contiguous() and xi.is_contiguous()):
                raise AmpPcgError("b[i] and x[i] must be contiguous float64 CUDA tensors with the rank's n entries")
        st = (Stats * len(self.handles))()
        self._streams()
        rc = self._L.amp_pcg_solve_sharded(_vp_array([h._h for h in self.handles]), len(self.handles),
                                           _vp_array([t.data_ptr() for t in b]), _vp_array([t.data_ptr() for t in x]),
                                           float(tol), int(maxit), C.byref(policy) if policy is not None else None, st)
        if rc not in (0, 1, -2):
            raise AmpPcgError(f"amp_pcg_solve_sharded error {rc}: {_last_error(self._L)}")
        for h, s in zip(self.handles, st):
            h._last_iters = int(s.iters)
        return list(st)

    def spmv(self, p, mat_prec: int = FP64):
        """amp_spmv_sharded: q = A p; p[i] = the local ranks' blocks (float64 / float32 / float16 CUDA tensors)."""
        torch = self._torch
        vec_prec = {torch.float64: FP64, torch.float32: FP32, torch.float16: FP16}[p[0].dtype]
        qdt = torch.float64 if mat_prec == FP64 else torch.float32
        q = [torch.empty(h.n, dtype=qdt, device=h.device) for h in self.handles]
        for h, pi in zip(self.handles, p):
            if pi.numel() != h.n or not pi.is_cuda or not pi.is_contiguous() or pi.dtype != p[0].dtype:
                raise AmpPcgError("p[i] must be a contiguous CUDA tensor with the rank's n entries")
        self._streams()
        rc = self._L.amp_spmv_sharded(_vp_array([h._h for h in self.handles]), len(self.handles), int(mat_prec), vec_prec,
                                      _vp_array([t.data_ptr() for t in p]), _vp_array([t.data_ptr() for t in q]))
        if rc != 0:
            raise AmpPcgError(f"amp_spmv_sharded error {rc}: {_last_error(self._L)}")
        return q

    def close(self):
        for h in self.handles:
            h.close()
