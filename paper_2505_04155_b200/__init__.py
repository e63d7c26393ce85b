"""B200-native AMP-PCG iteration loop (arXiv 2505.04155) — thin Python binding over the C ABI.

Everything numerical runs inside ``libamp_pcg.so`` (hand-written sm_100a CUDA, see
``csrc/`` and ``include/amp_pcg.h``).  This module only marshals arguments: torch tensors
provide device memory and the current stream.  There is no CPU fallback — if the CUDA library
or a GPU is missing, calls raise.
"""
from .binding import (  # noqa: F401
    AmpPcg,
    Policy,
    Stats,
    CreateOpts,
    KernelTime,
    FormatInfo,
    DebugStep,
    AmpPcgError,
    bytes_per_row,
    xr_update_static, XR_STATIC_MAX_N,
    load_library,
    library_path,
    FP64, FP32, FP16,
    ETA_DELAY, ETA_LINEAR, ETA_NEVER,
    SCALE_NORM2, SCALE_RMS, SCALE_POW2, SCALE_NONE, SCALE_LAGGED,
    LOOP_AUTO, LOOP_STREAM, LOOP_GRAPH, LOOP_PERSISTENT,
    PRECOND_NONE, PRECOND_JACOBI, PRECOND_CHEBJACOBI,
    INDEX_AUTO, INDEX_NO_ALIGN, INDEX_FORCE32,
    SPMV_AUTO, SPMV_DIRECT, SPMV_PIPELINED,
    VEC_AUTO, VEC_DIRECT, VEC_STAGED,
    FUSE_AUTO, FUSE_OFF, FUSE_ON,
    K_Z, K_P, K_SPMV, K_XR, K_XRZ, K_CHEB0, K_CHEBSTEP, K_VEC_FUSED, KERNEL_NAMES,
    VEC_R, VEC_Q, VEC_Z, VEC_P, VEC_DINV, VEC_D,
    STEP_Z, STEP_P, STEP_SPMV, STEP_XR, STEP_XRZ, STEP_CHEB0, STEP_SPMV_Z, STEP_CHEBSTEP,
    EXPORTED_SYMBOLS,
    Shard, ShardExport, ShardGroup, shard_plan, shard_extract, SHARD_MAX_WORLD,
)
