"""Helpers for the -m gpu parity tests: move a seeded CSRSystem to the device, build the matching
oracle / CUDA policies from one description, compare results with the stated tolerances."""
from __future__ import annotations

import math

import numpy as np

# one description -> (oracle policy kwargs, CUDA policy kwargs)
POLICY_SPECS = {
    "pcg_fp64": dict(amp=0),
    "amp_fp64_delay": dict(amp=1, u0=0, eta_rule=0),
    "amp_fp16_linear": dict(amp=1, u0=2, eta_rule=1),
    "amp_fp64_delay_strict": dict(amp=1, u0=0, eta_rule=0, eta_safety=0.1, stop_safety=0.9),
    "amp_fp64_delay_strict_t02": dict(amp=1, u0=0, eta_rule=0, eta_safety=0.2, stop_safety=0.8),
    "amp_fp64_delay_strict_t03": dict(amp=1, u0=0, eta_rule=0, eta_safety=0.3, stop_safety=0.7),  # bench.py's headline policy
    "amp_fp64_delay_strict_t05": dict(amp=1, u0=0, eta_rule=0, eta_safety=0.5, stop_safety=0.5),
    "amp_fp32_never": dict(amp=1, u0=1, eta_rule=2),
    "amp_fp64_rms": dict(amp=1, u0=0, eta_rule=0, scale_mode=1),
    "amp_fp64_pow2": dict(amp=1, u0=0, eta_rule=0, scale_mode=2),
    "amp_fp64_delay_lagged": dict(amp=1, u0=0, eta_rule=0, scale_mode=4),
    "amp_fp64_delay_rms": dict(amp=1, u0=0, eta_rule=0, scale_mode=1),
    "amp_fp16_linear_rms": dict(amp=1, u0=2, eta_rule=1, scale_mode=1),
}


def oracle_policy(spec: dict, precond: int = 1):
    import oracle as O

    kw = dict(spec)
    if "C" in kw:
        kw["C_"] = kw.pop("C")
    return O.make_policy(precond=precond, **kw)


def cuda_policy(spec: dict, **extra):
    import paper_2505_04155_b200 as A

    return A.Policy.default(true_residual=1, **spec, **extra)


def to_device(s):
    import torch

    dev = torch.device("cuda", 0)
    return (torch.from_numpy(s.rowptr).to(dev), torch.from_numpy(s.colidx).to(dev), torch.from_numpy(s.vals).to(dev),
            torch.from_numpy(s.b).to(dev))


def iters_close(gpu_iters: int, ref_iters: int) -> bool:
    """north_star: FP64 PCG +-1; AMP within 5 % of the oracle's count (at least 1)."""
    return abs(gpu_iters - ref_iters) <= max(1, math.ceil(0.05 * ref_iters))


def switch_close(a: int, b: int, tol: int = 2) -> bool:
    if a < 0 or b < 0:
        return a == b
    return abs(a - b) <= tol
