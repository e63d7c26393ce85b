"""CPU-side checks of the C ABI (no compute calls): the library loads, exports every symbol that
include/amp_pcg.h declares, the ctypes structs match the C layout, the policy defaults are the
paper's, and the algorithmic byte model reproduces the paper's Table 2."""
import ctypes as C
import json
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = json.load(open(os.path.join(ROOT, "tests", "golden", "paper_printed_values.json")))


@pytest.fixture(scope="module")
def A():
    sys.path.insert(0, ROOT)
    from paper_2505_04155_b200 import build as B

    B.build()
    import paper_2505_04155_b200 as A

    return A


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "amp_pcg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(amp_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(A):
    L = A.load_library()
    names = _declared_functions()
    assert len(names) >= 11
    for nm in names:
        assert hasattr(L, nm), nm
    assert set(names) == set(A.EXPORTED_SYMBOLS)
    # the built code is sm_100a SASS
    out = subprocess.run(["cuobjdump", "-lelf", A.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_struct_layout_matches_c(A, tmp_path):
    # compile a tiny C program against the header and compare sizeof/offsetof with ctypes
    probes = [("amp_policy_t", A.Policy, ["C", "stop_safety", "profile_kernels"]),
              ("amp_stats_t", A.Stats, ["bnorm", "fp16_inf"]),
              ("amp_create_opts_t", A.CreateOpts, ["pdl", "cheb_degree", "cheb_lmax", "stream", "halo_lo", "halo_hi", "vec_kernel"]),
              ("amp_shard_t", A.Shard, ["row1", "halo_hi", "nnz"]),
              ("amp_format_info_t", A.FormatInfo, ["uniform_slices", "guard", "index_bits", "uniform_width"]),
              ("amp_shard_export_t", A.ShardExport, ["guard", "mem", "off"]),
              ("amp_kernel_time_t", A.KernelTime, ["launches", "bytes_per_launch"]),
              ("amp_debug_step_t", A.DebugStep, ["first", "omega", "sum1"])]
    body, want = [], []
    for cname, ct, fields in probes:
        body.append(f'printf("%zu\\n", sizeof({cname}));')
        want.append(C.sizeof(ct))
        for f in fields:
            body.append(f'printf("%zu\\n", offsetof({cname}, {f}));')
            want.append(getattr(ct, f).offset)
    src = tmp_path / "layout.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "amp_pcg.h"\nint main(void){' + "".join(body) + 'return 0;}\n')
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(t) for t in subprocess.check_output([str(exe)], text=True).split()]
    assert got == want


def test_create_opts_defaults_and_validation(A):
    o = A.CreateOpts.default()
    assert o.struct_bytes == C.sizeof(A.CreateOpts) and o.precond == A.PRECOND_JACOBI
    assert (o.index_format, o.spmv_kernel, o.spmv_grid_mult, o.pdl) == (A.INDEX_AUTO, A.SPMV_AUTO, 0, 1)
    assert (o.cheb_degree, o.cheb_lmin, o.cheb_lmax) == (2, 0.0, 0.0)  # PAPER.md:461 "second-order"; bounds computed in create()
    # a struct of another size (an older / newer header) is refused before anything touches the device
    import numpy as np

    L = A.load_library()
    bad = A.CreateOpts.default()
    bad.struct_bytes = 8
    a = np.array([0, 1], dtype=np.int32)
    h = L.amp_pcg_create_ex(1, 1, a.ctypes.data, a.ctypes.data, np.array([1.0]).ctypes.data, C.byref(bad))
    assert not h and b"struct_bytes" in L.amp_pcg_last_error()


def test_policy_defaults_are_the_papers(A):
    p = A.Policy.default()
    d = GOLD["defaults"]
    t = GOLD["thresholds_5_1"]
    assert (p.d, p.ell, p.C) == (d["d"], d["ell"], d["C"])
    assert (p.tau_zs, p.tau_zh) == (t["tau_zs"], t["tau_zh"])
    assert p.eps32 == 2.0 ** -24 and p.amp == 1 and p.u0 == A.FP64 and p.eta_rule == A.ETA_DELAY
    assert p.eta_safety == 1.0 and p.stop_safety == 1.0 and p.scale_mode == A.SCALE_NORM2


def test_byte_model_reproduces_table2(A):
    # Table 2 rows (vector kernels) = our K_z (+ the inner product re-read), K_p, K_xr models.
    # bytes_per_row(m=0) - rowptr/p/q of the SpMV leaves exactly the three vector kernels.
    t2 = GOLD["table2_bytes_per_dof"]
    phases = [(A.FP64, A.FP64), (A.FP16, A.FP64), (A.FP16, A.FP32)]  # (u_z, u_r): FP64, phase 1, phase 2
    for i, (uz, ur) in enumerate(phases):
        sz = {A.FP64: 8, A.FP32: 4, A.FP16: 2}[uz]
        sr = {A.FP64: 8, A.FP32: 4}[ur]
        vec = A.bytes_per_row(0.0, uz, ur) - (4 + sz + sr)
        # paper: axpy and updatePCG exactly; zamx+innerProd are ONE fused kernel here, which saves the
        # innerProd re-read (z, r) and keeps 1/diag in FP32 instead of FP16 (+2 B, R6)
        k_p, k_xr = 3 * sz, 16 + sz + 3 * sr
        assert k_p == t2["axpy"][i] and k_xr == t2["updatePCG"][i]
        k_z = vec - k_p - k_xr
        paper_zamx = t2["zamx"][i]
        assert k_z == paper_zamx + (2 if uz == A.FP16 else 0)
        assert k_z < paper_zamx + t2["innerProd"][i]
    # totals of BASELINE.md section 3: 12m+116, 12m+76, 8m+56
    m = 6.95
    assert A.bytes_per_row(m, A.FP64, A.FP64) == pytest.approx(12 * m + 116)
    assert A.bytes_per_row(m, A.FP16, A.FP64) == pytest.approx(12 * m + 76)
    assert A.bytes_per_row(m, A.FP16, A.FP32) == pytest.approx(8 * m + 56)
    assert A.bytes_per_row(m, A.FP32, A.FP32) == pytest.approx(8 * m + 68)


def test_theorem_3_1_worked_numbers():
    # transcription check of the formula with the paper's example numbers
    import math

    g = GOLD["theorem_3_1_example"]
    delta, kappa = g["delta"], g["kappa"]
    theta = math.asin(delta)
    dprime = 2 * math.sin(theta) * math.sqrt(kappa)
    kp = kappa * (1 + delta) / (1 - delta)
    sigma = (math.sqrt(kp) - 1) / (math.sqrt(kp) + 1)
    K = math.sqrt((2 + 16 * dprime * kp / (kp - 1) ** 2) / (1 + sigma ** 4))
    assert dprime < 1
    assert K == pytest.approx(g["K_approx"], abs=0.005)
    assert kp / kappa - 1 == pytest.approx(g["kappa_rel_increase_approx"], abs=2e-4)


def test_no_cpu_fallback_without_gpu(A):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np

    rp = torch.tensor([0, 1], dtype=torch.int32)
    with pytest.raises(A.AmpPcgError):
        A.AmpPcg(rp, torch.tensor([0], dtype=torch.int32), torch.tensor([1.0], dtype=torch.float64))
    # calling the C entry point directly with host memory must fail loudly too
    L = A.load_library()
    a = np.array([0, 1], dtype=np.int32)
    h = L.amp_pcg_create(1, 1, a.ctypes.data, a.ctypes.data, np.array([1.0]).ctypes.data, 1)
    assert not h and b"CUDA" in L.amp_pcg_last_error()
