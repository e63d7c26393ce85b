"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(loop_mode AUTO, x0 = 0), against values the CPU oracle wrote to
tests/golden/oracle_full_size.json (tests/golden/make_oracle_golden.py, oracle-only script):

* SpMV: 64 sampled rows of q = A p for a fixed probe vector, <= 1e-13 relative, plus ||q||_2 (stored values), and the
  WHOLE vector bit for bit against the oracle's mat-vec called here, in FP64 and in the u_r = FP32 phase with FP16 p
  (both sides: one fma chain per row in CSR order);
* solves: iteration count within 5 % (+-1 for FP64 PCG), switch iterations +-2, status,
  true residual <= 2 tol (paper policy) / <= tol (strict policy) recomputed here in FP64 by torch
  (an independent sparse mat-vec, not the library's).
"""
import json
import os

import numpy as np
import pytest

from workloads import make_config
from gpu_util import POLICY_SPECS, cuda_policy, iters_close, switch_close, to_device

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")

GOLD_PATH = os.path.join(os.path.dirname(__file__), "golden", "oracle_full_size.json")
GOLD = json.load(open(GOLD_PATH)) if os.path.exists(GOLD_PATH) else {}


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4", "c5"])
def test_full_size_against_oracle_golden(name):
    if name not in GOLD:
        pytest.skip("no golden for " + name)
    g = GOLD[name]
    s = make_config(name)
    assert (s.n, s.nnz) == (g["n"], g["nnz"])
    rp, ci, va, b = to_device(s)
    with A.AmpPcg(rp, ci, va) as h:
        # --- SpMV on sampled rows ---
        p = 2.0 * np.modf(np.arange(s.n) * 0.6180339887498949)[0] - 1.0
        q = h.spmv(torch.from_numpy(p).cuda(), A.FP64)
        rows = np.array(g["spmv_probe"]["rows"])
        qs = q[torch.from_numpy(rows).cuda()].cpu().numpy()
        qref = np.array(g["spmv_probe"]["q"])
        assert np.max(np.abs(qs - qref)) <= 1e-13 * max(np.max(np.abs(qref)), float(q.abs().max()))
        assert float(torch.linalg.norm(q)) == pytest.approx(g["spmv_probe"]["q_norm2"], rel=1e-12)
        # the whole vector, bit for bit (FP64; FP32 matrix copy with FP16-stored p), against the oracle called here
        import oracle as O

        assert np.array_equal(q.cpu().numpy(), O.spmv_fp64(s.rowptr, s.colidx, s.vals, p))
        npad = (s.n + 7) // 8 * 8
        p16 = torch.zeros(npad, dtype=torch.float16, device="cuda")
        p16[:s.n] = torch.from_numpy(p).cuda().to(torch.float16)
        q32 = h.spmv(p16, A.FP32).cpu().numpy()
        q32_ref = O.spmv_fp32(s.rowptr, s.colidx, s.vals, p16[:s.n].cpu().numpy().astype(np.float64))
        assert np.array_equal(q32.astype(np.float64), q32_ref)
        # the IN-LOOP mat-vec kernels (k_spmv / k_spmv_uni / k_spmv_pipe through amp_pcg_debug_step, not the stand-alone
        # k_spmv_any above) over the whole vector at full size — the full grid of k_spmv_uni, every round of k_spmv_pipe's
        # stage ring (31 on c4): q bit for bit, gamma = q^T p to reduction accuracy (Alg 4.1 lines 11-13)
        if name in ("c2", "c3", "c4"):
            rnd = {0: lambda a: a, 2: lambda a: a.astype(np.float16).astype(np.float64)}
            tdt = {0: torch.float64, 1: torch.float32, 2: torch.float16}
            for ur, uz in ((0, 0), (1, 0), (1, 2)):
                pz = rnd[uz](p)
                q_ref = O.spmv_fp64(s.rowptr, s.colidx, s.vals, pz) if ur == 0 else O.spmv_fp32(s.rowptr, s.colidx, s.vals, pz)
                h.debug_set_vector(A.VEC_P, torch.from_numpy(pz).cuda().to(tdt[uz]))
                h.debug_set_vector(A.VEC_Q, torch.full((s.n,), 7.0, dtype=tdt[ur], device="cuda"))
                io = h.debug_step(A.STEP_SPMV, rs=ur, ur=ur, uz=uz, ps=uz, ur_n=ur, uz_n=uz)
                q_in = h.debug_get_vector(A.VEC_Q, ur).cpu().numpy().astype(np.float64)
                assert np.array_equal(q_in, q_ref), (name, ur, uz, int((q_in != q_ref).sum()))
                bound = s.n * 2.0 ** -53 * float(np.abs(q_ref * pz).sum())
                assert abs(io.sum0 - O.dot(q_ref, pz)) <= bound, (name, ur, uz, io.sum0)
        # independent FP64 mat-vec for the true residual
        crow = rp.to(torch.int64)
        At = torch.sparse_csr_tensor(crow, ci.to(torch.int64), va, size=(s.n, s.n))
        bn = float(torch.linalg.norm(b))
        for pname, ref in g["policies"].items():
            spec = POLICY_SPECS[pname]
            x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
            st = h.solve(b, x, s.tol, s.maxit, cuda_policy(spec, loop_mode=A.LOOP_AUTO, x0_zero=1))
            assert st.status == ref["status"] == 0
            assert iters_close(st.iters, ref["iters"]), (pname, st.iters, ref["iters"])
            if pname == "pcg_fp64":
                assert abs(st.iters - ref["iters"]) <= 1
            for key in ("it_ur32", "it_uz32", "it_uz16"):
                assert switch_close(getattr(st, key), ref[key]), (pname, key, getattr(st, key), ref[key])
            true = float(torch.linalg.norm(b - At @ x)) / bn
            assert st.relres_true == pytest.approx(true, rel=1e-5)
            strict = spec.get("eta_safety", 1.0) < 1.0
            assert true <= (1.0 if strict else 2.0) * s.tol, (pname, true)
            assert st.relres_updated <= s.tol
            if s.xstar is not None and name != "c3":
                err = float(torch.linalg.norm(x - torch.from_numpy(s.xstar).cuda())) / np.linalg.norm(s.xstar)
                assert err <= 1e-4
