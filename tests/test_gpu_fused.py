"""-m gpu: the fused vector kernel (csrc/vec_fused.cuh; create option fuse_vec = AMP_FUSE_ON): x/r of iteration k and
z, p of iteration k + 1 in ONE cooperative kernel with a grid barrier at each of the two true dependencies of
Algorithm 4.1 (delta before the scaling of z, rho before beta).  Same phase functions as the stand-alone kernels (bitwise
per-step parity: tests/test_gpu_steps.py), so the whole solves must agree with the oracle and with the unfused loop to the
tolerances of DESIGN.md section 4: iteration counts, switch iterations, residual history, true residual, x."""
import numpy as np
import pytest

from workloads import make_config
from gpu_util import POLICY_SPECS, cuda_policy, iters_close, oracle_policy, switch_close, to_device

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")
O = pytest.importorskip("oracle")

POLICIES = ["pcg_fp64", "amp_fp64_delay", "amp_fp16_linear", "amp_fp64_delay_strict", "amp_fp64_delay_lagged", "amp_fp32_never",
            "amp_fp64_delay_rms"]


@pytest.mark.parametrize("name,size", [("c3", 21), ("c2", 33), ("c4", 40), ("c5", 30011), ("c1", 9), ("c2", 64)])
def test_fused_loop_matches_oracle_and_unfused_loop(name, size):
    s = make_config(name, size)
    rp, ci, va, b = to_device(s)
    with A.AmpPcg(rp, ci, va, fuse_vec=A.FUSE_ON) as hf, A.AmpPcg(rp, ci, va, fuse_vec=A.FUSE_OFF) as hd:
        for pname in POLICIES:
            spec = POLICY_SPECS[pname]
            ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, oracle_policy(spec))
            for lm in (A.LOOP_GRAPH, A.LOOP_STREAM):
                x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
                xd = torch.zeros(s.n, dtype=torch.float64, device="cuda")
                st = hf.solve(b, x, s.tol, s.maxit, cuda_policy(spec, x0_zero=1, loop_mode=lm))
                sd = hd.solve(b, xd, s.tol, s.maxit, cuda_policy(spec, x0_zero=1, loop_mode=lm))
                assert st.status == ref.status == 0, (pname, lm, st.status)
                assert iters_close(st.iters, ref.iters) and abs(st.iters - sd.iters) <= 1, (pname, st.iters, sd.iters, ref.iters)
                for key in ("it_ur32", "it_uz32", "it_uz16"):
                    assert switch_close(getattr(st, key), getattr(ref, key)), (pname, key, getattr(st, key), getattr(ref, key))
                assert st.relres_true <= (1.0 if spec.get("eta_safety", 1.0) < 1.0 else 2.0) * s.tol
                assert float(torch.linalg.norm(x - xd)) <= 1e-6 * float(torch.linalg.norm(xd))
                assert np.allclose(hf.residual_history()[:15], ref.hist[:15], rtol=1e-4)
                assert hf.last_launch_count() <= (3 if hf.format_info().spmv_pipelined else 2) * (st.iters + 3) + 6


def test_fused_loop_edge_cases():
    s = make_config("c3", 16)
    rp, ci, va, b = to_device(s)
    spec = POLICY_SPECS["amp_fp64_delay"]
    with A.AmpPcg(rp, ci, va, fuse_vec=A.FUSE_ON) as h:
        rng = np.random.default_rng(2)
        x0 = rng.uniform(-1, 1, s.n)
        ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, oracle_policy(spec), x0=x0)
        x = torch.from_numpy(x0).cuda()
        st = h.solve(b, x, s.tol, s.maxit, cuda_policy(spec))
        assert st.status == 0 and abs(st.iters - ref.iters) <= 1 and st.relres_true <= 2 * s.tol
        # b = 0; maxit; an exact initial guess; breakdown on an indefinite matrix
        x = torch.from_numpy(x0).cuda()
        st = h.solve(torch.zeros_like(b), x, s.tol, s.maxit, cuda_policy(spec))
        assert st.status == 0 and st.iters == 0 and float(x.abs().max()) == 0.0
        x = torch.zeros_like(b)
        st = h.solve(b, x, s.tol, 5, cuda_policy(spec, x0_zero=1))
        assert st.status == 1 and st.iters == 5
        xs = torch.from_numpy(ref.x).cuda()
        st = h.solve(b, xs, 1e-6, s.maxit, cuda_policy(spec))
        assert st.status == 0 and st.iters == 0
        # per-kernel profile names the fused kernel
        x = torch.zeros_like(b)
        h.solve(b, x, s.tol, s.maxit, cuda_policy(spec, x0_zero=1, loop_mode=A.LOOP_STREAM, profile_kernels=1))
        names = {r["kernel"] for r in h.kernel_times()}
        assert names == {"k_spmv", "k_vec_fused"}
    n = 64
    rp_ = np.arange(n + 1, dtype=np.int32)
    ci_ = np.arange(n, dtype=np.int32)
    va_ = np.ones(n)
    va_[n // 2] = -1.0  # indefinite: p^T A p < 0 appears
    with A.AmpPcg(torch.from_numpy(rp_).cuda(), torch.from_numpy(ci_).cuda(), torch.from_numpy(va_).cuda(), A.PRECOND_NONE,
                  fuse_vec=A.FUSE_ON) as h:
        bb = torch.ones(n, dtype=torch.float64, device="cuda")
        bb[n // 2] = 20.0
        x = torch.zeros(n, dtype=torch.float64, device="cuda")
        st = h.solve(bb, x, 1e-12, 50, A.Policy.default(amp=0, loop_mode=A.LOOP_GRAPH))
        assert st.status == -2
