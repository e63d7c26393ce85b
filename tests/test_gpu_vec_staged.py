"""-m gpu: the bulk-copy staged vector kernels (csrc/vec_pipe.cuh; create option vec_kernel = AMP_VEC_STAGED) in whole
solves: same iteration counts, switch iterations and residuals as the oracle (tolerances of DESIGN.md section 4) and as
the direct kernels, for every policy and loop driver that uses them, on sizes that exercise one partial stage, several
stages per block, fewer elements than blocks, and n < 8 (only the direct tail).  The per-step bitwise comparison of both
kernel families against the oracle is tests/test_gpu_steps.py."""
import numpy as np
import pytest

from workloads import make_config
from gpu_util import POLICY_SPECS, cuda_policy, iters_close, oracle_policy, switch_close, to_device

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")
O = pytest.importorskip("oracle")

POLICIES = ["pcg_fp64", "amp_fp64_delay", "amp_fp16_linear", "amp_fp64_delay_strict", "amp_fp64_delay_lagged", "amp_fp32_never"]


@pytest.mark.parametrize("name,size", [("c3", 21), ("c2", 33), ("c4", 40), ("c5", 30011), ("c1", 9)])
def test_staged_vector_kernels_in_whole_solves(name, size):
    s = make_config(name, size)
    rp, ci, va, b = to_device(s)
    with A.AmpPcg(rp, ci, va, vec_kernel=A.VEC_STAGED) as hs, A.AmpPcg(rp, ci, va, vec_kernel=A.VEC_DIRECT) as hd:
        for pname in POLICIES:
            spec = POLICY_SPECS[pname]
            ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, oracle_policy(spec))
            for lm in (A.LOOP_GRAPH, A.LOOP_STREAM):
                x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
                xd = torch.zeros(s.n, dtype=torch.float64, device="cuda")
                st = hs.solve(b, x, s.tol, s.maxit, cuda_policy(spec, x0_zero=1, loop_mode=lm))
                sd = hd.solve(b, xd, s.tol, s.maxit, cuda_policy(spec, x0_zero=1, loop_mode=lm))
                assert st.status == ref.status == 0, (pname, st.status)
                assert iters_close(st.iters, ref.iters) and abs(st.iters - sd.iters) <= 1, (pname, st.iters, sd.iters, ref.iters)
                for key in ("it_ur32", "it_uz32", "it_uz16"):
                    assert switch_close(getattr(st, key), getattr(ref, key)), (pname, key, getattr(st, key), getattr(ref, key))
                assert st.relres_true <= (1.0 if spec.get("eta_safety", 1.0) < 1.0 else 2.0) * s.tol
                assert float(torch.linalg.norm(x - xd)) <= 1e-6 * float(torch.linalg.norm(xd))
                hist = hs.residual_history()
                assert np.allclose(hist[:15], ref.hist[:15], rtol=1e-4)   # as tests/test_gpu_parity.py: the sums are added in another order


def test_tiny_systems_and_x0():
    # n < 8: no full group of 8 elements, everything goes through the direct tail; n = 9: one group + tail
    for n in (1, 5, 9, 17):
        rng = np.random.default_rng(n)
        dense = rng.standard_normal((n, n))
        M = dense @ dense.T + n * np.eye(n)
        rp = np.arange(0, n * n + 1, n, dtype=np.int32)
        ci = np.tile(np.arange(n, dtype=np.int32), n)
        va = M.reshape(-1).copy()
        b = rng.standard_normal(n)
        x0 = rng.standard_normal(n)
        ref = O.amp_pcg(rp, ci, va, b, 1e-10, 100, O.make_policy(), x0=x0)
        t = [torch.from_numpy(a).cuda() for a in (rp, ci, va)]
        with A.AmpPcg(*t, A.PRECOND_JACOBI, vec_kernel=A.VEC_STAGED) as h:
            x = torch.from_numpy(x0).cuda()
            st = h.solve(torch.from_numpy(b).cuda(), x, 1e-10, 100, A.Policy.default(true_residual=1, loop_mode=A.LOOP_GRAPH))
            assert st.status == 0 and abs(st.iters - ref.iters) <= 1 and st.relres_true <= 2e-10
            assert np.allclose(x.cpu().numpy(), np.linalg.solve(M, b), rtol=1e-8, atol=1e-10)
