"""-m gpu: the lagged variant AMP_SCALE_LAGGED (three kernels per iteration: k_p, k_spmv, k_xrz) against the oracle's
SCALE_LAGGED mode on the same seeded systems: status, iteration count within 5 %, switch iterations +-2, true residual
<= 2 tol (paper policy), in the graph, stream and persistent loops."""
import numpy as np
import pytest

import oracle as O
from workloads import make_config
from gpu_util import iters_close, switch_close, to_device

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")

SMALL = [("c1", 37), ("c2", 19), ("c3", 21), ("c4", 17), ("c5", 30000)]
POLICIES = {"amp_fp64_delay": dict(u0=0, eta_rule=0), "amp_fp16_linear": dict(u0=2, eta_rule=1),
            "amp_fp32_never": dict(u0=1, eta_rule=2)}


@pytest.mark.parametrize("name,size", SMALL)
@pytest.mark.parametrize("pname", list(POLICIES))
def test_lagged_parity(name, size, pname):
    s = make_config(name, size)
    kw = POLICIES[pname]
    ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(scale_mode=O.SCALE_LAGGED, **kw))
    rp, ci, va, b = to_device(s)
    for fuse in (A.FUSE_OFF, A.FUSE_ON):
        with A.AmpPcg(rp, ci, va, fuse_vec=fuse) as h:
            for loop in (A.LOOP_GRAPH, A.LOOP_STREAM, A.LOOP_PERSISTENT, A.LOOP_AUTO):
                x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
                st = h.solve(b, x, s.tol, s.maxit,
                             A.Policy.default(scale_mode=A.SCALE_LAGGED, loop_mode=loop, true_residual=1, x0_zero=1, **kw))
                assert st.status == ref.status == 0
                assert iters_close(st.iters, ref.iters), (st.iters, ref.iters)
                for key in ("it_ur32", "it_uz32", "it_uz16"):
                    assert switch_close(getattr(st, key), getattr(ref, key)), (key, getattr(st, key), getattr(ref, key))
                true = np.linalg.norm(s.b - O.spmv_fp64(s.rowptr, s.colidx, s.vals, x.cpu().numpy())) / np.linalg.norm(s.b)
                assert st.relres_true == pytest.approx(true, rel=1e-6) and true <= 2 * s.tol
                assert st.relres_updated <= s.tol
                if st.loop_mode != A.LOOP_PERSISTENT:
                    # unfused: 3 kernels per iteration + setup, first k_z, residual SpMV, finalize;
                    # fused: mat-vec + k_vec_fused per iteration + setup, first k_z and k_p, residual SpMV, finalize
                    # (a GRAPH body holds 4 iterations: the launches after the last one return at once but count)
                    its = st.iters if st.loop_mode != A.LOOP_GRAPH else (st.iters + 3) // 4 * 4
                    assert h.last_launch_count() == (3 * its + 4 if fuse == A.FUSE_OFF else 2 * its + 5)


def test_lagged_edge_cases():
    s = make_config("c2", 11)
    rp, ci, va, b = to_device(s)
    with A.AmpPcg(rp, ci, va) as h:
        pol = dict(scale_mode=A.SCALE_LAGGED, true_residual=1)
        # x0 != 0, maxit reached, b = 0, x0 exact
        x0 = np.random.default_rng(4).standard_normal(s.n)
        x = torch.from_numpy(x0).cuda()
        st = h.solve(b, x, s.tol, s.maxit, A.Policy.default(**pol))
        ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(scale_mode=O.SCALE_LAGGED), x0=x0)
        assert st.status == 0 and iters_close(st.iters, ref.iters) and st.relres_true <= 2 * s.tol
        x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
        st = h.solve(b, x, 1e-14, 3, A.Policy.default(x0_zero=1, **pol))
        assert st.status == 1 and st.iters == 3
        st = h.solve(torch.zeros_like(b), x, s.tol, 50, A.Policy.default(**pol))
        assert st.status == 0 and st.iters == 0 and float(x.abs().max()) == 0.0
        x = torch.from_numpy(s.xstar).cuda()
        st = h.solve(b, x, s.tol, 50, A.Policy.default(**pol))
        assert st.status == 0 and st.iters == 0
        x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
        st = h.solve(b, x, s.tol, s.maxit, A.Policy.default(loop_mode=A.LOOP_PERSISTENT, x0_zero=1, **pol))
        assert st.status == 0 and st.loop_mode == A.LOOP_PERSISTENT and st.relres_true <= 2 * s.tol
