"""-m gpu: attainable-accuracy runs (policy.no_stop) and the a-posteriori indicator (4.7) through the
C ABI: amp_pcg_eta_posteriori on the library's own residual history equals the oracle's definition applied to the same
history, and bounds the true residual the GPU run stagnates at."""
import numpy as np
import pytest

import oracle as O
from workloads import make_config, paper_example

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")


def _dev(s):
    return [torch.from_numpy(a).cuda() for a in (s.rowptr, s.colidx, s.vals, s.b)]


@pytest.mark.parametrize("ex,tol", [(1, 1e-6), (1, 1e-8), (4, 1e-8), (6, 1e-6)])
def test_attainable_accuracy_of_the_paper_examples(ex, tol):
    s = paper_example(ex)
    rp, ci, va, b = _dev(s)
    ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, tol, 150,
                    O.make_policy(amp=1, u0=0, eta_rule=0, precond=0, no_stop=1, tau_zs=0.0, tau_zh=0.0))
    with A.AmpPcg(rp, ci, va, A.PRECOND_NONE) as h:
        x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
        st = h.solve(b, x, tol, 150, A.Policy.default(no_stop=1, tau_zs=0.0, tau_zh=0.0, true_residual=1, x0_zero=1))
        hist = h.residual_history()
        eh = h.eta_posteriori()
    # 150 iterations, or fewer when the recursive residual underflows to 0 first (Example 4: rho = 0 ends both runs)
    assert abs(st.iters - ref.iters) <= 2 and st.status == ref.status
    assert len(hist) == st.iters + 1 and len(eh) == st.iters + 1
    assert abs(st.it_ur32 - ref.it_ur32) <= 2 and st.it_uz32 < 0
    want = np.array([O.eta_posteriori(hist, k) for k in range(len(hist))])
    assert np.allclose(eh, want, rtol=1e-12, atol=0.0)
    bound = eh[st.it_ur32] / st.bnorm
    assert st.relres_true <= bound <= 10.0 * st.relres_true and bound <= tol
    # same stagnation level as the oracle's run (rounding-level differences move it by small factors only)
    assert 0.2 * ref.relres_true <= st.relres_true <= 5.0 * ref.relres_true


def test_indicator_on_a_full_size_like_solve():
    s = make_config("c3", 30)
    rp, ci, va, b = _dev(s)
    with A.AmpPcg(rp, ci, va) as h:
        x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
        st = h.solve(b, x, s.tol, s.maxit, A.Policy.default(true_residual=1, x0_zero=1))
        hist, eh = h.residual_history(), h.eta_posteriori()
        assert st.status == 0 and st.it_ur32 > 0
        want = np.array([O.eta_posteriori(hist, k) for k in range(len(hist))])
        assert np.allclose(eh, want, rtol=1e-12, atol=0.0)
        assert np.all(np.diff(eh) < 0)
        # (3.11)/(4.7): true residual <~ ||zeta|| + ||r_m|| with ||zeta|| estimated by eta_hat at the switch
        assert st.relres_true * st.bnorm <= eh[st.it_ur32] + hist[-1]
        # C and eps32 are parameters: doubling eps32 doubles the FP32 part
        eh2 = h.eta_posteriori(1.0, 2.0 ** -23)
        assert np.all(eh2 > eh) and eh2[0] == pytest.approx(2.0 * eh[0], rel=1e-6)
