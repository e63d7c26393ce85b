"""-m gpu: the Chebyshev-accelerated Jacobi preconditioner (AMP_PRECOND_CHEBJACOBI: the paper's smoother, PAPER.md:461,
as M^-1 of the loop; reading R18) against the oracle:

* the spectrum bound computed in create() equals the oracle's (same row sums in the same order);
* the two vector kernels (first sweep, further sweeps) bit for bit in every precision instance, and the mat-vec q = A z
  inside M^-1 bit for bit, through amp_pcg_debug_step (the kernels the loop launches);
* whole solves: iteration counts within 5 % (FP64 PCG +-1), switch iterations +-2, true residual <= 2 tol, and the
  iteration count falls with the degree as the oracle's does;
* the combinations the library does not offer are refused.
"""
import numpy as np
import pytest

import oracle as O
from workloads import make_config
from gpu_util import iters_close, switch_close, to_device

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")

NP = {0: np.float64, 1: np.float32, 2: np.float16}
RND = {0: lambda a: np.asarray(a, dtype=np.float64), 1: O.round_fp32, 2: O.round_fp16}


def dev(a, prec):
    return torch.from_numpy(np.ascontiguousarray(a.astype(NP[prec]))).cuda()


def host(t):
    return t.cpu().numpy().astype(np.float64)


def assert_bits(got, want, what):
    same = ((got == want) | (np.isnan(got) & np.isnan(want))) & (np.signbit(got) == np.signbit(want))
    assert same.all(), (what, int((~same).sum()), np.flatnonzero(~same)[:5], got[~same][:5], want[~same][:5])


DEG = 4


@pytest.fixture(scope="module", params=[("c3", 11, A.SPMV_AUTO), ("c4", 32, A.SPMV_PIPELINED), ("c2", 47, A.SPMV_DIRECT)],
                ids=lambda p: f"{p[0]}@{p[1]}")
def handle(request):
    name, size, kern = request.param
    s = make_config(name, size)
    h = A.AmpPcg(*(torch.from_numpy(a).cuda() for a in (s.rowptr, s.colidx, s.vals)), A.PRECOND_CHEBJACOBI,
                 cheb_degree=DEG, spmv_kernel=kern)
    rows = np.repeat(np.arange(s.n), np.diff(s.rowptr))
    diag = s.vals[s.colidx == rows]
    dinv = {0: 1.0 / diag, 1: O.round_fp32(1.0 / diag)}
    lmin, lmax = O.cheb_default_bounds(s.rowptr, s.colidx, s.vals)
    yield s, h, dinv, O.cheb_coeffs(DEG, lmin, lmax)
    h.close()


@pytest.mark.parametrize("rs,ur,uz", [(rs, ur, uz) for rs, ur in ((0, 0), (0, 1), (1, 1)) for uz in (0, 1, 2)])
def test_first_sweep_bitwise(handle, rs, ur, uz):
    s, h, dinv, (inv_theta, c1, c2) = handle
    rng = np.random.default_rng(10 + 9 * rs + 3 * ur + uz)
    r = RND[rs](rng.standard_normal(s.n))
    r[:6] = RND[rs](np.array([0.0, 2.0 ** -20, -3e-8, 65504.0, 1e5, -1.0]))
    omega = 1.0 / 17.3
    h.debug_set_vector(A.VEC_R, dev(r, rs))
    h.debug_step(A.STEP_CHEB0, rs=rs, ur=ur, uz=uz, ps=uz, ur_n=ur, uz_n=uz, omega=omega)
    r_used = RND[ur](r)
    d_ref, z_ref = O.cheb_first(r_used, omega, dinv[0 if uz == 0 else 1], inv_theta, uz)
    assert_bits(host(h.debug_get_vector(A.VEC_Z, uz)), z_ref, "z")
    assert_bits(host(h.debug_get_vector(A.VEC_D, uz)), d_ref, "d")
    assert_bits(host(h.debug_get_vector(A.VEC_R, ur)), r_used, "r")


@pytest.mark.parametrize("ur,uz", [(ur, uz) for ur in (0, 1) for uz in (0, 1, 2)])
@pytest.mark.parametrize("sweep", [1, DEG - 1])
def test_further_sweeps_and_inner_matvec_bitwise(handle, ur, uz, sweep):
    s, h, dinv, (inv_theta, c1, c2) = handle
    rng = np.random.default_rng(20 + 3 * ur + uz + sweep)
    r = RND[ur](rng.standard_normal(s.n))
    z = RND[uz](rng.standard_normal(s.n) * 0.05)
    d = RND[uz](rng.standard_normal(s.n) * 0.05)
    z[:4] = RND[uz](np.array([0.0, 2.0 ** -21, -2.0 ** -15, 1.0]))
    omega = 1.0 / 9.7
    h.debug_set_vector(A.VEC_R, dev(r, ur))
    h.debug_set_vector(A.VEC_Z, dev(z, uz))
    h.debug_set_vector(A.VEC_D, dev(d, uz))
    # the mat-vec inside M^-1: w = A z in u_r, written to the q buffers
    h.debug_step(A.STEP_SPMV_Z, rs=ur, ur=ur, uz=uz, ps=uz, ur_n=ur, uz_n=uz)
    w_ref = O.spmv_fp64(s.rowptr, s.colidx, s.vals, z) if ur == 0 else O.spmv_fp32(s.rowptr, s.colidx, s.vals, z)
    assert_bits(host(h.debug_get_vector(A.VEC_Q, ur)), w_ref, "w = A z")
    io = h.debug_step(A.STEP_CHEBSTEP, rs=ur, ur=ur, uz=uz, ps=uz, ur_n=ur, uz_n=uz, omega=omega, first=sweep)
    d_ref, z_ref = O.cheb_step(r, omega, w_ref, dinv[0 if uz == 0 else 1], c1[sweep], c2[sweep], uz, d, z)
    assert_bits(host(h.debug_get_vector(A.VEC_D, uz)), d_ref, "d")
    assert_bits(host(h.debug_get_vector(A.VEC_Z, uz)), z_ref, "z")
    if sweep == DEG - 1:  # the last sweep also forms rho = r^T z
        ref = O.dot(r, z_ref)
        assert abs(io.sum0 - ref) <= s.n * 2.0 ** -53 * float(np.abs(r * z_ref).sum()) + 1e-300


def test_default_spectrum_bound_matches_the_oracle():
    s = make_config("c3", 21)
    lmin, lmax = O.cheb_default_bounds(s.rowptr, s.colidx, s.vals)
    rp, ci, va, b = to_device(s)
    # give the oracle's bounds explicitly and let create() compute them: identical solves, bit for bit
    res = []
    for kw in (dict(), dict(cheb_lmin=lmin, cheb_lmax=lmax)):
        with A.AmpPcg(rp, ci, va, A.PRECOND_CHEBJACOBI, cheb_degree=3, **kw) as h:
            x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
            st = h.solve(b, x, s.tol, s.maxit, A.Policy.default(x0_zero=1))
            res.append((st.iters, x.cpu().numpy()))
    assert res[0][0] == res[1][0] and np.array_equal(res[0][1], res[1][1])


SMALL = [("c1", 64), ("c2", 33), ("c3", 31), ("c4", 32), ("c5", 30011)]
POL = {"pcg_fp64": dict(amp=0), "amp_fp64_delay": dict(amp=1, u0=0, eta_rule=0), "amp_fp16_linear": dict(amp=1, u0=2, eta_rule=1),
       "amp_fp64_delay_strict": dict(amp=1, u0=0, eta_rule=0, eta_safety=0.1, stop_safety=0.9)}


@pytest.mark.parametrize("loop", [A.LOOP_STREAM, A.LOOP_GRAPH])
@pytest.mark.parametrize("pname", sorted(POL))
@pytest.mark.parametrize("name,size", SMALL)
def test_solve_parity_with_chebyshev(name, size, pname, loop):
    s = make_config(name, size)
    rp, ci, va, b = to_device(s)
    for deg in (2, 3):
        ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit,
                        O.make_policy(precond=O.PRECOND_CHEBJACOBI, cheb_degree=deg, **POL[pname]))
        with A.AmpPcg(rp, ci, va, A.PRECOND_CHEBJACOBI, cheb_degree=deg) as h:
            x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
            st = h.solve(b, x, s.tol, s.maxit, A.Policy.default(x0_zero=1, true_residual=1, loop_mode=loop, **POL[pname]))
            assert st.status == ref.status == 0 and st.loop_mode == loop
            assert iters_close(st.iters, ref.iters), (deg, st.iters, ref.iters)
            if pname == "pcg_fp64":
                assert abs(st.iters - ref.iters) <= 1
            for a, r_ in ((st.it_ur32, ref.it_ur32), (st.it_uz32, ref.it_uz32), (st.it_uz16, ref.it_uz16)):
                assert switch_close(a, r_), (pname, a, r_)
            true = np.linalg.norm(s.b - O.spmv_fp64(s.rowptr, s.colidx, s.vals, x.cpu().numpy())) / np.linalg.norm(s.b)
            assert st.relres_true == pytest.approx(true, rel=1e-6, abs=1e-18)
            assert true <= (1.0 if "strict" in pname else 2.0) * s.tol
            hist = h.residual_history()
            k = min(len(hist), len(ref.hist), 10)
            assert np.allclose(hist[:k], ref.hist[:k], rtol=1e-4)


def test_iterations_fall_with_the_degree_and_auto_loop_is_the_graph():
    s = make_config("c2", 48)
    rp, ci, va, b = to_device(s)
    its = {}
    for deg in (1, 2, 4):
        with A.AmpPcg(rp, ci, va, A.PRECOND_CHEBJACOBI, cheb_degree=deg) as h:
            x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
            st = h.solve(b, x, s.tol, s.maxit, A.Policy.default(x0_zero=1))
            assert st.status == 0 and st.loop_mode == A.LOOP_GRAPH  # n < 2^20, but the persistent kernel has no Chebyshev path
            its[deg] = st.iters
            ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(precond=2, cheb_degree=deg))
            assert iters_close(st.iters, ref.iters)
    assert its[2] < 0.75 * its[1] and its[4] < 0.45 * its[1]


def test_unsupported_combinations_are_refused():
    s = make_config("c1", 64)
    rp, ci, va, b = to_device(s)
    with pytest.raises(A.AmpPcgError):
        A.AmpPcg(rp, ci, va, A.PRECOND_CHEBJACOBI, cheb_degree=0)
    with pytest.raises(A.AmpPcgError):
        A.AmpPcg(rp, ci, va, A.PRECOND_CHEBJACOBI, cheb_lmin=2.0, cheb_lmax=1.0)
    with A.AmpPcg(rp, ci, va, A.PRECOND_CHEBJACOBI) as h:
        x = torch.zeros(s.n, dtype=torch.float64, device="cuda")
        with pytest.raises(A.AmpPcgError):
            h.solve(b, x, s.tol, s.maxit, A.Policy.default(scale_mode=A.SCALE_LAGGED))
        with pytest.raises(A.AmpPcgError):
            h.solve(b, x, s.tol, s.maxit, A.Policy.default(loop_mode=A.LOOP_PERSISTENT))
    with A.AmpPcg(rp, ci, va, A.PRECOND_JACOBI) as h:
        with pytest.raises(A.AmpPcgError):
            h.debug_step(A.STEP_CHEB0, rs=0, ur=0, uz=0)
