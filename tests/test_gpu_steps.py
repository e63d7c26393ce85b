"""-m gpu: every vector step of the loop, in EVERY precision instance that can occur, element by element and bit for
bit against the oracle's step functions (Algorithm 4.1 lines 4-5, 10, 15-16).

The library's diagnostic entry point amp_pcg_debug_step runs ONE step with caller-given scalars through the same
__global__ kernel, grid and grid reduction that the stream / graph loop launches (k_z, k_p, k_spmv, k_xr, k_xrz), on
the handle's own work vectors.  Covered: phase_z 9 instances (3 of them the fused r <- RN32(r) transition a6),
phase_p 6 (3 transitions p <- RN_{u_z}(p)), phase_xr 6, phase_xrz 18, in-loop SpMV 6; on odd n not a multiple of 8
(ragged chunk tail, x exactly n long), several blocks and trips, with values that land on FP16 subnormals, +-65504,
overflow to inf and exact zeros.

Bit-exactness holds because both sides do the same FP64 operations on the same stored values and round ONCE
(DESIGN.md section 4); the reductions are FP64 sums in different fixed orders: relative n 2^-53 of sum |a_i b_i|.
"""
import numpy as np
import pytest

import oracle as O
from workloads import make_config

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
A = pytest.importorskip("paper_2505_04155_b200")

NP = {0: np.float64, 1: np.float32, 2: np.float16}
RND = {0: lambda a: np.asarray(a, dtype=np.float64), 1: O.round_fp32, 2: O.round_fp16}


def dev(a, prec):
    return torch.from_numpy(np.ascontiguousarray(a.astype(NP[prec]))).cuda()


def host(t):
    return t.cpu().numpy().astype(np.float64)


def special(rng, n, scale=1.0):
    """standard normals * scale with hand-made entries: zeros, FP16 subnormal range, the largest FP16, overflow"""
    v = rng.standard_normal(n) * scale
    k = min(n, 12)
    v[:k] = np.array([0.0, -0.0, 2.0 ** -15, -2.0 ** -20, 2.0 ** -24, 3.0e-8, 2.0 ** -25, 65504.0, -65504.0, 65519.9, 65520.0,
                      1.0e5])[:k]
    return v


# every case with the direct vector kernels and with the bulk-copy staged ones (vec_pipe.cuh): same chunk bodies, same bits
@pytest.fixture(scope="module", params=[("c3", 11, "direct"), ("c2", 47, "direct"), ("c3", 107, "direct"),
                                        ("c3", 11, "staged"), ("c2", 47, "staged"), ("c3", 107, "staged")],
                ids=lambda p: f"{p[0]}@{p[1]}-{p[2]}")
def handle(request):
    name, size, vec = request.param
    s = make_config(name, size)
    assert s.n % 2 == 1 and s.n % 8 != 0
    h = A.AmpPcg(*(torch.from_numpy(a).cuda() for a in (s.rowptr, s.colidx, s.vals)), A.PRECOND_JACOBI,
                 vec_kernel={"direct": A.VEC_DIRECT, "staged": A.VEC_STAGED}[vec])
    rows = np.repeat(np.arange(s.n), np.diff(s.rowptr))
    diag = s.vals[s.colidx == rows]
    assert len(diag) == s.n
    dinv = {0: 1.0 / diag, 1: O.round_fp32(1.0 / diag)}
    # the library's own 1/diag copies are what the oracle-side formula says (reading R6)
    assert np.array_equal(host(h.debug_get_vector(A.VEC_DINV, A.FP64)), dinv[0])
    assert np.array_equal(host(h.debug_get_vector(A.VEC_DINV, A.FP32)), dinv[1])
    yield s, h, dinv
    h.close()


def assert_bits(got, want, what):
    got = np.asarray(got, dtype=np.float64)
    same = (got == want) | (np.isnan(got) & np.isnan(want))
    # signed zeros must agree too
    same &= np.signbit(got) == np.signbit(want)
    assert same.all(), (what, int((~same).sum()), np.flatnonzero(~same)[:5], got[~same][:5], want[~same][:5])


def sum_close(got, a, b):
    ref = O.dot(a, b)
    if not np.isfinite(ref):  # an overflowed product: the GPU sum must not come out finite either
        return not np.isfinite(got)
    bound = len(a) * 2.0 ** -53 * float(np.abs(a * b).sum()) + 1e-300
    return abs(got - ref) <= bound


Z_INST = [(rs, ur, uz) for rs, ur in ((0, 0), (0, 1), (1, 1)) for uz in (0, 1, 2)]


@pytest.mark.parametrize("rs,ur,uz", Z_INST)
def test_step_z_bitwise(handle, rs, ur, uz):
    s, h, dinv = handle
    rng = np.random.default_rng(100 + 9 * rs + 3 * ur + uz)
    for omega, scale in ((1.0 / 37.5, 1.0), (2.0 ** -3, 1e-3), (1.0, 4e3)):
        r = RND[rs](special(rng, s.n, scale))
        h.debug_set_vector(A.VEC_R, dev(r, rs))
        io = h.debug_step(A.STEP_Z, rs=rs, ur=ur, uz=uz, ps=uz, ur_n=ur, uz_n=uz, omega=omega)
        r_used = RND[ur](r)  # a6: r <- RN32(r) at the u_r switch, fused into this pass
        z_ref, _ = O.step_z(r_used, omega, dinv[0 if uz == 0 else 1], ur, uz)
        assert_bits(host(h.debug_get_vector(A.VEC_Z, uz)), z_ref, "z")
        assert_bits(host(h.debug_get_vector(A.VEC_R, ur)), r_used, "r after the step")
        fin = np.isfinite(z_ref)
        if fin.all():
            assert sum_close(io.sum0, r_used, z_ref), (io.sum0, O.dot(r_used, z_ref))
        else:
            assert not np.isfinite(io.sum0) or np.isnan(io.sum0)


P_INST = [(0, 0), (0, 1), (1, 1), (0, 2), (1, 2), (2, 2)]


@pytest.mark.parametrize("ps,uz", P_INST)
@pytest.mark.parametrize("first", [0, 1])
def test_step_p_bitwise(handle, ps, uz, first):
    s, h, _ = handle
    rng = np.random.default_rng(200 + 3 * ps + uz)
    for beta, scale in ((0.937, 1.0), (1.0 / 3.0, 2e-5), (17.25, 3e3)):
        if first:
            beta = 0.0
        z = RND[uz](special(rng, s.n, scale))
        z[~np.isfinite(z)] = 0.0
        p = RND[ps](special(rng, s.n, scale)[::-1].copy())
        p[~np.isfinite(p)] = 1.0
        h.debug_set_vector(A.VEC_Z, dev(z, uz))
        h.debug_set_vector(A.VEC_P, dev(p, ps))
        h.debug_step(A.STEP_P, rs=0, ur=0, uz=uz, ps=ps, ur_n=0, uz_n=uz, beta=beta, first=first)
        p_in = np.zeros(s.n) if first else RND[uz](p)  # a6 / R9: p_{k-1} <- RN_{u_z}(p_{k-1}) at a u_z switch
        p_ref, _ = O.step_p(beta, p_in, z, uz)
        assert_bits(host(h.debug_get_vector(A.VEC_P, uz)), p_ref, "p")


def test_step_p_writes_the_fp32_copy_in_phase_fp64_fp32(handle):
    # while u_z = FP64 and u_r = FP32 the mat-vec gathers RN32(p_j) (reading R7): the p update stores that copy
    s, h, _ = handle
    rng = np.random.default_rng(77)
    z = special(rng, s.n); z[~np.isfinite(z)] = 0.0
    p = rng.standard_normal(s.n)
    h.debug_set_vector(A.VEC_Z, dev(z, 0))
    h.debug_set_vector(A.VEC_P, dev(p, 0))
    h.debug_step(A.STEP_P, rs=1, ur=1, uz=0, ps=0, ur_n=1, uz_n=0, beta=0.61)
    p_ref, _ = O.step_p(0.61, p, z, 0)
    assert_bits(host(h.debug_get_vector(A.VEC_P, 0)), p_ref, "p")
    assert_bits(host(h.debug_get_vector(A.VEC_P, 1)), O.round_fp32(p_ref), "RN32(p)")


XR_INST = [(ur, uz) for ur in (0, 1) for uz in (0, 1, 2)]


@pytest.mark.parametrize("ur,uz", XR_INST)
def test_step_xr_bitwise(handle, ur, uz):
    s, h, _ = handle
    rng = np.random.default_rng(300 + 3 * ur + uz)
    for alpha, scale in ((0.731, 1.0), (-2.5e-3, 1e3), (1.0e-7, 1e-2)):
        p = RND[uz](special(rng, s.n, scale)); p[~np.isfinite(p)] = 0.5
        q = RND[ur](rng.standard_normal(s.n) * scale)
        r = RND[ur](special(rng, s.n, scale))
        x = rng.standard_normal(s.n)
        h.debug_set_vector(A.VEC_P, dev(p, uz))
        h.debug_set_vector(A.VEC_Q, dev(q, ur))
        h.debug_set_vector(A.VEC_R, dev(r, ur))
        xd = torch.from_numpy(x).cuda()
        io = h.debug_step(A.STEP_XR, x=xd, rs=ur, ur=ur, uz=uz, ps=uz, ur_n=ur, uz_n=uz, alpha=alpha)
        x_ref, r_ref = O.step_xr(alpha, p, q, x, r, ur)
        assert_bits(host(xd), x_ref, "x")
        assert_bits(host(h.debug_get_vector(A.VEC_R, ur)), r_ref, "r")
        want = np.sqrt(O.dot(r_ref, r_ref))
        assert io.sum0 == pytest.approx(want, rel=s.n * 2.0 ** -53)


XRZ_INST = [(ur, urn, uz, uzn) for ur, urn in ((0, 0), (0, 1), (1, 1)) for uz, uzn in P_INST]


@pytest.mark.parametrize("ur,urn,uz,uzn", XRZ_INST)
def test_step_xrz_bitwise(handle, ur, urn, uz, uzn):
    s, h, dinv = handle
    rng = np.random.default_rng(400 + 27 * ur + 9 * urn + 3 * uz + uzn)
    for alpha, omega_n, scale in ((0.731, 1.0 / 12.5, 1.0), (-1.0e-3, 2.0 ** 4, 1e-4)):
        p = RND[uz](special(rng, s.n, scale)); p[~np.isfinite(p)] = 0.5
        q = RND[ur](rng.standard_normal(s.n) * scale)
        r = RND[ur](special(rng, s.n, scale)); r[~np.isfinite(r)] = 1.0
        x = rng.standard_normal(s.n)
        h.debug_set_vector(A.VEC_P, dev(p, uz))
        h.debug_set_vector(A.VEC_Q, dev(q, ur))
        h.debug_set_vector(A.VEC_R, dev(r, ur))
        xd = torch.from_numpy(x).cuda()
        io = h.debug_step(A.STEP_XRZ, x=xd, rs=ur, ur=ur, uz=uz, ps=uz, ur_n=urn, uz_n=uzn, alpha=alpha, omega_n=omega_n)
        x_ref, r_ref = O.step_xr(alpha, p, q, x, r, urn)  # r_{k+1} is stored directly in u_r of iteration k+1 (R17)
        z_ref, _ = O.step_z(r_ref, omega_n, dinv[0 if uzn == 0 else 1], urn, uzn)
        assert_bits(host(xd), x_ref, "x")
        assert_bits(host(h.debug_get_vector(A.VEC_R, urn)), r_ref, "r")
        assert_bits(host(h.debug_get_vector(A.VEC_Z, uzn)), z_ref, "z")
        assert io.sum0 == pytest.approx(np.sqrt(O.dot(r_ref, r_ref)), rel=s.n * 2.0 ** -53)
        if np.isfinite(z_ref).all():
            assert sum_close(io.sum1, r_ref, z_ref)


@pytest.fixture(scope="module", params=[("c3", 32), ("c4", 32), ("c2", 64), ("c1", 320)], ids=lambda p: f"{p[0]}@{p[1]}")
def spmv_handles(request):
    """the same matrix behind both in-loop SpMV kernels: the direct one and the bulk-copy pipelined one"""
    name, size = request.param
    s = make_config(name, size)
    devm = [torch.from_numpy(a).cuda() for a in (s.rowptr, s.colidx, s.vals)]
    hs = [A.AmpPcg(*devm, A.PRECOND_JACOBI, spmv_kernel=k) for k in (A.SPMV_DIRECT, A.SPMV_PIPELINED)]
    yield s, hs
    for h in hs:
        h.close()


@pytest.mark.parametrize("ur,uz", XR_INST)
def test_step_spmv_in_loop_kernel_bitwise(spmv_handles, ur, uz):
    # the in-loop SpMV kernels (not the stand-alone amp_spmv kernel): q bit-identical, gamma to reduction accuracy
    s, hs = spmv_handles
    rng = np.random.default_rng(500 + 3 * ur + uz)
    p = RND[uz](rng.standard_normal(s.n))
    q_ref = O.spmv_fp64(s.rowptr, s.colidx, s.vals, p) if ur == 0 else O.spmv_fp32(s.rowptr, s.colidx, s.vals, p)
    for h in hs:
        h.debug_set_vector(A.VEC_P, dev(p, uz))
        h.debug_set_vector(A.VEC_Q, dev(np.full(s.n, 7.0), ur))
        io = h.debug_step(A.STEP_SPMV, rs=ur, ur=ur, uz=uz, ps=uz, ur_n=ur, uz_n=uz)
        assert_bits(host(h.debug_get_vector(A.VEC_Q, ur)), q_ref, "q")
        assert sum_close(io.sum0, q_ref, p)


def test_debug_step_rejects_impossible_combinations(handle):
    s, h, _ = handle
    with pytest.raises(A.AmpPcgError):
        h.debug_step(A.STEP_Z, rs=1, ur=0, uz=0)          # precision never goes back up
    with pytest.raises(A.AmpPcgError):
        h.debug_step(A.STEP_XR, x=None, rs=0, ur=0, uz=0)  # x missing
    with pytest.raises(A.AmpPcgError):
        h.debug_set_vector(A.VEC_R, torch.zeros(s.n, dtype=torch.float16, device="cuda"))  # r is never FP16
