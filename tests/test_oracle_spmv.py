"""Pin P1 — the oracle's CSR SpMV (q = A p) against facts that do not
come from the oracle: dense long-double mat-vec on tiny matrices, the closed-form eigenpairs
of the FD / trilinear-FE Laplacians, and the row-sum pattern of the stencils.
"""
import numpy as np
import pytest

import oracle as O
from workloads import make_config, poisson2d_5pt, poisson3d_7pt, fe27_laplacian


def _dense(rowptr, colidx, vals, n):
    A = np.zeros((n, n), dtype=np.longdouble)
    for i in range(n):
        for e in range(rowptr[i], rowptr[i + 1]):
            A[i, colidx[e]] += np.longdouble(vals[e])
    return A


@pytest.mark.parametrize("name,size", [("c1", 9), ("c2", 6), ("c3", 6), ("c4", 5), ("c5", 300)])
def test_spmv_fp64_vs_dense_longdouble(name, size):
    s = make_config(name, size)
    assert s.n <= 512
    rng = np.random.default_rng(3)
    p = rng.standard_normal(s.n)
    q = O.spmv_fp64(s.rowptr, s.colidx, s.vals, p)
    A = _dense(s.rowptr, s.colidx, s.vals, s.n)
    ref = A @ p.astype(np.longdouble)
    absAp = np.abs(A) @ np.abs(p).astype(np.longdouble)
    m = int(np.diff(s.rowptr).max())
    assert np.all(np.abs(q - ref) <= m * 2.0 ** -53 * absAp + 1e-300)


def test_spmv_unsymmetric_pattern_catches_transpose():
    # a non-symmetric matrix: A p and A^T p differ, so a transposed-operand bug cannot hide
    rowptr = np.array([0, 2, 3, 6], dtype=np.int32)
    colidx = np.array([0, 2, 1, 0, 1, 2], dtype=np.int32)
    vals = np.array([1.0, 2.0, 3.0, 4.0, 5.0, 6.0])
    p = np.array([1.0, 10.0, 100.0])
    assert np.array_equal(O.spmv_fp64(rowptr, colidx, vals, p), np.array([201.0, 30.0, 654.0]))
    assert np.array_equal(O.spmv_fp32(rowptr, colidx, vals, p), np.array([201.0, 30.0, 654.0]))


def test_laplacian_2d_closed_form_eigenpairs():
    # A v = lam v with v = sin(i pi x/(N+1)) sin(j pi y/(N+1)), lam = sum_d (2 - 2 cos(i_d pi/(N+1)))
    N = 17
    rowptr, colidx, vals = poisson2d_5pt(N)
    g = np.arange(1, N + 1) * np.pi / (N + 1)
    for (i, j) in [(1, 1), (3, 5), (N, N), (N, 1)]:
        v = np.outer(np.sin(j * g), np.sin(i * g)).ravel()  # x fastest
        lam = (2 - 2 * np.cos(i * np.pi / (N + 1))) + (2 - 2 * np.cos(j * np.pi / (N + 1)))
        q = O.spmv_fp64(rowptr, colidx, vals, v)
        assert np.max(np.abs(q - lam * v)) <= 1e-14 * 8


def test_laplacian_3d_closed_form_eigenpairs():
    N = 9
    rowptr, colidx, vals = poisson3d_7pt(N)
    g = np.arange(1, N + 1) * np.pi / (N + 1)
    for (i, j, k) in [(1, 1, 1), (2, 7, 4), (N, N, N)]:
        v = np.einsum("k,j,i->kji", np.sin(k * g), np.sin(j * g), np.sin(i * g)).ravel()
        lam = sum(2 - 2 * np.cos(t * np.pi / (N + 1)) for t in (i, j, k))
        q = O.spmv_fp64(rowptr, colidx, vals, v)
        assert np.max(np.abs(q - lam * v)) <= 1e-13


def test_fe27_closed_form_eigenpairs_and_kappa():
    # trilinear FE: lam = k_i m_j m_k + m_i k_j m_k + m_i m_j k_k, k(t)=2-2cos t, m(t)=(2+cos t)/3
    N = 8
    rowptr, colidx, vals = fe27_laplacian(N)
    assert rowptr[-1] == (3 * N - 2) ** 3  # all 27 pattern entries are stored, zero faces included
    g = np.arange(1, N + 1) * np.pi / (N + 1)
    kf = lambda t: 2 - 2 * np.cos(t)
    mf = lambda t: (2 + np.cos(t)) / 3
    for (i, j, k) in [(1, 1, 1), (3, 2, 8), (N, N, N)]:
        ti, tj, tk = (t * np.pi / (N + 1) for t in (i, j, k))
        v = np.einsum("k,j,i->kji", np.sin(k * g), np.sin(j * g), np.sin(i * g)).ravel()
        lam = kf(ti) * mf(tj) * mf(tk) + mf(ti) * kf(tj) * mf(tk) + mf(ti) * mf(tj) * kf(tk)
        q = O.spmv_fp64(rowptr, colidx, vals, v)
        assert np.max(np.abs(q - lam * v)) <= 1e-13


def test_stencil_row_sums():
    # A*1: interior rows of the Laplacians sum to zero, boundary rows to the number of cut neighbours
    N = 12
    rowptr, colidx, vals = poisson3d_7pt(N)
    q = O.spmv_fp64(rowptr, colidx, vals, np.ones(N ** 3)).reshape(N, N, N)
    assert np.all(q[1:-1, 1:-1, 1:-1] == 0.0)
    assert q[0, 0, 0] == 3.0 and q[0, 5, 5] == 1.0 and q[0, 0, 5] == 2.0
    s = make_config("c3", 8)  # variable coefficient: interior rows still sum to zero (to rounding)
    q = O.spmv_fp64(s.rowptr, s.colidx, s.vals, np.ones(s.n)).reshape(8, 8, 8)
    d = s.scipy().diagonal().reshape(8, 8, 8)
    assert np.all(np.abs(q[1:-1, 1:-1, 1:-1]) <= 1e-14 * d[1:-1, 1:-1, 1:-1])
    assert np.all(q[0] > 0)  # Dirichlet boundary faces add a_c to the diagonal


def test_spmv_fp32_error_bound_and_exact_cases():
    s = make_config("c5", 400)
    rng = np.random.default_rng(5)
    p = rng.standard_normal(s.n)
    p16 = O.round_fp16(p)  # a vector stored in FP16 is converted exactly to float
    A = _dense(s.rowptr, s.colidx, s.vals.astype(np.float32).astype(np.float64), s.n)
    m = int(np.diff(s.rowptr).max())
    for acc64 in (0, 1):
        q = O.spmv_fp32(s.rowptr, s.colidx, s.vals, p16, accumulate64=acc64)
        assert np.array_equal(q, q.astype(np.float32).astype(np.float64))  # q is stored in FP32
        ref = A @ p16.astype(np.longdouble)
        absAp = np.abs(A) @ np.abs(p16).astype(np.longdouble)
        bound = (m if acc64 == 0 else 1.001) * 2.0 ** -24 * absAp
        assert np.all(np.abs(q - ref) <= bound)
    # small integers: every product and partial sum is exact in FP32
    rowptr, colidx, vals = poisson3d_7pt(5)
    pi = rng.integers(-50, 50, 125).astype(np.float64)
    assert np.array_equal(O.spmv_fp32(rowptr, colidx, vals, pi), O.spmv_fp64(rowptr, colidx, vals, pi))


def test_dot_matches_longdouble():
    rng = np.random.default_rng(7)
    a, b = rng.standard_normal(100001), rng.standard_normal(100001)
    ref = float(np.sum(a.astype(np.longdouble) * b.astype(np.longdouble)))
    assert abs(O.dot(a, b) - ref) <= 1e-13 * float(np.sum(np.abs(a * b)))
