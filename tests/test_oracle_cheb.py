"""Pins of the oracle's Chebyshev-accelerated Jacobi preconditioner (the paper's smoother; its use as the
loop's M^-1 is reading R18 of DESIGN.md).  The vector recurrence is checked against what it must equal by the theory of
Chebyshev iteration: z_s = (I - q_s(D^-1 A)) A^-1 y with q_s(l) = T_s((theta - l)/dc) / T_s(theta/dc), evaluated densely
through an eigendecomposition and the CLOSED FORM of T_s (cos / cosh) — no three-term recurrence on that side."""
import math

import numpy as np
import pytest

import oracle as O
from workloads import make_config


def dense(s):
    import scipy.sparse as sp

    return sp.csr_matrix((s.vals, s.colidx, s.rowptr), shape=(s.n, s.n)).toarray()


def cheb_T(k, x):
    x = np.asarray(x, dtype=np.float64)
    out = np.empty_like(x)
    m = np.abs(x) <= 1.0
    out[m] = np.cos(k * np.arccos(x[m]))
    xp = x[~m]
    out[~m] = np.sign(xp) ** k * np.cosh(k * np.arccosh(np.abs(xp)))
    return out


def dense_chebyshev(Ad, y, s, lmin, lmax):
    dg = np.diag(Ad)
    S = Ad / np.sqrt(np.outer(dg, dg))           # D^-1/2 A D^-1/2: symmetric, same spectrum as D^-1 A
    lam, V = np.linalg.eigh(S)
    theta, dc = (lmax + lmin) / 2, (lmax - lmin) / 2
    q = cheb_T(s, (theta - lam) / dc) / cheb_T(s, np.array([theta / dc]))[0]
    g = (1.0 - q) / lam                          # z = D^-1/2 V g(Lambda) V^T D^-1/2 y
    return (V @ (g * (V.T @ (y / np.sqrt(dg))))) / np.sqrt(dg)


@pytest.mark.parametrize("name,size", [("c1", 12), ("c3", 6), ("c4", 6), ("c5", 300)])
@pytest.mark.parametrize("deg", [1, 2, 3, 5])
def test_recurrence_equals_the_dense_chebyshev_polynomial(name, size, deg):
    s = make_config(name, size)
    assert s.n <= 512
    Ad = dense(s)
    rng = np.random.default_rng(5)
    y = rng.standard_normal(s.n)
    lmin, lmax = O.cheb_default_bounds(s.rowptr, s.colidx, s.vals)
    lam = np.linalg.eigvalsh(Ad / np.sqrt(np.outer(np.diag(Ad), np.diag(Ad))))
    assert lam.max() <= lmax * (1 + 1e-12)       # Gershgorin: a true upper bound of the spectrum of D^-1 A
    assert lmin == lmax / 30.0
    z = O.cheb_apply(s.rowptr, s.colidx, s.vals, y, 1.0, 1.0 / np.diag(Ad), deg, lmin, lmax)
    zd = dense_chebyshev(Ad, y, deg, lmin, lmax)
    assert np.linalg.norm(z - zd) <= 1e-11 * np.linalg.norm(zd)
    # omega scales linearly (the scaled residual y = omega r is what is preconditioned)
    z2 = O.cheb_apply(s.rowptr, s.colidx, s.vals, y, 0.25, 1.0 / np.diag(Ad), deg, lmin, lmax)
    assert np.allclose(z2, 0.25 * z, rtol=1e-13, atol=0)


def test_coefficients_closed_form():
    # rho_i = T_i(sigma) / T_{i+1}(sigma): the classical identity behind the three-term recurrence
    lmin, lmax = 0.07, 2.3
    it, c1, c2 = O.cheb_coeffs(6, lmin, lmax)
    theta, dc = (lmax + lmin) / 2, (lmax - lmin) / 2
    sig = theta / dc
    rho = [float(cheb_T(i, np.array([sig]))[0] / cheb_T(i + 1, np.array([sig]))[0]) for i in range(6)]
    assert it == pytest.approx(1 / theta, rel=1e-15)
    for i in range(1, 6):
        assert c1[i] == pytest.approx(rho[i] * rho[i - 1], rel=1e-12)
        assert c2[i] == pytest.approx(2 * rho[i] / dc, rel=1e-12)


def test_degree_one_is_scaled_jacobi_and_the_operator_is_spd():
    s = make_config("c3", 7)
    Ad = dense(s)
    dinv = 1.0 / np.diag(Ad)
    lmin, lmax = O.cheb_default_bounds(s.rowptr, s.colidx, s.vals)
    rng = np.random.default_rng(2)
    y = rng.standard_normal(s.n)
    z1 = O.cheb_apply(s.rowptr, s.colidx, s.vals, y, 1.0, dinv, 1, lmin, lmax)
    assert np.array_equal(z1, (y * dinv) * (1.0 / ((lmax + lmin) / 2)))
    # PCG iterates do not change when M is scaled by a constant: degree 1 = Jacobi (iteration count, to rounding)
    a = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(amp=0))
    b = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(amp=0, precond=O.PRECOND_CHEBJACOBI, cheb_degree=1))
    assert b.status == 0 and abs(a.iters - b.iters) <= 1
    assert np.allclose(a.hist[:20], b.hist[:20], rtol=1e-9)
    # M^-1 is symmetric positive definite for every degree (what PCG needs): u^T M^-1 v = v^T M^-1 u, u^T M^-1 u > 0
    u, v = rng.standard_normal(s.n), rng.standard_normal(s.n)
    for deg in (2, 3, 4):
        Pu = O.cheb_apply(s.rowptr, s.colidx, s.vals, u, 1.0, dinv, deg, lmin, lmax)
        Pv = O.cheb_apply(s.rowptr, s.colidx, s.vals, v, 1.0, dinv, deg, lmin, lmax)
        assert v @ Pu == pytest.approx(u @ Pv, rel=1e-12)
        assert u @ Pu > 0 and v @ Pv > 0


def test_stored_values_are_representable_and_steps_follow_the_stated_operation_order():
    s = make_config("c3", 8)
    rows = np.repeat(np.arange(s.n), np.diff(s.rowptr))
    dinv32 = O.round_fp32(1.0 / s.vals[s.colidx == rows])
    rng = np.random.default_rng(3)
    r = O.round_fp32(rng.standard_normal(s.n))
    omega = 1.0 / np.linalg.norm(r)
    it, c1, c2 = O.cheb_coeffs(3, 0.1, 2.0)
    d, z = O.cheb_first(r, omega, dinv32, it, O.FP16)
    assert np.array_equal(d, O.round_fp16(((r * omega) * dinv32) * it)) and np.array_equal(z, d)
    w = O.spmv_fp32(s.rowptr, s.colidx, s.vals, z)
    d2, z2 = O.cheb_step(r, omega, w, dinv32, c1[1], c2[1], O.FP16, d, z)
    # fma(c1, d, c2 u) with u = (r omega - w) dinv: exact rational check of the single rounding of the fma
    from fractions import Fraction

    for i in range(0, s.n, 37):
        u = float(Fraction(float(Fraction(r[i]) * Fraction(omega))) - Fraction(w[i])) * dinv32[i]
        c2u = c2[1] * u
        dn = float(Fraction(c1[1]) * Fraction(d[i]) + Fraction(c2u))
        assert d2[i] == O.round_fp16(dn)[0]
        assert z2[i] == O.round_fp16(z[i] + d2[i])[0]
    assert np.array_equal(d2, O.round_fp16(d2)) and np.array_equal(z2, O.round_fp16(z2))


@pytest.mark.parametrize("name,size", [("c1", 64), ("c2", 24)])
def test_iterations_drop_with_the_degree(name, size):
    # degree s costs s mat-vecs per iteration (s - 1 in M^-1 + one for q = A p) and cuts the iteration count by about
    # s: the total number of mat-vecs must not grow by more than a fifth, and the iterations must fall well below half
    s = make_config(name, size)
    base = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(amp=0))
    its = {1: base.iters}
    for deg in (2, 3, 4):
        r = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit,
                      O.make_policy(amp=0, precond=O.PRECOND_CHEBJACOBI, cheb_degree=deg))
        assert r.status == 0 and r.relres_true <= 2 * s.tol
        its[deg] = r.iters
    assert its[2] < 0.75 * its[1] and its[3] < 0.55 * its[1] and its[4] < 0.45 * its[1]
    for deg in (2, 3, 4):
        assert deg * its[deg] <= 1.35 * its[1]


@pytest.mark.parametrize("name,size", [("c1", 64), ("c3", 19), ("c4", 13)])
def test_amp_pcg_with_chebyshev_keeps_the_papers_guarantees(name, size):
    # AMP-PCG(FP64) and AMP-PCG(FP16) with the Chebyshev-Jacobi M^-1: same iteration count as FP64 PCG with the same
    # preconditioner (within 5 %), true residual <= 2 tol, all three switches still happen
    s = make_config(name, size)
    kw = dict(precond=O.PRECOND_CHEBJACOBI, cheb_degree=3)
    ref = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(amp=0, **kw))
    for pol in (dict(), dict(u0=O.FP16, eta_rule=O.ETA_LINEAR)):
        r = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(**pol, **kw))
        assert r.status == 0
        assert abs(r.iters - ref.iters) <= max(1, math.ceil(0.05 * ref.iters))
        assert r.relres_true <= 2 * s.tol
        assert r.it_ur32 >= 0
    # unsupported combinations are refused, not silently changed
    bad = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, 10, O.make_policy(scale_mode=O.SCALE_LAGGED, **kw))
    assert bad.status == -1
