"""Pins of the oracle's vector steps (orc_step_z / orc_step_p / orc_step_xr), of classify_fp16 and of the
strict_rounding diagnostic.  The steps are checked against EXACT rational arithmetic (fractions.Fraction):
the FP64 operations must be the correctly rounded exact results, and the stored value must be a nearest
representable number of the storage format (ties to even) — a formulation that shares nothing with the
oracle's own rounding routine (frexp/nearbyint)."""
from fractions import Fraction

import numpy as np
import pytest

import oracle as O
from workloads import make_config

NP_T = {O.FP64: np.float64, O.FP32: np.float32, O.FP16: np.float16}


def rn64(fr: Fraction) -> float:
    """correctly rounded (RN-even) double of an exact rational: CPython's Fraction -> float conversion"""
    return float(fr)


def assert_nearest_in_format(v64: float, stored: float, prec: int):
    """stored must be a nearest value of the format to v64, ties to even; overflow to inf by the IEEE rule"""
    T = NP_T[prec]
    s = T(stored)
    assert float(s) == stored, "stored value is not representable in its format"
    if prec == O.FP64:
        assert stored == v64
        return
    if np.isinf(s):
        fmax = float(np.finfo(T).max)
        half_ulp = (fmax - float(np.nextafter(T(fmax), T(0)))) / 2
        assert abs(v64) >= fmax + half_ulp  # RN-even: the midpoint rounds to the even neighbour = 2^(emax+1) = inf
        return
    err = abs(Fraction(v64) - Fraction(float(s)))
    for nb in (np.nextafter(s, T(np.inf)), np.nextafter(s, T(-np.inf))):
        if np.isinf(nb):
            continue
        enb = abs(Fraction(v64) - Fraction(float(nb)))
        assert err <= enb
        if err == enb:  # tie: the stored one has the even significand
            bits = s.view({np.float16: np.uint16, np.float32: np.uint32}[T])
            assert int(bits) % 2 == 0


def _cases(rng, n):
    r = rng.standard_normal(n)
    r[:8] = [0.0, 1.0, -1.0, 2.0 ** -20, 65504.0, 65520.0, 1e-8, -3.0e-5]
    return r


@pytest.mark.parametrize("uz", [O.FP64, O.FP32, O.FP16])
@pytest.mark.parametrize("ur", [O.FP64, O.FP32])
def test_step_z_against_exact_arithmetic(ur, uz):
    rng = np.random.default_rng(1)
    n = 300
    r = O.round_fp32(_cases(rng, n)) if ur == O.FP32 else _cases(rng, n)
    dinv = np.abs(rng.standard_normal(n)) * 10.0 ** rng.integers(-6, 3, n)
    if uz != O.FP64:
        dinv = O.round_fp32(dinv)  # reading R6: FP32 copy of 1/diag once u_z < FP64
    for omega in (1.0, 0.37, 2.0 ** -7, 1234.5):
        z, counts = O.step_z(r, omega, dinv, ur, uz)
        for i in range(n):
            t = rn64(Fraction(r[i]) * Fraction(omega))
            v = rn64(Fraction(t) * Fraction(dinv[i]))
            assert_nearest_in_format(v, z[i], uz)
        if uz == O.FP16:
            assert counts.sum() > 0  # the hand-made tiny / huge entries are classified


@pytest.mark.parametrize("uz", [O.FP64, O.FP32, O.FP16])
def test_step_p_is_one_fma_and_one_rounding(uz):
    rng = np.random.default_rng(2)
    n = 300
    rnd = {O.FP64: lambda a: a, O.FP32: O.round_fp32, O.FP16: O.round_fp16}[uz]
    z = rnd(_cases(rng, n) * 0.01)
    p = rnd(rng.standard_normal(n) * 0.01)
    for beta in (0.0, 0.93, 1.0 / 3.0, 17.25):
        pn, _ = O.step_p(beta, p, z, uz)
        for i in range(n):
            v = rn64(Fraction(beta) * Fraction(p[i]) + Fraction(z[i]))  # fma: ONE rounding of the exact value
            assert_nearest_in_format(v, pn[i], uz)
    # a product-then-add (two roundings in FP64) differs from the fma somewhere: the step must be the fma
    pn, _ = O.step_p(1.0 / 3.0, p, z, O.FP64)
    two = p * (1.0 / 3.0) + z
    assert np.any(pn != two)


@pytest.mark.parametrize("ur", [O.FP64, O.FP32])
def test_step_xr_against_exact_arithmetic(ur):
    rng = np.random.default_rng(3)
    n = 300
    rnd = {O.FP64: lambda a: a, O.FP32: O.round_fp32}[ur]
    p = O.round_fp16(rng.standard_normal(n) * 0.01)
    q = rnd(rng.standard_normal(n))
    r = rnd(_cases(rng, n))
    x = rng.standard_normal(n)
    for alpha in (0.0, 0.731, -2.5e-3):
        xn, rn = O.step_xr(alpha, p, q, x, r, ur)
        for i in range(n):
            assert xn[i] == rn64(Fraction(alpha) * Fraction(p[i]) + Fraction(x[i]))     # line 15, FP64 fma
            v = rn64(Fraction(-alpha) * Fraction(q[i]) + Fraction(r[i]))                # line 16, FP64 fma ...
            assert_nearest_in_format(v, rn[i], ur)                                      # ... then one rounding


def test_steps_compose_to_the_solver_iteration():
    # one traced iteration of orc_amp_pcg equals the steps applied by hand (O2-O11 of SURVEY.md section 8(c))
    s = make_config("c3", 9)
    rec = {}
    O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, 40, O.make_policy(u0=O.FP16, eta_rule=O.ETA_LINEAR),
              trace=lambda k, d: rec.setdefault(k, d))
    diag = np.array([s.vals[s.rowptr[i]:s.rowptr[i + 1]][s.colidx[s.rowptr[i]:s.rowptr[i + 1]] == i][0] for i in range(s.n)])
    dinv32 = O.round_fp32(1.0 / diag)
    k = max(rec) - 1
    a, b = rec[k], rec[k + 1]
    ur = int(b["ur"])
    assert ur == O.FP32 and int(b["uz"]) == O.FP16
    z, _ = O.step_z(a["r"], b["omega"], dinv32, ur, O.FP16)
    assert np.array_equal(z, b["z"])
    assert O.dot(a["r"], z) == b["rho"]
    p, _ = O.step_p(b["beta"], a["p"], z, O.FP16)
    assert np.array_equal(p, b["p"])
    q = O.spmv_fp32(s.rowptr, s.colidx, s.vals, p)
    assert np.array_equal(q, b["q"]) and O.dot(q, p) == b["gamma"]
    x, r = O.step_xr(b["alpha"], p, q, a["x"], a["r"], ur)
    assert np.array_equal(x, b["x"]) and np.array_equal(r, b["r"])
    assert np.sqrt(O.dot(r, r)) == b["delta_next"]


def test_classify_fp16_on_hand_made_values():
    # 1 = became inf, 2 = flushed to zero, 3 = subnormal, 0 = other (underflow is what breaks naive FP16)
    tiny = 2.0 ** -14  # smallest normal binary16
    assert O.classify_fp16(70000.0, np.inf) == 1
    assert O.classify_fp16(np.inf, np.inf) == 0          # was already inf: not an overflow of the store
    assert O.classify_fp16(1e-9, 0.0) == 2
    assert O.classify_fp16(-2.0 ** -26, -0.0) == 2
    assert O.classify_fp16(0.0, 0.0) == 0                # an exact zero is not a flush
    assert O.classify_fp16(3.0e-5, float(np.float16(3.0e-5))) == 3
    assert O.classify_fp16(tiny - 2.0 ** -24, tiny - 2.0 ** -24) == 3   # largest subnormal
    assert O.classify_fp16(2.0 ** -24, 2.0 ** -24) == 3                  # smallest subnormal
    assert O.classify_fp16(tiny, tiny) == 0                              # smallest normal
    assert O.classify_fp16(-tiny * 1.5, -tiny * 1.5) == 0
    assert O.classify_fp16(1.0, 1.0) == 0 and O.classify_fp16(65504.0, 65504.0) == 0
    # and through step_z: values chosen to land in each class
    r = np.array([1.0, 2.0 ** -20, 2.0 ** -30, 1e6, 0.0])
    z, counts = O.step_z(r, 1.0, np.ones(5), O.FP64, O.FP16)
    assert list(counts) == [1, 1, 1]  # inf: 1e6; flushed: 2^-30; subnormal: 2^-20
    assert z[0] == 1.0 and z[1] == 2.0 ** -20 and z[2] == 0.0 and np.isinf(z[3]) and z[4] == 0.0


@pytest.mark.parametrize("name,size", [("c1", 64), ("c2", 21), ("c3", 19), ("c4", 13), ("c5", 20011)])
def test_strict_rounding_diagnostic_changes_nothing_that_matters(name, size):
    # reading R6: rounding y and M^-1 to u_z separately (the paper's literal :238-239, Table 2's FP16 M)
    # instead of once gives the same iteration and switch counts and the same attainable accuracy
    s = make_config(name, size)
    for kw in (dict(), dict(u0=O.FP16, eta_rule=O.ETA_LINEAR)):
        a = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(**kw))
        b = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(strict_rounding=1, **kw))
        assert b.status == a.status == 0
        assert abs(b.iters - a.iters) <= 1
        assert (b.it_ur32, b.it_uz32, b.it_uz16) == (a.it_ur32, a.it_uz32, a.it_uz16)
        assert b.relres_true <= 2 * s.tol
        assert not np.array_equal(a.hist, b.hist)  # it IS a different rounding: the branch is exercised


def test_duplicate_diagonal_entries_add_up():
    # amp_pcg.h: duplicate entries are summed by the mat-vec, so M = diag(A) sums them too
    rowptr = np.array([0, 3, 5], dtype=np.int32)
    colidx = np.array([0, 0, 1, 0, 1], dtype=np.int32)
    vals = np.array([1.5, 2.5, 1.0, 1.0, 3.0])      # A = [[4, 1], [1, 3]]
    b = np.array([1.0, 2.0])
    r = O.amp_pcg(rowptr, colidx, vals, b, 1e-12, 10, O.make_policy(amp=0))
    assert r.status == 0 and r.iters <= 2
    assert np.allclose(r.x, np.linalg.solve(np.array([[4.0, 1.0], [1.0, 3.0]]), b), rtol=1e-12)
    rec = {}
    O.amp_pcg(rowptr, colidx, vals, b, 1e-12, 1, O.make_policy(amp=0), trace=lambda k, d: rec.setdefault(k, d))
    assert np.array_equal(rec[0]["z"], b / np.array([4.0, 3.0]))  # z_0 = M^-1 r_0 with M = diag(4, 3)
