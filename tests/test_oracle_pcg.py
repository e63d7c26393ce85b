"""Pins P2/P3 — the oracle's FP64 PCG (Algorithm 3.1) and dynamic scaling
(Algorithm 3.2 / Theorem 3.2) against textbook CG facts:

* finite termination in at most (#distinct eigenvalues) <= n steps;
* A-orthogonality of the search directions and M^-1-orthogonality of the residuals (:46);
* the dense Cholesky / LAPACK solution for n <= 512 and monotone decrease of ||e_k||_A;
* the bound ||e_k||_A <= 2 ((sqrt(kappa)-1)/(sqrt(kappa)+1))^k ||e_0||_A with closed-form kappa;
* Theorem 3.2: DS-PCG == PCG (bit-identical for power-of-two omega, ~1e-14 for omega = 1/||r||).
"""
import json
import os

import numpy as np
import pytest

import oracle as O
from workloads import make_config, dense_spd_from_spectrum, fe27_laplacian

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _trace_run(s, policy, tol=None, maxit=None):
    rec = []
    res = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, tol or s.tol, maxit or s.maxit, policy,
                    trace=lambda k, d: rec.append(d))
    return res, rec


def test_finite_termination_distinct_eigenvalues():
    # 5 distinct eigenvalues, n = 40, well conditioned: CG converges in <= 5 steps
    lam = np.repeat([1.0, 1.5, 2.0, 3.0, 4.0], 8)
    rowptr, colidx, vals = dense_spd_from_spectrum(lam, seed=3)
    b = np.random.default_rng(0).standard_normal(40)
    res = O.pcg_fp64(rowptr, colidx, vals, b, 1e-12, 100, precond=O.PRECOND_NONE)
    assert res.status == 0 and res.iters <= 5
    assert res.relres_true <= 1e-11
    # full spectrum, n = 12, kappa = 4: at most n steps
    lam = np.linspace(1.0, 4.0, 12)
    rowptr, colidx, vals = dense_spd_from_spectrum(lam, seed=4)
    b = np.random.default_rng(1).standard_normal(12)
    res = O.pcg_fp64(rowptr, colidx, vals, b, 1e-13, 100, precond=O.PRECOND_NONE)
    assert res.status == 0 and res.iters <= 12


@pytest.mark.parametrize("name,size", [("c3", 5), ("c5", 200), ("c4", 5)])
def test_orthogonality_relations(name, size):
    s = make_config(name, size)
    A = s.scipy().toarray()
    dinv = 1.0 / np.diag(A)
    res, rec = _trace_run(s, O.make_policy(amp=0), tol=1e-12)
    K = min(8, len(rec))
    P = np.array([rec[k]["p"] for k in range(K)])
    # residual r_k (before the update of iteration k) = b - A x_{k}; r after update is rec[k]["r"]
    R = np.array([s.b] + [rec[k]["r"] for k in range(K - 1)])
    PAP = P @ A @ P.T
    RMR = (R * dinv) @ R.T
    dP, dR = np.sqrt(np.diag(PAP)), np.sqrt(np.diag(RMR))
    offP = np.abs(PAP / np.outer(dP, dP) - np.eye(K)).max()
    offR = np.abs(RMR / np.outer(dR, dR) - np.eye(K)).max()
    assert offP < 1e-9 and offR < 1e-9
    # scalars are what the algorithm says they are (Alg 3.1 lines 4, 10, 11)
    for k in range(K):
        z = R[k] * dinv
        assert rec[k]["rho"] == pytest.approx(R[k] @ z, rel=1e-13)
        assert rec[k]["gamma"] == pytest.approx(P[k] @ A @ P[k], rel=1e-12)
        assert rec[k]["alpha"] == pytest.approx(rec[k]["rho"] / rec[k]["gamma"], rel=1e-15)


@pytest.mark.parametrize("name,size", [("c1", 16), ("c2", 8), ("c3", 8), ("c4", 7), ("c5", 500)])
def test_against_dense_cholesky(name, size):
    s = make_config(name, size)
    assert s.n <= 512
    A = s.scipy().toarray()
    L = np.linalg.cholesky(A)  # LAPACK potrf: also certifies A is SPD
    xc = np.linalg.solve(L.T, np.linalg.solve(L, s.b))
    res, rec = _trace_run(s, O.make_policy(amp=0), tol=1e-13, maxit=2000)
    assert res.status == 0
    e = res.x - xc
    assert np.sqrt(e @ A @ e) <= 1e-10 * np.sqrt(xc @ A @ xc)
    # ||e_k||_A decreases monotonically (CG minimises the A-norm of the error over the Krylov space)
    errs = [np.sqrt(xc @ A @ xc)] + [np.sqrt((d["x"] - xc) @ A @ (d["x"] - xc)) for d in rec]
    errs = np.array(errs)
    head = errs[errs > 1e-9 * errs[0]]
    assert np.all(np.diff(head) <= 1e-12 * errs[0])
    # the updated residual equals the true residual to rounding in FP64
    d = rec[min(5, len(rec) - 1)]
    assert np.linalg.norm(s.b - A @ d["x"] - d["r"]) <= 1e-12 * np.linalg.norm(s.b)
    if s.xstar is not None:
        assert np.linalg.norm(res.x - s.xstar) <= 1e-8 * np.linalg.norm(s.xstar)


def test_closed_form_kappa_values():
    gold = json.load(open(os.path.join(GOLD, "closed_forms.json")))["kappa"]
    assert 1.0 / np.tan(np.pi / 130) ** 2 == pytest.approx(gold["c1_poisson2d_N64"]["value"], rel=1e-5)
    assert 1.0 / np.tan(np.pi / 258) ** 2 == pytest.approx(gold["c2_poisson3d_N128"]["value"], rel=1e-5)
    kf = lambda t: 2 - 2 * np.cos(t)
    mf = lambda t: (2 + np.cos(t)) / 3

    def fe_spectrum(N):
        t = np.arange(1, N + 1) * np.pi / (N + 1)
        k, m = kf(t), mf(t)
        return (np.einsum("i,j,k->ijk", k, m, m) + np.einsum("i,j,k->ijk", m, k, m)
                + np.einsum("i,j,k->ijk", m, m, k)).ravel()

    # the formula itself is pinned by LAPACK on a tiny grid
    N = 5
    rowptr, colidx, vals = fe27_laplacian(N)
    import scipy.sparse as sp
    A = sp.csr_matrix((vals, colidx, rowptr), shape=(N ** 3, N ** 3)).toarray()
    assert np.allclose(np.sort(np.linalg.eigvalsh(A)), np.sort(fe_spectrum(N)), atol=1e-12)
    lam = fe_spectrum(200)
    g = gold["c4_fe27_N200"]
    assert lam.min() == pytest.approx(g["lam_min"], rel=1e-3)
    assert lam.max() == pytest.approx(g["lam_max"], rel=1e-5)
    assert lam.max() / lam.min() == pytest.approx(g["value"], rel=1e-4)


def test_cg_error_bound_config1():
    # c1 full size: kappa = cot^2(pi/130) (Jacobi-invariant, constant diagonal); x* known
    s = make_config("c1")
    kappa = 1.0 / np.tan(np.pi / 130) ** 2
    sig = (np.sqrt(kappa) - 1) / (np.sqrt(kappa) + 1)
    A = s.scipy()
    res, rec = _trace_run(s, O.make_policy(amp=0))
    e0 = np.sqrt(s.xstar @ (A @ s.xstar))
    for k, d in enumerate(rec):
        e = d["x"] - s.xstar
        ek = np.sqrt(e @ (A @ e))
        assert ek <= 2.0 * sig ** (k + 1) * e0 * (1 + 1e-9) + 1e-13 * e0
    # iterations to tol are below the bound's count (396 for tol 1e-8) and not absurdly below
    bound_its = int(np.ceil(np.log(s.tol / 2) / np.log(sig)))
    assert 50 < res.iters <= bound_its
    assert res.relres_true <= s.tol * 1.01


# ------------------------------------------------------------------ Theorem 3.2 ------------
def _no_switch_policy(scale_mode):
    # Algorithm 3.2 = Algorithm 4.1 with every vector kept in FP64
    return O.make_policy(amp=1, u0=O.FP64, eta_rule=O.ETA_NEVER, tau_zs=0.0, tau_zh=0.0, scale_mode=scale_mode)


@pytest.mark.parametrize("name,size", [("c3", 10), ("c5", 2000)])
def test_theorem_3_2_pow2_scaling_is_bit_identical(name, size):
    s = make_config(name, size)
    _, ref = _trace_run(s, O.make_policy(amp=0), tol=1e-10)
    _, ds = _trace_run(s, _no_switch_policy(O.SCALE_POW2), tol=1e-10)
    assert len(ref) == len(ds) and len(ref) > 5
    for a, b in zip(ref, ds):
        assert np.array_equal(a["x"], b["x"]) and np.array_equal(a["r"], b["r"])
        w = b["omega"]
        assert w == 2.0 ** round(np.log2(w))
        # hatted quantities of the proof: z^ = w z, rho^ = w rho, gamma^ = w^2 gamma, alpha^ = alpha / w
        assert np.array_equal(b["z"], w * a["z"])
        assert b["rho"] == w * a["rho"] and b["gamma"] == w * w * a["gamma"] and b["alpha"] == a["alpha"] / w


@pytest.mark.parametrize("mode", [O.SCALE_NORM2, O.SCALE_RMS])
def test_theorem_3_2_norm_scaling_agrees_to_rounding(mode):
    s = make_config("c3", 10)
    A = s.scipy().toarray()
    d = np.diag(A)
    r1, ref = _trace_run(s, O.make_policy(amp=0), tol=1e-10)
    r2, ds = _trace_run(s, _no_switch_policy(mode), tol=1e-10)
    assert abs(r1.iters - r2.iters) <= 1
    for k in range(min(len(ref), len(ds), 60)):
        a, b = ref[k], ds[k]
        assert np.linalg.norm(a["x"] - b["x"]) <= 1e-11 * np.linalg.norm(a["x"])
        # invariant of the scaled residual: ||y_k|| = ||M z_k|| = 1 (NORM2) or sqrt(n) (RMS)
        ynorm = np.linalg.norm(b["z"] * d)
        assert ynorm == pytest.approx(1.0 if mode == O.SCALE_NORM2 else np.sqrt(s.n), rel=1e-13)
        assert b["omega"] * b["delta_k"] == pytest.approx(1.0 if mode == O.SCALE_NORM2 else np.sqrt(s.n), rel=1e-15)
        assert b["rho"] / b["omega"] == pytest.approx(a["rho"], rel=1e-9)


def test_edge_cases():
    s = make_config("c2", 6)
    # b = 0 -> x = 0, 0 iterations
    res = O.amp_pcg(s.rowptr, s.colidx, s.vals, np.zeros(s.n), 1e-8, 100, O.make_policy())
    assert res.status == 0 and res.iters == 0 and np.all(res.x == 0)
    # x0 = exact solution -> 0 iterations
    res = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, 1e-8, 100, O.make_policy(), x0=s.xstar)
    assert res.status == 0 and res.iters == 0
    # maxit reached -> status 1, iters = maxit
    res = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, 1e-14, 3, O.make_policy())
    assert res.status == 1 and res.iters == 3 and len(res.hist) == 4
    # a non-zero x0 is honoured: r0 = b - A x0
    x0 = np.random.default_rng(3).standard_normal(s.n)
    res = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, 1e-10, 500, O.make_policy(), x0=x0)
    assert res.status == 0 and res.relres_true <= 2e-10
    assert res.hist[0] == pytest.approx(np.linalg.norm(s.b - s.scipy() @ x0), rel=1e-14)
    # indefinite matrix -> breakdown status
    vals = s.vals.copy()
    vals[s.colidx == np.repeat(np.arange(s.n), np.diff(s.rowptr))] = 0.5  # diag 0.5 < row sum: indefinite
    res = O.amp_pcg(s.rowptr, s.colidx, vals, s.b, 1e-10, 500, O.make_policy(amp=0))
    assert res.status == -2


def test_theorem_3_2_lagged_scaling():
    """SCALE_LAGGED (reading R17): omega_k = 1/||r_{k-1}|| is one more admissible scaling of Algorithm 3.2
    (PAPER.md:223 offers ||z_{k-1}||^-1; Theorem 3.2 holds for any non-zero omega_k): with every vector in FP64 the
    iterates agree with PCG to rounding, omega_k ||r_{k-1}|| = 1 exactly, and ||y_k|| = ||r_k|| / ||r_{k-1}||."""
    s = make_config("c3", 10)
    d = np.diag(s.scipy().toarray())
    r1, ref = _trace_run(s, O.make_policy(amp=0), tol=1e-10)
    r2, ds = _trace_run(s, _no_switch_policy(O.SCALE_LAGGED), tol=1e-10)
    assert abs(r1.iters - r2.iters) <= 1
    hist = np.asarray(r2.hist)
    for k in range(min(len(ref), len(ds), 60)):
        a, b = ref[k], ds[k]
        assert np.linalg.norm(a["x"] - b["x"]) <= 1e-11 * np.linalg.norm(a["x"])
        prev = hist[max(k - 1, 0)]
        assert b["omega"] * prev == pytest.approx(1.0, rel=1e-15)
        assert np.linalg.norm(b["z"] * d) == pytest.approx(hist[k] / prev, rel=1e-12)
        assert b["rho"] / b["omega"] == pytest.approx(a["rho"], rel=1e-9)


@pytest.mark.parametrize("name,size", [("c1", 48), ("c2", 24), ("c3", 20), ("c4", 16)])
def test_lagged_decisions_take_effect_one_iteration_later(name, size):
    """In the lagged variant the selector (4.1) and the indicator (4.9)/(4.10) of iteration k see the norms up to
    ||r_{k-1}||: on these runs (same residual history to rounding) every switch happens exactly one iteration after the
    paper's, the iteration count is unchanged and the attainable accuracy (<= 2 tol) is kept."""
    s = make_config(name, size)
    for kw in (dict(u0=O.FP64, eta_rule=O.ETA_DELAY), dict(u0=O.FP16, eta_rule=O.ETA_LINEAR)):
        a = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(**kw))
        b = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(scale_mode=O.SCALE_LAGGED, **kw))
        assert a.status == b.status == 0
        if kw["u0"] == O.FP64:
            assert abs(a.iters - b.iters) <= 1
        else:
            # z, p in FP16 from the start: ||y_k|| = ||r_k|| / ||r_{k-1}|| < 1 uses less of FP16's range than the paper's
            # ||y_k|| = 1, which can cost a few iterations on fast-converging small systems (c4 at 16^3: 41 vs 37)
            assert a.iters - 1 <= b.iters <= 1.15 * a.iters + 1
        for key in ("it_ur32", "it_uz32", "it_uz16"):
            va, vb = getattr(a, key), getattr(b, key)
            assert (va < 0 and vb < 0) or vb == va + 1, (key, va, vb)
        assert b.relres_true <= 2 * s.tol
