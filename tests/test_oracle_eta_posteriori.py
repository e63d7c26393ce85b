"""Pins of the oracle's a-posteriori indicator eta_hat_m(k), eq. (4.7), against what the
formula itself fixes: a closed form on a geometric residual history, its two limiting cases, its relation to
the computable indicator (4.9), and the monotonicity the paper states (:356 "eta_hat_m(k-d) > eta_hat_m(k)")."""
import numpy as np
import pytest

import oracle as O

E32, E64 = 2.0 ** -24, 2.0 ** -53


def _geometric(m, rho):
    return rho ** np.arange(m + 1, dtype=np.float64)


@pytest.mark.parametrize("rho,C", [(0.5, 1.0), (0.9, 1.0), (0.25, 0.0), (0.7, 3.0)])
def test_closed_form_on_geometric_history(rho, C):
    # ||r_t|| = rho^t, ||r_{-1}|| := ||r_0|| = 1.  c_0 = 5 + 2C, c_t = rho^(t-1) ((3+C) + (2+C) rho) for t >= 1.
    m = 40
    h = _geometric(m, rho)
    g = (3.0 + C) + (2.0 + C) * rho

    def csum(a, b):  # sum_{t=a..b} c_t
        s = (5.0 + 2.0 * C) if a == 0 else 0.0
        lo = max(a, 1)
        if b >= lo:
            s += g * (rho ** (lo - 1) - rho ** b) / (1.0 - rho)
        return s

    for k in (0, 1, 7, 23, m):
        expect = E64 * csum(0, k) + E32 * csum(k, m)
        assert O.eta_posteriori(h, k, C) == pytest.approx(expect, rel=1e-12)


def test_limiting_cases_and_monotonicity():
    rng = np.random.default_rng(3)
    h = np.abs(rng.standard_normal(60)) * 10.0 ** (-np.arange(60) / 6.0)
    m = len(h) - 1
    c = 4.0 * np.concatenate([[h[0]], h[:-1]]) + 3.0 * h  # C = 1
    # switching at k = m: everything in FP64 but the last term; at k = 0: everything in FP32 but the first
    assert O.eta_posteriori(h, m) == pytest.approx(E64 * c.sum() + E32 * c[m], rel=1e-12)
    assert O.eta_posteriori(h, 0) == pytest.approx(E64 * c[0] + E32 * c.sum(), rel=1e-12)
    # the later the switch, the better the attainable accuracy
    vals = [O.eta_posteriori(h, k) for k in range(m + 1)]
    assert all(a > b for a, b in zip(vals, vals[1:]))
    # the eps32 and eps64 parts are separately linear in their epsilon
    assert O.eta_posteriori(h, 17, 1.0, 2 * E32, E64) - O.eta_posteriori(h, 17) == pytest.approx(E32 * c[17:].sum(), rel=1e-9)


def test_computable_indicator_is_the_dominant_part():
    # (4.9): eta_k = the eps32 terms t = k-d..k, i.e. eta_hat_m(k-d) minus its eps64 part and minus the terms after k
    h = _geometric(80, 0.8)
    pol = O.make_policy(d=10)
    for k in (10, 25, 60):
        full = O.eta_posteriori(h, k - 10, 1.0, E32, 0.0)          # eps64 part switched off
        after = O.eta_posteriori(h, k + 1, 1.0, E32, 0.0)          # terms t = k+1..m
        assert O.eta(pol, h, k) == pytest.approx(full - after, rel=1e-10)
        # and (4.8): with a decaying history the neglected part is small
        assert O.eta(pol, h, k) <= full


@pytest.mark.parametrize("ex", [1, 4, 6])
@pytest.mark.parametrize("tol", [1e-6, 1e-8])
def test_estimates_the_attainable_accuracy_of_the_paper_examples(ex, tol):
    """PAPER.md:350 ("estimates the best attainable accuracy"), :439 and Fig. 3: run AMP-PCG(u_r) (z, p stay FP64) far
    past convergence; the true residual stagnates at the attainable accuracy, which eta_hat_m(k_switch) must bound from
    above without being orders of magnitude off, and which respects the switching criterion (4.10)."""
    from workloads import paper_example

    s = paper_example(ex)
    pol = O.make_policy(amp=1, u0=0, eta_rule=0, precond=0, no_stop=1, tau_zs=0.0, tau_zh=0.0)
    r = O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, tol, 150, pol)
    assert r.it_ur32 > 0 and r.it_uz32 < 0
    eh = O.eta_posteriori(np.asarray(r.hist), r.it_ur32) / r.bnorm
    assert r.relres_updated < 1e-3 * r.relres_true      # the recursive residual keeps falling, the true one stagnates
    assert r.relres_true <= eh <= 10.0 * r.relres_true
    assert eh <= tol
