"""Pins P5-P8 — the oracle's AMP-PCG (Algorithm 4.1), precision selector
(4.1) (:245-253) and indicators (4.9)/(4.10)/(4.11) (:359-375) against what the paper prints:

* Example 9: u_z -> FP32 at iteration 9, -> FP16 at iteration 11, PCG(FP64) > 10 its;
* Example 1 (:48-55, :416-420, :439): naive FP16 breaks down, AMP-PCG(FP64) mirrors FP64,
  AMP-PCG(u_r) reaches tol = 1e-6 and 1e-8;
* Examples 4, 6, 10 (:445-487, :568-572): which variants track FP64 and which are slower;
* ||b - A x_m|| <~ 2 tol ||b|| (:377-381).
"""
import json
import os

import numpy as np
import pytest

import oracle as O
from workloads import make_config, paper_example

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_printed_values.json")))
NOPC = O.PRECOND_NONE  # the paper's small examples use M = I


def _run(s, pol, tol=None, maxit=None):
    return O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, tol or s.tol, maxit or s.maxit, pol)


# ------------------------------------------------------------------ Example 9 (hard pin) ---
@pytest.mark.parametrize("identity_q,seed", [(True, 1), (False, 1), (False, 2), (False, 3), (False, 4)])
def test_example9_switch_iterations(identity_q, seed):
    g = GOLD["example9"]
    s = paper_example(9, seed=seed, identity_q=identity_q)
    assert s.n == g["n"]
    t = GOLD["thresholds_5_1"]
    # "all other vectors are maintained in double precision" -> u_r never switches
    pol = O.make_policy(u0=O.FP64, eta_rule=O.ETA_NEVER, tau_zs=t["tau_zs"], tau_zh=t["tau_zh"], precond=NOPC)
    amp = _run(s, pol)
    ref = _run(s, O.make_policy(amp=0, precond=NOPC))
    assert amp.it_uz32 == g["uz_to_fp32_iteration"]
    assert amp.it_uz16 == g["uz_to_fp16_iteration"]
    assert ref.iters > g["pcg_fp64_needs_more_than"] and ref.status == 0
    assert amp.status == 0 and amp.iters >= ref.iters  # "a few additional iterations"
    assert amp.iters <= ref.iters + 8


# ------------------------------------------------------------------ selector (4.1) ---------
def test_selector_table():
    pol = O.make_policy(u0=O.FP64, tau_zs=1e-4, tau_zh=1e-6)
    assert O.select_uz(pol, 1.0) == O.FP64
    assert O.select_uz(pol, 1e-4) == O.FP64  # nu >= tau_zs keeps u0
    assert O.select_uz(pol, 0.999e-4) == O.FP32
    assert O.select_uz(pol, 1e-6) == O.FP32  # tau_zh <= nu < tau_zs
    assert O.select_uz(pol, 0.999e-6) == O.FP16
    for u0 in (O.FP32, O.FP16):  # min{u0, .} returns the lower precision
        pol = O.make_policy(u0=u0)
        assert O.select_uz(pol, 1.0) == u0
        assert O.select_uz(pol, 1e-5) == max(u0, O.FP32)
        assert O.select_uz(pol, 1e-9) == O.FP16
    pol = O.make_policy(u0=O.FP64, tau_zs=1e-4, tau_zh=0.0)  # tau_zh = 0: never half
    assert O.select_uz(pol, 1e-300) == O.FP32


# ------------------------------------------------------------------ eta closed forms -------
def test_eta_delay_closed_forms():
    d, Cc, e32 = 10, 1.0, 2.0 ** -24
    pol = O.make_policy(eta_rule=O.ETA_DELAY, d=d, C_=Cc)
    # constant history h: eta = (d+1) eps32 (5+2C) h
    h = np.full(40, 3.0)
    for k in (0, 3, 10, 25):
        assert O.eta(pol, h, k) == pytest.approx((d + 1) * e32 * (5 + 2 * Cc) * 3.0, rel=1e-14)
    # geometric history h_t = g^t, k >= d+1: sum of a geometric series
    g = 0.7
    h = g ** np.arange(60.0)
    k = 30
    t = np.arange(k - d, k + 1)
    want = e32 * ((3 + Cc) * np.sum(g ** (t - 1.0)) + (2 + Cc) * np.sum(g ** (t * 1.0)))
    assert O.eta(pol, h, k) == pytest.approx(want, rel=1e-13)
    # early window (reading R2): norms with negative index are ||r_0||
    k = 2
    hh = np.array([5.0, 4.0, 3.0])
    terms = [(5.0, 5.0)] * (d - 2) + [(5.0, 5.0), (5.0, 4.0), (4.0, 3.0)]  # t = k-d .. k, (h_{t-1}, h_t)
    want = e32 * sum((3 + Cc) * a + (2 + Cc) * b for a, b in terms)
    assert O.eta(pol, hh, k) == pytest.approx(want, rel=1e-14)
    # other d, C
    pol2 = O.make_policy(eta_rule=O.ETA_DELAY, d=3, C_=2.0)
    assert O.eta(pol2, np.full(10, 1.0), 7) == pytest.approx(4 * e32 * 9.0, rel=1e-14)


def test_eta_linear_bounds_the_geometric_tail():
    # (4.11): for ||r_t|| = ||r_k|| g^(t-k) the tail sum is <= eps32 (5+2C) ||r_{k-1}|| / (1-g)
    e32, Cc, ell = 2.0 ** -24, 1.0, 5
    pol = O.make_policy(eta_rule=O.ETA_LINEAR, ell=ell, C_=Cc)
    for g in (0.3, 0.9, 0.99):
        h = 7.0 * g ** np.arange(80.0)
        k = 40
        eta = O.eta(pol, h, k)
        t = np.arange(k, 20000)
        tail = e32 * np.sum((3 + Cc) * 7.0 * g ** (t - 1.0) + (2 + Cc) * 7.0 * g ** (t * 1.0))
        assert eta == pytest.approx(e32 * (5 + 2 * Cc) * h[k - 1] / (1 - g), rel=1e-10)
        assert tail <= eta * (1 + 1e-12)
        assert eta <= tail * (5 + 2 * Cc) / ((3 + Cc) + (2 + Cc) * g) * (1 + 1e-9)
    # not defined before ell iterations or when the residual did not decrease: +inf (no switch)
    assert O.eta(pol, h, ell - 1) == np.inf
    assert O.eta(pol, np.array([1.0, 1, 1, 1, 1, 1, 2.0]), 6) == np.inf
    assert O.eta(O.make_policy(eta_rule=O.ETA_NEVER), h, 30) == np.inf


# ------------------------------------------------------------------ Example 1 --------------
def test_example1_naive_fp16_breaks_down_and_amp_mirrors_fp64():
    for seed in (1, 2, 3):
        s = paper_example(1, seed=seed)
        ref = _run(s, O.make_policy(amp=0, precond=NOPC))
        assert ref.status == 0 and ref.relres_true <= 1.5e-10
        # naive low precision: z, p in FP16, no scaling: z underflows, rho -> 0,
        # breakdown (the oracle reports it as status -2) or stagnation far above tol
        naive = _run(s, O.make_policy(u0=O.FP16, eta_rule=O.ETA_NEVER, scale_mode=O.SCALE_NONE, precond=NOPC),
                     maxit=400)
        assert naive.status != 0
        assert naive.fp16_flushed > 0
        # same precisions WITH the dynamic scaling of Alg 4.1: no flush-to-zero breakdown
        scaled = _run(s, O.make_policy(u0=O.FP16, eta_rule=O.ETA_NEVER, precond=NOPC), maxit=400)
        assert scaled.status == 0
        # AMP-PCG(FP64) "closely mirrors" PCG(FP64)
        amp = _run(s, O.make_policy(precond=NOPC))
        assert amp.status == 0 and abs(amp.iters - ref.iters) <= max(4, ref.iters // 10)
        assert amp.relres_true <= 2.0 * s.tol
        assert 0 <= amp.it_uz32 <= amp.it_uz16 and amp.it_ur32 >= 0


@pytest.mark.parametrize("tol", [1e-6, 1e-8])
def test_example1_ur_switch_reaches_tolerance(tol):
    # AMP-PCG(u_r): u_z fixed FP64, iterations not stopped; the true residual
    # is driven below tol.  This decides the early-window reading R2 (zero padding fails it).
    for seed in (1, 2, 3):
        s = paper_example(1, seed=seed)
        pol = O.make_policy(u0=O.FP64, tau_zs=0.0, tau_zh=0.0, no_stop=1, precond=NOPC)
        res = _run(s, pol, tol=tol, maxit=150)
        assert res.it_ur32 > 0
        assert res.relres_true <= tol
        # and with FP32 from the start the attainable accuracy is worse than with the switch
        early = _run(s, O.make_policy(u0=O.FP64, tau_zs=0.0, tau_zh=0.0, no_stop=1, precond=NOPC, eps32=1e-30),
                     tol=tol, maxit=150)
        assert early.it_ur32 == 0 and early.relres_true > res.relres_true


# ------------------------------------------------------------------ Examples 4, 6, 10 ------
def test_example4_fp16_throughout_tracks_fp64():
    s = paper_example(4)
    ref = _run(s, O.make_policy(amp=0, precond=NOPC))
    amp = _run(s, O.make_policy(u0=O.FP16, eta_rule=O.ETA_LINEAR, precond=NOPC))
    assert ref.status == 0 and amp.status == 0
    assert abs(amp.iters - ref.iters) <= 2  # "nearly identical"
    assert amp.it_ur32 > 0 and amp.relres_true <= 2 * s.tol


def test_example6_fp16_is_slower_fp64_start_is_not():
    s = paper_example(6)
    ref = _run(s, O.make_policy(amp=0, precond=NOPC))
    a64 = _run(s, O.make_policy(u0=O.FP64, precond=NOPC))
    a16 = _run(s, O.make_policy(u0=O.FP16, precond=NOPC), maxit=1000)
    assert abs(a64.iters - ref.iters) <= 3  # "nearly identical"
    assert a16.iters > ref.iters * 1.2  # "converges more slowly"
    assert a64.relres_true <= 2 * s.tol


def test_example10_threshold_sensitivity():
    s = paper_example(10)
    ref = _run(s, O.make_policy(amp=0, precond=NOPC), maxit=2000)
    hi = _run(s, O.make_policy(u0=O.FP64, eta_rule=O.ETA_NEVER, tau_zs=1e-4, tau_zh=0.0, precond=NOPC), maxit=2000)
    lo = _run(s, O.make_policy(u0=O.FP64, eta_rule=O.ETA_NEVER, tau_zs=1e-8, tau_zh=0.0, precond=NOPC), maxit=2000)
    assert hi.it_uz16 == -1 and lo.it_uz16 == -1  # tau_zh = 0: never half
    assert abs(lo.iters - ref.iters) <= 2  # "almost identical"
    assert hi.iters >= ref.iters + 5  # tau_zs = 1e-4 degrades convergence


# ------------------------------------------------------------------ accuracy guarantee ------
@pytest.mark.parametrize("name,size", [("c1", 32), ("c2", 20), ("c3", 16), ("c4", 14), ("c5", 20000)])
def test_final_true_residual_within_2tol(name, size):
    s = make_config(name, size)
    ref = _run(s, O.make_policy(amp=0))
    for pol in (O.make_policy(), O.make_policy(u0=O.FP16, eta_rule=O.ETA_LINEAR)):
        res = _run(s, pol)
        assert res.status == 0
        assert res.relres_updated <= s.tol
        assert res.relres_true <= GOLD["final_accuracy_factor"]["factor"] * s.tol
        assert abs(res.iters - ref.iters) <= max(2, int(0.05 * ref.iters))
    # strict theta-split of (3.10) (reading R12): true residual <= tol
    strict = _run(s, O.make_policy(eta_safety=0.1, stop_safety=0.9))
    assert strict.relres_true <= s.tol


def test_switches_are_latched_and_ordered():
    s = make_config("c3", 14)
    hist_prec = []
    O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(),
              trace=lambda k, d: hist_prec.append((d["ur"], d["uz"])))
    ur = [a for a, _ in hist_prec]
    uz = [b for _, b in hist_prec]
    assert ur == sorted(ur) and uz == sorted(uz)  # monotone: precision only decreases (reading R5)
    assert ur[-1] == O.FP32 and uz[-1] == O.FP16


def test_stored_vectors_are_representable():
    s = make_config("c2", 10)
    seen = {"n": 0}

    def chk(k, d):
        if d["uz"] == O.FP16:
            assert np.array_equal(d["z"], O.round_fp16(d["z"])) and np.array_equal(d["p"], O.round_fp16(d["p"]))
            seen["n"] += 1
        elif d["uz"] == O.FP32:
            assert np.array_equal(d["z"], O.round_fp32(d["z"])) and np.array_equal(d["p"], O.round_fp32(d["p"]))
        if d["ur"] == O.FP32:
            assert np.array_equal(d["r"], O.round_fp32(d["r"])) and np.array_equal(d["q"], O.round_fp32(d["q"]))

    O.amp_pcg(s.rowptr, s.colidx, s.vals, s.b, s.tol, s.maxit, O.make_policy(), trace=chk)
    assert seen["n"] > 0
