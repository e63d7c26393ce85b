"""Pin P4 — the oracle's storage-rounding emulation against IEEE 754 facts.

binary16 / binary32 are the storage formats of z, p and r, q.  The
pins are facts of IEEE 754 (format tables, tie cases) and two independent implementations
(numpy's float16/float32 casts, g++'s _Float16 via a separately compiled helper is not needed:
numpy's cast is a different code base from the oracle's frexp/nearbyint arithmetic).
"""
import numpy as np

import oracle as O


def test_fp16_exhaustive_roundtrip():
    # every one of the 65 536 binary16 patterns is a fixed point of the rounding
    bits = np.arange(65536, dtype=np.uint16)
    h = bits.view(np.float16).astype(np.float64)
    finite = np.isfinite(h)
    out = O.round_fp16(h[finite])
    assert np.array_equal(out, h[finite])
    assert np.array_equal(np.signbit(out), np.signbit(h[finite]))  # -0.0 keeps its sign


def test_fp16_midpoints_tie_to_even_exhaustive():
    # the midpoint of every pair of adjacent positive finite halves rounds to the one with even pattern
    bits = np.arange(0, 0x7BFF, dtype=np.uint16)  # up to the one below 65504
    lo = bits.view(np.float16).astype(np.float64)
    hi = (bits + 1).astype(np.uint16).view(np.float16).astype(np.float64)
    mid = 0.5 * (lo + hi)  # exact in double
    want = np.where(bits % 2 == 0, lo, hi)
    assert np.array_equal(O.round_fp16(mid), want)
    assert np.array_equal(O.round_fp16(-mid), -want)
    # just off the midpoint goes to the nearer neighbour (direct rounding, no double rounding)
    eps = np.maximum(mid, 1e-30) * 2.0 ** -40
    assert np.array_equal(O.round_fp16(mid + eps), hi)
    assert np.array_equal(O.round_fp16(mid - eps), lo)


def test_fp16_special_values():
    r = lambda v: float(O.round_fp16(v)[0])
    assert r(65504.0) == 65504.0
    assert r(65519.999) == 65504.0
    assert r(65520.0) == np.inf and r(-65520.0) == -np.inf  # overflow -> inf (reading R11)
    assert r(1e300) == np.inf
    assert r(2.0 ** -14) == 2.0 ** -14  # smallest normal
    assert r(2.0 ** -24) == 2.0 ** -24  # smallest subnormal
    assert r(2.0 ** -25) == 0.0  # half-way to the smallest subnormal ties to even = 0
    assert r(2.0 ** -25 * (1 + 2.0 ** -30)) == 2.0 ** -24
    assert r(3 * 2.0 ** -25) == 2.0 ** -23  # tie between 1 and 2 quanta -> even (2)
    assert r(1.0 + 2.0 ** -11) == 1.0  # tie -> even mantissa
    assert r(1.0 + 2.0 ** -10 + 2.0 ** -11) == 1.0 + 2.0 ** -9
    # double-rounding trap: through float this would land on the tie and go to 1.0
    assert r(1.0 + 2.0 ** -11 + 2.0 ** -40) == 1.0 + 2.0 ** -10
    assert np.isnan(r(np.nan))


def test_fp16_random_vs_numpy():
    rng = np.random.default_rng(1)
    v = np.concatenate([
        rng.standard_normal(200000) * 10.0 ** rng.uniform(-9, 5, 200000),
        rng.uniform(-7e4, 7e4, 50000),
        rng.uniform(-1e-4, 1e-4, 50000),
    ])
    with np.errstate(over="ignore"):
        want = v.astype(np.float16).astype(np.float64)
    assert np.array_equal(O.round_fp16(v), want)


def test_fp32_random_vs_numpy_and_specials():
    rng = np.random.default_rng(2)
    v = rng.standard_normal(200000) * 10.0 ** rng.uniform(-50, 40, 200000)
    with np.errstate(over="ignore"):
        want = v.astype(np.float32).astype(np.float64)
    assert np.array_equal(O.round_fp32(v), want)
    r = lambda x: float(O.round_fp32(x)[0])
    assert r(1.0 + 2.0 ** -24) == 1.0  # tie -> even
    assert r(1.0 + 2.0 ** -24 + 2.0 ** -50) == 1.0 + 2.0 ** -23
    assert r(2.0 ** -149) == 2.0 ** -149 and r(2.0 ** -150) == 0.0
    assert r(3.5e38) == np.inf
