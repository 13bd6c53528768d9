"""Pins for the oracle's storage-format codecs (DESIGN.md readings
Q6, Q7).  None of these re-types the oracle's formula: they use numpy's casts (library), exact
rational arithmetic, exhaustive enumeration and the closed forms the paper's definition implies."""
from fractions import Fraction

import numpy as np
import pytest

import oracle

MAXINT = {"int32": 2147483647, "int16": 32767}


def _rng(seed):
    return np.random.default_rng(seed)


# ----------------------------------------------------------------------------- fp64 / fp32
def test_fp64_identity():
    v = _rng(10).standard_normal(1000)
    p, s = oracle.enc("fp64", v)
    assert s == 1.0 and np.array_equal(p, v) and np.array_equal(oracle.dec("fp64", p, s), v)


def test_fp32_equals_numpy_cast_bitwise():
    rng = _rng(11)
    v = np.concatenate([rng.uniform(-1, 1, 500_000), rng.standard_normal(400_000) * 1e-3,
                        rng.uniform(-1, 1, 100_000) * 10.0 ** rng.uniform(-46, 0, 100_000), [0.0, -0.0, 1.0, -1.0]])
    p, s = oracle.enc("fp32", v)
    assert s == 1.0
    assert np.array_equal(p.view(np.uint32), v.astype(np.float32).view(np.uint32))
    assert np.array_equal(oracle.dec("fp32", p, s), p.astype(np.float64))


def test_fp32_midpoints_tie_to_even_and_neighbours_round_to_nearest():
    rng = _rng(12)
    a = np.abs(rng.uniform(-1, 1, 20000).astype(np.float32))
    a = np.concatenate([a, np.float32([0.0, 1e-45, 1.1754942e-38, 1.17549435e-38, 0.5, 0.99999994])])
    up = np.nextafter(a, np.float32(np.inf))
    mid = (a.astype(np.float64) + up.astype(np.float64)) / 2  # exact in fp64
    even = np.where((a.view(np.uint32) & 1) == 0, a, up)
    for sign in (1.0, -1.0):
        got, _ = oracle.enc("fp32", sign * mid)
        assert np.array_equal(got, (sign * even).astype(np.float32))
        lo, _ = oracle.enc("fp32", sign * np.nextafter(mid, 0.0))
        hi, _ = oracle.enc("fp32", sign * np.nextafter(mid, np.inf))
        assert np.array_equal(lo, (sign * a).astype(np.float32))
        assert np.array_equal(hi, (sign * up).astype(np.float32))


# ----------------------------------------------------------------------------- fp16
def _all_finite_halves():
    bits = np.arange(0x10000, dtype=np.uint32).astype(np.uint16)
    h = bits.view(np.float16)
    return h[np.isfinite(h)]


def test_fp16_exhaustive_round_trip():
    h = _all_finite_halves()
    assert h.size == 63488
    d = oracle.dec("fp16", h)
    assert np.array_equal(d, h.astype(np.float64))  # exact widening, incl. subnormals and -0
    back, s = oracle.enc("fp16", d)
    assert s == 1.0
    assert np.array_equal(back.view(np.uint16), h.view(np.uint16))


def test_fp16_midpoints_single_rounding():
    """Every adjacent pair of non-negative halves: the exact midpoint ties to even, and the fp64
    neighbours of the midpoint round to the nearer half.  Values just above a midpoint are the
    ones a double rounding through fp32 gets wrong (reading Q7: one rounding)."""
    bits = np.arange(0, 0x7BFF, dtype=np.uint16)  # up to the pair (65472, 65504)
    a = bits.view(np.float16)
    up = (bits + 1).astype(np.uint16).view(np.float16)
    mid = (a.astype(np.float64) + up.astype(np.float64)) / 2
    even_bits = np.where((bits & 1) == 0, bits, bits + 1).astype(np.uint16)
    for sign, sbit in ((1.0, 0), (-1.0, 0x8000)):
        got, _ = oracle.enc("fp16", sign * mid)
        assert np.array_equal(got.view(np.uint16), even_bits | sbit)
        lo, _ = oracle.enc("fp16", sign * np.nextafter(mid, 0.0))
        hi, _ = oracle.enc("fp16", sign * np.nextafter(mid, np.inf))
        assert np.array_equal(lo.view(np.uint16), bits | sbit)
        assert np.array_equal(hi.view(np.uint16), (bits + 1).astype(np.uint16) | sbit)


def test_fp16_double_rounding_witness():
    # 1 + 2^-11 + 2^-30 lies just above the half midpoint between 1 and 1+2^-10; through fp32 it
    # would first round to the midpoint and then tie down to 1.0.  One rounding gives 1+2^-10.
    x = 1.0 + 2.0 ** -11 + 2.0 ** -30
    assert np.float32(x) == np.float32(1.0 + 2.0 ** -11)
    got, _ = oracle.enc("fp16", np.array([x]))
    assert float(got[0]) == 1.0 + 2.0 ** -10


def test_fp16_equals_numpy_cast_and_gradual_underflow():
    rng = _rng(13)
    v = np.concatenate([rng.uniform(-1, 1, 300_000), rng.standard_normal(300_000) * 5e-4,
                        rng.uniform(-1, 1, 100_000) * 10.0 ** rng.uniform(-9, 0, 100_000)])
    p, _ = oracle.enc("fp16", v)
    assert np.array_equal(p.view(np.uint16), v.astype(np.float16).view(np.uint16))
    # gradual underflow: values below the smallest normal 2^-14 are kept as subnormals, not flushed
    tiny = np.array([3.0e-5, -2.0e-6, 6.0e-8, 2.0 ** -25 * 1.0001, 2.0 ** -25, 2.0 ** -26])
    q, _ = oracle.enc("fp16", tiny)
    assert np.array_equal(q.astype(np.float64)[:3] != 0, [True, True, True])
    assert float(q[3]) == 2.0 ** -24 and float(q[4]) == 0.0 and float(q[5]) == 0.0


# ----------------------------------------------------------------------------- fixed point
@pytest.mark.parametrize("fmt", ["int32", "int16"])
def test_fixed_point_closed_forms(fmt):
    M = MAXINT[fmt]
    rng = _rng(14)
    n = 100_000
    w = rng.standard_normal(n)
    v = w / np.linalg.norm(w)  # a unit vector, entries bounded by 1
    q, sigma = oracle.enc(fmt, v)
    a = np.abs(v).max()
    # sigma_j = (||w||inf / ||w||2) / max_int == ||v||inf / max_int
    assert sigma == a / M
    assert abs(sigma - (np.abs(w).max() / np.linalg.norm(w)) / M) <= 4 * np.finfo(float).eps * sigma
    # the entry of largest magnitude uses the full integer range; nothing exceeds it
    assert abs(int(q[np.argmax(np.abs(v))])) == M
    assert np.abs(q.astype(np.int64)).max() == M
    d = oracle.dec(fmt, q, sigma)
    assert np.abs(d).max() <= a and np.abs(d).max() <= 1.0
    # rounding to nearest: error at most half a step (+ fp64 round-off of s*sigma != 1)
    assert np.all(np.abs(d - v) <= sigma / 2 + 2.0 ** -50 * np.abs(v))
    # odd symmetry
    qn, sn = oracle.enc(fmt, -v)
    assert sn == sigma and np.array_equal(qn, -q)
    # decode is q * sigma in one fp64 multiply
    assert np.array_equal(d, q.astype(np.float64) * sigma)


@pytest.mark.parametrize("fmt", ["int32", "int16"])
def test_fixed_point_lossless_on_grid(fmt):
    # entries that are exact multiples of sigma = 2^-k/... : choose a = 1 * 2^-3 * M/M so that
    # v_i = q_i * 2^-3 / M is not exactly representable in general; use a power-of-two step instead:
    M = MAXINT[fmt]
    rng = _rng(15)
    q0 = rng.integers(-M, M + 1, size=5000)
    q0[0] = M
    # v = q0 * sigma with sigma = a/M, a = M * 2^-40  ->  sigma = 2^-40 exactly, products exact
    v = q0.astype(np.float64) * 2.0 ** -40
    q, sigma = oracle.enc(fmt, v)
    assert sigma == 2.0 ** -40
    assert np.array_equal(q.astype(np.int64), q0)
    assert np.array_equal(oracle.dec(fmt, q, sigma), v)


@pytest.mark.parametrize("fmt", ["int32", "int16"])
def test_fixed_point_against_exact_rationals(fmt):
    """Brute force with fractions.Fraction: s = fl(M/a), t = fl(v*s), q = round-half-even(t),
    each fl() realised as the correctly rounded float of the exact rational."""
    M = MAXINT[fmt]
    rng = _rng(16)
    for trial in range(40):
        n = 7
        v = rng.uniform(-1, 1, n) * 10.0 ** rng.integers(-6, 1)
        a = max(abs(float(x)) for x in v)
        s = float(Fraction(M) / Fraction(a))  # Fraction -> float is correctly rounded
        exp_q = []
        for x in v:
            t = float(Fraction(float(x)) * Fraction(s))
            exp_q.append(max(-M, min(M, int(round(Fraction(t))))))  # round(): ties to even
        q, sigma = oracle.enc(fmt, v)
        assert [int(z) for z in q] == exp_q
        assert sigma == float(Fraction(a) / Fraction(M))


def test_fixed_point_ties_round_to_even_and_clamp():
    # a = 32767 * 2^-20 makes s = 2^20 exactly, so v*s is exact and half-integers are real ties
    M = 32767
    a = M * 2.0 ** -20
    ties = np.array([0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 32766.5, -32766.5, 3.25, -3.75]) * 2.0 ** -20
    v = np.concatenate([[a], ties])
    q, sigma = oracle.enc("int16", v)
    assert sigma == 2.0 ** -20
    assert [int(z) for z in q] == [M, 0, 2, 2, 0, -2, -2, 32766, -32766, 3, -4]
    # the most negative code is never produced (symmetric clamp, reading Q6)
    q2, _ = oracle.enc("int16", np.array([-1.0, 1.0, 0.3]))
    assert int(q2.min()) == -M


@pytest.mark.parametrize("fmt", ["int32", "int16"])
def test_fixed_point_zero_vector(fmt):
    q, sigma = oracle.enc(fmt, np.zeros(17))
    assert sigma == 0.0 and not q.any()
    assert not oracle.dec(fmt, q, sigma).any()


def test_format_bytes():
    assert [oracle.format_bytes(f) for f in oracle.FORMATS] == [8, 4, 2, 4, 2]
