"""Pins of oracle/splitprec.py (reading A-18) against what the
number format and the mathematics fix: hand-worked TF32 roundings, the bit pattern of a TF32 value, the split
remainder bound, exactness on inputs that need no split, the error bound against the exact product, and
brute-force evaluation of the three-term formula with Python fractions."""
from fractions import Fraction

import numpy as np

from oracle import splitprec as sp


def test_tf32_round_hand_worked_values():
    # TF32 keeps 10 explicit mantissa bits: spacing 2^-10 in [1, 2)
    cases = {
        1.0: 1.0,
        1.0 + 2.0 ** -10: 1.0 + 2.0 ** -10,              # representable
        1.0 + 2.0 ** -12: 1.0,                           # below half a unit: down
        1.0 + 2.0 ** -11: 1.0 + 2.0 ** -10,              # exactly half: ties AWAY from zero
        -(1.0 + 2.0 ** -11): -(1.0 + 2.0 ** -10),
        1.0 + 2.0 ** -11 + 2.0 ** -20: 1.0 + 2.0 ** -10,
        1.0 + 3 * 2.0 ** -11: 1.0 + 2 * 2.0 ** -10,      # tie between 1 and 2 units: away
        3.0 + 2.0 ** -10: 3.0 + 2.0 ** -9,               # spacing 2^-9 in [2, 4): tie, away
        0.0: 0.0,
        2.0 - 2.0 ** -12: 2.0,                           # rounds up into the next binade
        2.0 ** -100 * (1 + 2.0 ** -11): 2.0 ** -100 * (1 + 2.0 ** -10),
    }
    for x, want in cases.items():
        got = float(sp.tf32_round(np.float32(x)).reshape(-1)[0])
        assert got == want, (x, got, want)
    f = np.random.default_rng(1).standard_normal(4096).astype(np.float32)
    r = sp.tf32_round(f)
    assert np.all(r.view(np.uint32) & np.uint32(0x1FFF) == 0)          # 13 low mantissa bits are zero
    # round11 (on doubles) is the same rounding: equal on every float32 number, hand-worked values included
    assert np.array_equal(sp.round11(f.astype(np.float64)), r.astype(np.float64))
    for x, want in cases.items():
        assert float(sp.round11(np.array([x]))[0]) == want, x
    assert float(sp.round11(np.array([1.0 + 2.0 ** -11 - 2.0 ** -40]))[0]) == 1.0          # just below the tie: down
    assert float(sp.round11(np.array([2.0 ** -130]))[0]) == 0.0                          # below float32's normal range


def test_split_remainder_bound_and_tf32_valued_parts():
    rng = np.random.default_rng(2)
    x = np.concatenate([rng.standard_normal(20000) * 10.0 ** rng.integers(-6, 7, 20000), [0.0, 1.0, -1.0, 1 / 3, np.pi, 1e-30]])
    hi, lo = sp.split_tf32(x)
    for part in (hi, lo):
        assert part.dtype == np.float32 and np.all(part.view(np.uint32) & np.uint32(0x1FFF) == 0)
    r = x - hi.astype(np.float64) - lo.astype(np.float64)
    assert np.all(np.abs(r) <= 2.0 ** -22 * np.abs(x))
    assert np.all(np.abs(x - hi) <= 2.0 ** -11 * np.abs(x))
    assert np.abs(r).max() > 2.0 ** -26 * np.abs(x).max() * 1e-3         # the remainder is really there (22, not 53 bits)


def test_exact_when_no_split_is_needed():
    """Small integers are TF32 numbers: hi = x, lo = 0, and the three-term product is the exact product."""
    rng = np.random.default_rng(3)
    A = rng.integers(-30, 31, (9, 14)) + 1j * rng.integers(-30, 31, (9, 14))
    B = rng.integers(-30, 31, (14, 5)) + 1j * rng.integers(-30, 31, (14, 5))
    A2 = rng.integers(-30, 31, (9, 3)) + 1j * rng.integers(-30, 31, (9, 3))
    B2 = rng.integers(-30, 31, (3, 5)) + 1j * rng.integers(-30, 31, (3, 5))
    C = sp.zgemm_split([(2.0, A, B), (-0.5, A2, B2)], 9, 5)
    assert np.array_equal(C, 2.0 * (A @ B) - 0.5 * (A2 @ B2))
    hi, lo = sp.split_tf32(np.array([5.0, -1024.0, 0.375]))
    assert np.array_equal(hi, [5.0, -1024.0, 0.375]) and not lo.any()


def test_three_term_formula_brute_force_with_fractions():
    """One element, every term written out with exact rational arithmetic: catches a dropped or doubled term, a
    wrong sign in the complex product, alpha applied on the wrong side of the split."""
    rng = np.random.default_rng(4)
    K = 6
    a = rng.standard_normal(K) + 1j * rng.standard_normal(K)
    b = rng.standard_normal(K) + 1j * rng.standard_normal(K)
    alpha = -1.7
    got = sp.zgemm_split([(alpha, a.reshape(1, K), b.reshape(K, 1))], 1, 1)[0, 0]

    def parts(v):
        h, l = sp.split_tf32(np.array([v]))
        return Fraction(float(h[0])), Fraction(float(l[0]))

    re = im = Fraction(0)
    for k in range(K):
        ar, ai = parts(alpha * a[k].real), parts(alpha * a[k].imag)
        br, bi = parts(b[k].real), parts(b[k].imag)

        def three(p, q):
            return p[0] * q[0] + p[0] * q[1] + p[1] * q[0]

        re += three(ar, br) - three(ai, bi)
        im += three(ar, bi) + three(ai, br)
    assert abs(got.real - float(re)) <= 4e-16 * abs(float(re)) + 1e-300
    assert abs(got.imag - float(im)) <= 4e-16 * abs(float(im)) + 1e-300


def test_split_error_bound_against_exact_product():
    rng = np.random.default_rng(5)
    segs = []
    for K in (37, 128, 5):
        segs.append((float(rng.uniform(-2, 2)), rng.standard_normal((23, K)) + 1j * rng.standard_normal((23, K)),
                     rng.standard_normal((K, 17)) + 1j * rng.standard_normal((K, 17))))
    exact = sum(al * (A @ B) for al, A, B in segs)
    C = sp.zgemm_split(segs, 23, 17)
    acc, split = sp.split_bounds(segs, 23, 17)
    err = np.abs(C - exact)
    assert np.all(err <= split)
    assert err.max() > 1e-3 * split.max()                # and the bound is not vacuous: single-precision class error
    assert np.linalg.norm(C - exact) / np.linalg.norm(exact) < 2e-6
    assert np.all(acc > 0) and acc.shape == (23, 17)
    # two-term variant (lo_a hi_b dropped) breaks the bound: the third term is needed
    A, B = segs[1][1], segs[1][2]
    ah, al_ = sp.split_tf32(A.real)
    bh, bl = sp.split_tf32(B.real)
    two = ah.astype(np.float64) @ bh + ah.astype(np.float64) @ bl
    three = two + al_.astype(np.float64) @ bh
    S = np.abs(A.real) @ np.abs(B.real)
    assert np.all(np.abs(three - A.real @ B.real) <= 3.1 * 2.0 ** -22 * S)
    assert np.any(np.abs(two - A.real @ B.real) > 3.1 * 2.0 ** -22 * S)
