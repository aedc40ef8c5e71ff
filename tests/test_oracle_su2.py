"""Pins for oracle/su2.py: CG against sympy + orthogonality; the six-CG recoupling sums
against the closed forms of DESIGN.md reading F-5 evaluated with sympy's Wigner 9j."""
import random
from math import sqrt

import pytest
from sympy import Rational
from sympy.physics.quantum.cg import CG
from sympy.physics.wigner import wigner_9j

from oracle import su2


def test_cg_matches_sympy():
    rnd = random.Random(7)
    n = 0
    while n < 150:
        tj1, tj2 = rnd.randint(0, 7), rnd.randint(0, 4)
        tJ = rnd.choice(range(abs(tj1 - tj2), tj1 + tj2 + 1, 2))
        tm1 = rnd.choice(range(-tj1, tj1 + 1, 2))
        tm2 = rnd.choice(range(-tj2, tj2 + 1, 2))
        tM = tm1 + tm2
        if abs(tM) > tJ:
            continue
        ref = float(CG(Rational(tj1, 2), Rational(tm1, 2), Rational(tj2, 2), Rational(tm2, 2),
                       Rational(tJ, 2), Rational(tM, 2)).doit())
        assert abs(su2.cg(tj1, tm1, tj2, tm2, tJ, tM) - ref) < 1e-14
        n += 1


def test_cg_orthogonality_and_selection():
    for tj1 in range(0, 6):
        for tj2 in range(0, 3):
            for tJ in range(abs(tj1 - tj2), tj1 + tj2 + 1, 2):
                for tJ2 in range(abs(tj1 - tj2), tj1 + tj2 + 1, 2):
                    for tM in range(-min(tJ, tJ2), min(tJ, tJ2) + 1, 2):
                        s = sum(su2.cg(tj1, m1, tj2, tM - m1, tJ, tM) * su2.cg(tj1, m1, tj2, tM - m1, tJ2, tM)
                                for m1 in range(-tj1, tj1 + 1, 2))
                        assert abs(s - (1.0 if tJ == tJ2 else 0.0)) < 1e-14
    assert su2.cg(2, 0, 2, 0, 2, 0) == 0.0          # <1 0;1 0|1 0> = 0
    assert su2.cg(1, 1, 1, 1, 0, 2) == 0.0
    assert abs(su2.cg(1, 1, 1, -1, 0, 0) - 1 / sqrt(2)) < 1e-15
    assert abs(su2.cg(1, -1, 1, 1, 0, 0) + 1 / sqrt(2)) < 1e-15


def _nine_j(a, s, c, k, r, kp, ap, sp, cp):
    h = lambda t: Rational(t, 2)
    return float(wigner_9j(h(a), h(s), h(c), h(k), h(r), h(kp), h(ap), h(sp), h(cp), prec=64))


def _tuples(seed, count):
    """Random label tuples of the kind the hot path meets: s,s' in {0,1/2}, k,r,k' in {0,1/2}."""
    rnd = random.Random(seed)
    out = []
    while len(out) < count:
        ta = rnd.randint(0, 7)
        ts, tsp = rnd.choice([0, 1]), rnd.choice([0, 1])
        tk, tr = rnd.choice([0, 1]), rnd.choice([0, 1])
        tkp = rnd.choice(range(abs(tk - tr), tk + tr + 1, 2))
        if abs(ts - tr) > tsp or tsp > ts + tr or (ts + tr + tsp) % 2:
            continue
        tc = rnd.choice(range(abs(ta - ts), ta + ts + 1, 2))
        tap = rnd.choice(range(abs(ta - tk), ta + tk + 1, 2))
        tcp = rnd.choice(range(abs(tap - tsp), tap + tsp + 1, 2))
        if abs(tc - tkp) > tcp or tcp > tc + tkp or (tc + tkp + tcp) % 2:
            continue
        out.append((ta, ts, tc, tk, tr, tkp, tap, tsp, tcp))
    return out


def test_coef_left_closed_form():
    """coefL = sqrt((2c+1)(2k'+1)(2a'+1)(2s'+1)) {a s c; k r k'; a' s' c'}."""
    nz = 0
    for t in _tuples(11, 120):
        ta, ts, tc, tk, tr, tkp, tap, tsp, tcp = t
        ref = sqrt((tc + 1) * (tkp + 1) * (tap + 1) * (tsp + 1)) * _nine_j(*t)
        val = su2.coef_left(*t)
        assert abs(val - ref) < 1e-13, t
        nz += abs(ref) > 1e-6
    assert nz > 40


def test_coef_right_closed_form():
    """coefR = (2b'+1)/(2c'+1) sqrt((2b+1)(2k'+1)(2c'+1)(2s'+1)) {c s b; k r k'; c' s' b'}."""
    nz = 0
    for t in _tuples(13, 120):
        tc, ts, tb, tk, tr, tkp, tcp, tsp, tbp = t
        # for coefR the MPO multiplets couple on the other side: need triangle(b, k', b')
        if abs(tb - tkp) > tbp or tbp > tb + tkp or abs(tc - tk) > tcp or tcp > tc + tk \
                or (tc + tk + tcp) % 2:
            continue
        ref = (tbp + 1) / (tcp + 1) * sqrt((tb + 1) * (tkp + 1) * (tcp + 1) * (tsp + 1)) * _nine_j(*t)
        val = su2.coef_right(*t)
        assert abs(val - ref) < 1e-13, t
        nz += abs(ref) > 1e-6
    assert nz > 10


def test_trivial_mpo_coefficient_is_one():
    """With k = r = k' = 0 (identity MPO): coefL = 1 and coefR = (2b+1)/(2c+1) -- the weights
    of the left- and right-canonical conditions of reading F-6."""
    for ta in range(0, 6):
        for ts in (0, 1):
            for tc in range(abs(ta - ts), ta + ts + 1, 2):
                assert abs(su2.coef_left(ta, ts, tc, 0, 0, 0, ta, ts, tc) - 1.0) < 1e-14
                assert abs(su2.coef_right(ta, ts, tc, 0, 0, 0, ta, ts, tc) - (tc + 1) / (ta + 1)) < 1e-14
