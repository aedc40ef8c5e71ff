"""SU(2) algebra for the oracle: Clebsch-Gordan coefficients and recoupling sums.

TEST INFRASTRUCTURE (see oracle/__init__.py).  All spins are passed DOUBLED
(tj = 2j, tm = 2m) so that everything is integer arithmetic.

The paper defers the symmetric-tensor conventions to its refs 18-24
(PAPER.md:41, 47, 131-139); the conventions used here are the readings F-1,
F-4, F-5 of DESIGN.md.  The recoupling coefficients are *defined* here as the
explicit contraction of six Clebsch-Gordan coefficients that follows from the
tensor structures F-4; no closed form (6j/9j) is used in this file, so that the
closed forms used by the CUDA library's host layer are checked against an
independent definition.
"""
from fractions import Fraction
from functools import lru_cache
from math import factorial, isqrt, sqrt


def _sqrt_fraction(fr):
    """sqrt of a non-negative Fraction, exact when num/den are perfect squares."""
    n, d = fr.numerator, fr.denominator
    rn, rd = isqrt(n), isqrt(d)
    if rn * rn == n and rd * rd == d:
        return rn / rd
    return sqrt(n) / sqrt(d)


@lru_cache(maxsize=None)
def cg(tj1, tm1, tj2, tm2, tJ, tM):
    """Clebsch-Gordan <j1 m1; j2 m2 | J M>, Condon-Shortley phases (reading F-1).

    Racah's closed formula, evaluated in exact rational arithmetic with a single
    square root at the end.
    """
    if tm1 + tm2 != tM:
        return 0.0
    if tJ < abs(tj1 - tj2) or tJ > tj1 + tj2 or (tj1 + tj2 + tJ) % 2:
        return 0.0
    if abs(tm1) > tj1 or abs(tm2) > tj2 or abs(tM) > tJ:
        return 0.0
    if (tj1 + tm1) % 2 or (tj2 + tm2) % 2 or (tJ + tM) % 2:
        return 0.0
    f = factorial
    # all of the following are integers
    a = (tj1 + tj2 - tJ) // 2
    b = (tj1 - tj2 + tJ) // 2
    c = (-tj1 + tj2 + tJ) // 2
    d = (tj1 + tj2 + tJ) // 2 + 1
    pref2 = Fraction((tJ + 1) * f(a) * f(b) * f(c), f(d))
    pref2 *= (f((tJ + tM) // 2) * f((tJ - tM) // 2)
              * f((tj1 - tm1) // 2) * f((tj1 + tm1) // 2)
              * f((tj2 - tm2) // 2) * f((tj2 + tm2) // 2))
    s = Fraction(0)
    j1m = (tj1 - tm1) // 2      # j1 - m1
    j2p = (tj2 + tm2) // 2      # j2 + m2
    e = (tJ - tj2 + tm1) // 2   # J - j2 + m1
    g = (tJ - tj1 - tm2) // 2   # J - j1 - m2
    for k in range(0, a + 1):
        t = [k, a - k, j1m - k, j2p - k, e + k, g + k]
        if min(t) < 0:
            continue
        den = 1
        for x in t:
            den *= f(x)
        s += Fraction((-1) ** k, den)
    if s == 0:
        return 0.0
    val = _sqrt_fraction(pref2 * s * s)
    return val if s > 0 else -val


def _ms(tj):
    return range(-tj, tj + 1, 2)


@lru_cache(maxsize=None)
def coef_left(ta, ts, tc, tk, tr, tkp, tap, tsp, tcp):
    """coefL(a,s,c; k,r,k'; a',s',c')  (reading F-5, definition by CG contraction).

    It is the number x such that, with the dense structures of F-4,

        sum_{m,m',sig,sig',mu,rho}
            C(a' m', s' sig' | c' n') C(a m, k mu | a' m') C(s sig, r rho | s' sig')
            C(k mu, r rho | k' mu') C(a m, s sig | c n)        =  x * C(c n, k' mu' | c' n')

    i.e. (left environment L[a',k,a]) x (MPO element of rank r taking k -> k') x
    (ket A[a,s,c]) x (bra A[a',s',c']) has the CG structure of L'[c',k',c].
    Computed as the full six-CG sum at fixed n' = c' (using
    sum_{n,mu'} C(c n,k' mu'|c' n')^2 = 1).
    """
    npr = tcp  # fix n' = +c'
    tot = 0.0
    for mp in _ms(tap):
        sigp = npr - mp
        if abs(sigp) > tsp:
            continue
        c1 = cg(tap, mp, tsp, sigp, tcp, npr)
        if c1 == 0.0:
            continue
        for m in _ms(ta):
            mu = mp - m
            if abs(mu) > tk:
                continue
            c2 = cg(ta, m, tk, mu, tap, mp)
            if c2 == 0.0:
                continue
            for sig in _ms(ts):
                rho = sigp - sig
                if abs(rho) > tr:
                    continue
                c3 = cg(ts, sig, tr, rho, tsp, sigp)
                if c3 == 0.0:
                    continue
                mup = mu + rho
                if abs(mup) > tkp:
                    continue
                c4 = cg(tk, mu, tr, rho, tkp, mup)
                n = m + sig
                if abs(n) > tc:
                    continue
                c5 = cg(ta, m, ts, sig, tc, n)
                c6 = cg(tc, n, tkp, mup, tcp, npr)
                tot += c1 * c2 * c3 * c4 * c5 * c6
    return tot


@lru_cache(maxsize=None)
def coef_right(tc, ts, tb, tk, tr, tkp, tcp, tsp, tbp):
    """coefR(c,s,b; k,r,k'; c',s',b')  (reading F-5, definition by CG contraction).

    The number x such that

        sum  C(c' n', s' sig' | b' m') C(s sig, r rho | s' sig') C(k mu, r rho | k' mu')
             C(b m, k' mu' | b' m') C(c n, s sig | b m)            =  x * C(c n, k mu | c' n')

    i.e. (right environment R[b',k',b]) x (MPO element k -> k') x (ket A[c,s,b]) x
    (bra A[c',s',b']) has the CG structure of R'[c',k,c].  Full six-CG sum at
    fixed n' = c'.
    """
    npr = tcp
    tot = 0.0
    for sigp in _ms(tsp):
        mp = npr + sigp
        if abs(mp) > tbp:
            continue
        c1 = cg(tcp, npr, tsp, sigp, tbp, mp)
        if c1 == 0.0:
            continue
        for sig in _ms(ts):
            rho = sigp - sig
            if abs(rho) > tr:
                continue
            c2 = cg(ts, sig, tr, rho, tsp, sigp)
            if c2 == 0.0:
                continue
            for mu in _ms(tk):
                mup = mu + rho
                if abs(mup) > tkp:
                    continue
                c3 = cg(tk, mu, tr, rho, tkp, mup)
                if c3 == 0.0:
                    continue
                m = mp - mup
                if abs(m) > tb:
                    continue
                c4 = cg(tb, m, tkp, mup, tbp, mp)
                n = m - sig
                if abs(n) > tc:
                    continue
                c5 = cg(tc, n, ts, sig, tb, m)
                c6 = cg(tc, n, tk, mu, tcp, npr)
                tot += c1 * c2 * c3 * c4 * c5 * c6
    return tot
