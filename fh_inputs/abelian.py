"""Seeded synthetic inputs for the U(1) x U(1) mode.

Label bookkeeping only (which blocks exist) and seeded random numbers: no contraction, no MPO element, no
coefficient.  A bond label is the pair of additive charges (N_up - N_dn, N - k) on bond k (k sites to its left),
packed into ONE integer so that every key has the same shape as in the U(1) x SU(2) mode:

    label = (q, 0),   q = (N_up - N_dn) + 64 * (N - k)

(the second entry, the doubled spin of the SU(2) mode, is always 0).  Site states s = 0 |0>, 1 |up>, 2 |dn>,
3 |updn> change q by -64, +1, -1, +64; the six MPO bond states I, c+_up P, c+_dn P, c_up P, c_dn P, final carry
0, +65, +63, -65, -63, 0.
"""
from math import comb, exp

from .blocks import random_blocks

SITE_Q = (-64, 1, -1, 64)
MPO_Q = (0, 65, 63, -65, -63, 0)
SEED = 20260604


def unpack(q):
    """q -> (N_up - N_dn, N - k)."""
    dn = (q + 32) // 64
    return q - 64 * dn, dn


def fuse(a, s):
    return (a[0] + SITE_Q[s], 0)


def site_block_keys(dims_l, dims_r):
    return sorted((a, s, fuse(a, s)) for a in dims_l for s in range(4) if fuse(a, s) in dims_r)


def theta_block_keys(dims_l, dims_r):
    keys = []
    for a in dims_l:
        for s1 in range(4):
            c = fuse(a, s1)
            for s2 in range(4):
                b = fuse(c, s2)
                if b in dims_r:
                    keys.append((a, s1, c, s2, b))
    return sorted(keys)


def env_block_keys(dims_bra, dims_ket):
    return sorted((xp, w, x) for xp in dims_bra for w in range(6) for x in dims_ket if xp[0] == x[0] + MPO_Q[w])


def _capacity(k, q1, dn):
    """Number of product states of k sites with N_up - N_dn = q1 and N = k + dn."""
    n = k + dn
    if (n + q1) % 2 or n < 0:
        return 0
    nu, nd = (n + q1) // 2, (n - q1) // 2
    if nu < 0 or nd < 0 or nu > k or nd > k:
        return 0
    return comb(k, nu) * comb(k, nd)


def profile(k, chi, L=60):
    """Degeneracies on bond k of the half-filled chain: weight exp(-(q1 - q0)^2 / 18) exp(-dn^2 / 18) on all
    (q1, dn) with |q1 - q0| <= 9, |dn| <= 9 that k sites can carry and L - k sites can complete to (0, 0);
    q0 = +1 (odd k) or 0 (even k) is the Neel prefix's N_up - N_dn; d = floor(lambda w) with the largest lambda
    such that sum d <= chi, capped by the number of states on either side; zeros dropped."""
    q0 = k % 2
    cand = []
    for q1 in range(q0 - 9, q0 + 10):
        for dn in range(-9, 10):
            cap = min(_capacity(k, q1, dn), _capacity(L - k, -q1, -dn))
            if cap > 0:
                cand.append((q1 + 64 * dn, exp(-(q1 - q0) ** 2 / 18.0 - dn ** 2 / 18.0), cap))
    lo, hi = 0.0, 4.0 * chi

    def dims(lam):
        return {(q, 0): min(int(lam * w), cap) for q, w, cap in cand if min(int(lam * w), cap) > 0}

    for _ in range(60):
        mid = 0.5 * (lo + hi)
        if sum(dims(mid).values()) <= chi:
            lo = mid
        else:
            hi = mid
    return dict(sorted(dims(lo).items()))


def chain_dims(chi, L=60):
    return [profile(k, chi, L) for k in range(L + 1)]


def site_tensor(seed, site, dims_l, dims_r):
    keys = site_block_keys(dims_l, dims_r)
    return random_blocks(seed, 3000 + site, keys, {k: (dims_l[k[0]], dims_r[k[2]]) for k in keys})


def theta_random(seed, site, dims_l, dims_r):
    keys = theta_block_keys(dims_l, dims_r)
    shapes = {k: (dims_l[k[0]], dims_r[k[4]]) for k in keys}
    tot = sum(2.0 * shapes[k][0] * shapes[k][1] for k in keys)
    blocks = random_blocks(seed, 7000 + site, keys, shapes)
    return {k: v / tot ** 0.5 for k, v in blocks.items()}
