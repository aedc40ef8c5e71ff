"""Synthetic sector-degeneracy profiles (label bookkeeping only, no method arithmetic)."""
from math import exp, floor

# (q, 2j) of the three site multiplets: |up>, |dn>, {|0>, |updn>}
SITE_LABELS = ((1, 0), (-1, 0), (0, 1))


def fuse_labels(a, s):
    """Labels c reachable from bond label a and site multiplet s (selection rule only)."""
    qs, ts = SITE_LABELS[s]
    return [(a[0] + qs, tc) for tc in range(abs(a[1] - ts), a[1] + ts + 1, 2)]


def reachable_tables(L):
    """Per bond k = 0..L: the set of labels reachable from (0,0) on the left AND from which
    (0,0) is reachable on the right (half filling, total sector q = 0, j = 0)."""
    fwd = [{(0, 0)}]
    for _ in range(L):
        nxt = set()
        for a in fwd[-1]:
            for s in range(3):
                nxt.update(fuse_labels(a, s))
        fwd.append(nxt)
    bwd = [None] * (L + 1)
    bwd[L] = {(0, 0)}
    for k in range(L - 1, -1, -1):
        cur = set()
        for a in fwd[k]:
            for s in range(3):
                if any(c in bwd[k + 1] for c in fuse_labels(a, s)):
                    cur.add(a)
        bwd[k] = cur
    return [sorted(fwd[k] & bwd[k]) for k in range(L + 1)]


def _weights(k, L):
    q0 = 1 if k % 2 else 0
    out = {}
    lim = min(k, L - k)
    for q in range(q0 - 12, q0 + 13):
        for tj in range(0, min(lim, 30) + 1):
            if (q + tj - k) % 2:
                continue
            if abs(q) + tj > lim:
                continue
            out[(q, tj)] = exp(-((q - q0) ** 2) / (2.0 * 3.0 ** 2)) * exp(-(tj / 2.0) / 1.5)
    return out


def _fit(weights, chi, caps=None):
    """d = floor(lambda w) (capped) with the largest lambda such that sum d (2j+1) <= chi."""
    def dims(lam):
        d = {}
        for key, w in weights.items():
            v = int(floor(lam * w))
            if caps is not None:
                v = min(v, caps.get(key, 0))
            if v > 0:
                d[key] = v
        return d

    def full(d):
        return sum(v * (key[1] + 1) for key, v in d.items())

    lo, hi = 0.0, 1.0
    while full(dims(hi)) <= chi and hi < 1e15:
        hi *= 2.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if full(dims(mid)) <= chi:
            lo = mid
        else:
            hi = mid
    d = dims(lo)
    if not d:                      # chi too small for any floor() >= 1: keep the heaviest label
        key = max(sorted(weights), key=lambda t: weights[t])
        d = {key: 1}
    return dict(sorted(d.items()))


def gaussian_profile(k, chi, L=60):
    """BASELINE.json config 2 block profile on bond k (no neighbour caps)."""
    if k == 0 or k == L:
        return {(0, 0): 1}
    return _fit(_weights(k, L), chi)


def chain_profiles(chi, L=60):
    """Profiles on every bond k = 0..L, capped so that each bond can be supported by its
    neighbours: d_c <= sum over parents (a, s) of d_a and d_a <= sum over children (s, c)
    of d_c (only binding within a few sites of the chain ends)."""
    prof = [gaussian_profile(k, chi, L) for k in range(L + 1)]
    for k in range(1, L + 1):
        caps = {}
        for a, d in prof[k - 1].items():
            for s in range(3):
                for c in fuse_labels(a, s):
                    caps[c] = caps.get(c, 0) + d
        prof[k] = {c: min(d, caps.get(c, 0)) for c, d in prof[k].items() if caps.get(c, 0) > 0}
    for k in range(L - 1, -1, -1):
        new = {}
        for a, d in prof[k].items():
            cap = 0
            for s in range(3):
                for c in fuse_labels(a, s):
                    cap += prof[k + 1].get(c, 0)
            if cap > 0:
                new[a] = min(d, cap)
        prof[k] = new
    return [dict(sorted(p.items())) for p in prof]


# Table S2 of the paper: sector degeneracies at t=6, site 30,
# chi_SU(2) = 12288.  Keys (n, 2j); reading A-10 of DESIGN.md for the garbled j column.
TABLE_S2 = {
    (-6, 0): 8, (-6, 2): 1,
    (-5, 1): 86, (-5, 3): 13,
    (-4, 0): 241, (-4, 2): 233, (-4, 4): 19,
    (-3, 1): 799, (-3, 3): 307, (-3, 5): 10,
    (-2, 0): 920, (-2, 2): 1135, (-2, 4): 213,
    (-1, 1): 1735, (-1, 3): 837, (-1, 5): 80,
    (0, 0): 1097, (0, 2): 1387, (0, 4): 287, (0, 6): 8,
    (1, 1): 1157, (1, 3): 494, (1, 5): 42,
    (2, 0): 382, (2, 2): 421, (2, 4): 67,
    (3, 1): 178, (3, 3): 58,
    (4, 0): 35, (4, 2): 29,
    (5, 1): 8,
    (6, 0): 1,
}


def table_s2_profile(num=1, den=1):
    """Table S2 degeneracies scaled by num/den (rounded down, zeros dropped); even bond."""
    out = {}
    for key, d in TABLE_S2.items():
        v = (d * num) // den
        if v > 0:
            out[key] = v
    return dict(sorted(out.items()))


def neighbour_profile(dims, direction=+1):
    """A profile for the bond one site to the right (direction=+1) or left (-1) of `dims`:
    candidate labels by fusion with the site multiplets, degeneracy proportional to the
    summed parent degeneracies, rescaled (largest remainder) to the same sum d."""
    cand = {}
    for a, d in dims.items():
        for s in range(3):
            for c in fuse_labels(a, s):
                if direction < 0:
                    c = (2 * a[0] - c[0], c[1])      # remove instead of add the site charge
                cand[c] = cand.get(c, 0) + d
    target = sum(dims.values())
    tot = sum(cand.values())
    base = {c: (w * target) // tot for c, w in cand.items()}
    rem = sorted(cand, key=lambda c: (-((cand[c] * target) % tot), c))
    short = target - sum(base.values())
    for c in rem[:short]:
        base[c] += 1
    return dict(sorted((c, d) for c, d in base.items() if d > 0))
