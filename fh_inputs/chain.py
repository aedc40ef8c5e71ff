"""Seeded synthetic MPS chains shaped like the paper's L=60 quench (BASELINE.json configs 2-5).

Input recipe only: sector profiles per bond, iid complex Gaussian
site tensors from the counter-based generator of ``blocks.random_blocks``, and an optional
gauge fixing by a library QR that makes the synthetic MPS mixed-canonical around a chosen
bond, so that the environments contracted from it are well conditioned (as in a real TDVP
run).  None of the method's contractions (environments, H_eff, Lanczos, SVD split), recoupling
coefficients or task lists live here; both the oracle-side tests and the CUDA-side harness
consume the same numbers from this module and do everything else on their own.

The gauge fixing of the right half needs the metric under which a site tensor counts as
right-canonical, sum_{s,b} w(c,b)^2 A[c,s,b] A[c,s,b]^dagger = 1.  That metric is a convention of the
method (F-6) and is NOT defined here: the caller passes ``weight(c, b)`` -- the oracle-side tests take it
from ``oracle/``, the CUDA-side harness from the library -- and this module only applies it.
"""
from math import sqrt

import numpy as np

from .blocks import random_blocks, site_block_keys, theta_block_keys
from .profiles import chain_profiles, table_s2_profile, neighbour_profile

SEED = 20260604


def site_tensor(seed, site, dims_l, dims_r):
    """{(a, s, c): complex128 (d_a x d_c)} iid N(0,1) + i N(0,1), keyed by (seed, site, block)."""
    keys = site_block_keys(dims_l, dims_r)
    shapes = {k: (dims_l[k[0]], dims_r[k[2]]) for k in keys}
    return random_blocks(seed, 1000 + site, keys, shapes)


def left_canonical(A, dims_l, dims_r):
    """Gauge-fix a site tensor so that sum_{a,s} A[a,s,c]^dagger A[a,s,c] = 1 for every right
    sector c: stack the blocks with that c on top of each other (rows (a, s, alpha) in key
    order) and replace the stack by the Q factor of its QR decomposition.  Right sectors with
    fewer stacked rows than columns are dropped from the bond (returns the new dims_r)."""
    by_c = {}
    for k in sorted(A):
        by_c.setdefault(k[2], []).append(k)
    out, new_r = {}, {}
    for c, ks in by_c.items():
        M = np.concatenate([A[k] for k in ks], axis=0)
        if M.shape[0] < M.shape[1]:
            continue
        Q, _ = np.linalg.qr(M)
        new_r[c] = dims_r[c]
        o = 0
        for k in ks:
            out[k] = np.ascontiguousarray(Q[o:o + dims_l[k[0]]])
            o += dims_l[k[0]]
    return dict(sorted(out.items())), dict(sorted(new_r.items()))


def right_canonical(A, dims_l, dims_r, weight):
    """Gauge-fix so that sum_{s,b} weight(c,b)^2 A[c,s,b] A[c,s,b]^dagger = 1 for every left sector c
    (``weight`` is the caller's metric, see the module docstring): concatenate the weighted blocks of
    that c side by side, take the Q factor of the QR of the conjugate transpose, undo the weights."""
    by_c = {}
    for k in sorted(A):
        by_c.setdefault(k[0], []).append(k)
    out, new_l = {}, {}
    for c, ks in by_c.items():
        wts = [float(weight(c, k[2])) for k in ks]
        M = np.concatenate([w * A[k] for k, w in zip(ks, wts)], axis=1)
        if M.shape[1] < M.shape[0]:
            continue
        Q, _ = np.linalg.qr(M.conj().T)
        Mq = Q.conj().T
        new_l[c] = dims_l[c]
        o = 0
        for k, w in zip(ks, wts):
            out[k] = np.ascontiguousarray(Mq[:, o:o + dims_r[k[2]]] / w)
            o += dims_r[k[2]]
    return dict(sorted(out.items())), dict(sorted(new_l.items()))


def chain_dims(chi, L=60, profile="gaussian", table_s2_scale=(1, 1)):
    """Sector degeneracies on every bond k = 0..L.

    profile "gaussian": BASELINE.json config 2's recipe (``profiles.chain_profiles``).
    profile "table_s2": the paper's Table S2 degeneracies (scaled by num/den) on the even
    bonds within 6 sites of the centre and its fused-and-rescaled neighbour profile on the odd
    ones; further out the Gaussian profile of the same full chi (only the central bonds matter
    for the isolated-apply workloads)."""
    prof = chain_profiles(chi, L)
    if profile == "gaussian":
        return prof
    if profile != "table_s2":
        raise ValueError(profile)
    num, den = table_s2_scale
    even = table_s2_profile(num, den)
    mid = L // 2
    odd_r = neighbour_profile(even, +1)
    odd_l = neighbour_profile(even, -1)
    prof[mid] = even
    prof[mid + 1] = odd_r
    prof[mid - 1] = odd_l
    return prof


def theta_random(seed, site, dims_l, dims_r):
    """Two-site tensor on (site, site+1): iid N(0,1)+iN(0,1) blocks on every fusion-allowed key,
    scaled by 1/sqrt(sum_blocks (2 j_b + 1) rows cols 2) so that its weighted norm is ~1."""
    keys = theta_block_keys(dims_l, dims_r)
    shapes = {k: (dims_l[k[0]], dims_r[k[4]]) for k in keys}
    tot = sum((k[4][1] + 1) * shapes[k][0] * shapes[k][1] * 2.0 for k in keys)
    sc = 1.0 / sqrt(tot) if tot > 0 else 1.0
    blocks = random_blocks(seed, 5000 + site, keys, shapes)
    return {k: v * sc for k, v in blocks.items()}


def canonical_chain(chi, centre, L=60, seed=SEED, profile="gaussian", table_s2_scale=(1, 1),
                    sites=None, dims=None, weight=None):
    """Generator of (site, A_site, dims_l, dims_r) for a random MPS, left-canonical on sites
    < centre and right-canonical on sites > centre + 1 (sites centre, centre+1 are plain random).

    Left sites are yielded in increasing order first, then right sites in decreasing order, so
    that a consumer can stream environment updates without holding the chain (config 5).  QR
    can drop unsupported sectors from a bond; the dims yielded are the final ones, and the
    generator's ``dims`` list (returned through the ``dims`` argument if given) is updated."""
    if weight is None:
        raise ValueError("canonical_chain: the caller must pass weight(c, b), the metric of a right-canonical tensor")
    d = chain_dims(chi, L, profile, table_s2_scale) if dims is None else dims
    left = range(0, centre)
    right = range(L - 1, centre + 1, -1)
    for i in left:
        if sites is not None and i not in sites:
            continue
        A = site_tensor(seed, i, d[i], d[i + 1])
        A, new_r = left_canonical(A, d[i], d[i + 1])
        d[i + 1] = new_r
        yield i, A, d[i], d[i + 1]
    for i in right:
        if sites is not None and i not in sites:
            continue
        A = site_tensor(seed, i, d[i], d[i + 1])
        A, new_l = right_canonical(A, d[i], d[i + 1], weight)
        d[i] = new_l
        yield i, A, d[i], d[i + 1]
    for i in (centre, centre + 1):
        if 0 <= i < L and (sites is None or i in sites):
            yield i, site_tensor(seed, i, d[i], d[i + 1]), d[i], d[i + 1]
