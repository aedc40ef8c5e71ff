"""Vector operations of the Lanczos recurrence and the scaled block copy.

TEST INFRASTRUCTURE (see oracle/__init__.py): plain numpy, written from the definitions.

* ``wdot``: the multiplet-weighted inner product F-6, <x,y> = sum_blocks (2j_b+1) sum conj(x) y,
  on a flat vector cut into contiguous blocks.
* ``lanczos_update``: one step of the Lanczos three-term recurrence ("Krylov-based matrix
  exponential") on UNNORMALISED vectors u_j = b_j v_j, b_j = |u_j| (b_0 = 1): with w = H u_j
  and a_raw = <u_j, w>,
      alpha_j = a_raw / b_j^2,   u_{j+1} = (w - alpha_j u_j) / b_j - (b_j / b_{j-1}) u_{j-1},   beta_j = |u_{j+1}|.
  Dividing the standard recurrence beta_j v_{j+1} = H v_j - alpha_j v_j - beta_{j-1} v_{j-1} by nothing but
  substituting v_j = u_j / b_j gives exactly this (b_j = beta_{j-1}); pinned in tests/test_oracle_vecops.py
  against the textbook normalised recurrence on a random Hermitian matrix.
* ``lincomb``: y = sum_j c_j V_j.
* ``copy_blocks``: dst block = scale * src block, optionally transposed (pack / unpack of H8).
"""
import numpy as np


def wdot(blk_len, blk_weight, x, y):
    tot, pos = 0.0 + 0.0j, 0
    for n, w in zip(blk_len, blk_weight):
        tot += w * np.vdot(x[pos:pos + n], y[pos:pos + n])
        pos += n
    return tot


def lanczos_update(blk_len, blk_weight, a_raw, bj2, bjm2, tol, uj, uprev, w):
    """Returns (u_{j+1}, <u_{j+1}, u_{j+1}>).  bj2 <= 0: b_j = 1; uprev None or bjm2 <= 0: no u_{j-1} term; a norm
    below tol counts as zero and makes its reciprocal zero (happy breakdown)."""
    bj = np.sqrt(bj2) if bj2 > 0 else 1.0
    f = 0.0 if (bj < tol or bj == 0.0) else 1.0 / bj
    out = f * w - (a_raw * f * f) * f * uj
    if uprev is not None:
        if bjm2 > 0:
            bm = np.sqrt(bjm2)
            fm = 0.0 if (bm < tol or bm == 0.0) else 1.0 / bm
        else:
            fm = 1.0
        out = out - bj * fm * uprev
    return out, wdot(blk_len, blk_weight, out, out).real


def lincomb(coef, V):
    out = np.zeros_like(V[0])
    for c, v in zip(coef, V):
        out = out + c * v
    return out


def copy_blocks(blocks, src, dst):
    """blocks: iterable of (src_off, dst_off, rows, cols, ld_src, ld_dst, transpose, scale); writes into dst."""
    for so, do, r, c, ls, ld, tr, sc in blocks:
        for i in range(r):
            row = sc * src[so + i * ls: so + i * ls + c]
            if tr:
                dst[do + i: do + i + c * ld: ld] = row
            else:
                dst[do + i * ld: do + i * ld + c] = row
    return dst
