"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side harness.

This module holds NONE of the method's arithmetic (no Clebsch-Gordan, no recoupling, no
contraction, no SVD): only label bookkeeping needed to say *which* blocks exist (the fusion
selection rule q_c = q_a + q_s, |j_a - j_s| <= j_c <= j_a + j_s, which is part of the
statement of the input format, Eq. (7)) and seeded random numbers.

Recipes (BASELINE.json configs 2-5):

* ``gaussian_profile(k, chi)``: multiplet degeneracies d_{q,j} on bond k (k sites to its
  left) of the half-filled L=60 chain: weight w(q,j) = exp(-(q-q0)^2/(2*3^2)) exp(-j/1.5) on
  all (q, 2j) with q + 2j = k (mod 2), |q - q0| <= 12, 2j <= min(k, L-k, 30); q0 = +1 for odd
  k, 0 for even k; d = floor(lambda w) with the largest lambda such that
  sum d (2j+1) <= chi (bisection); zero entries dropped; additionally capped by what the
  neighbouring bonds can support (matters only near the chain ends).
* ``table_s2_profile(scale)``: the sector degeneracies the paper prints in Table S2
  (de-garbled as in DESIGN.md reading A-10), scaled.
* ``random_blocks(seed, tag, keys, shapes)``: complex128 iid N(0,1)+iN(0,1) entries from a
  counter-based Philox stream keyed by (seed, tag, block index).
"""
from .profiles import (SITE_LABELS, fuse_labels, gaussian_profile, chain_profiles,  # noqa: F401
                       table_s2_profile, TABLE_S2, reachable_tables, neighbour_profile)
from .blocks import random_blocks, site_block_keys, theta_block_keys, env_block_keys  # noqa: F401
from .chain import (SEED, site_tensor, left_canonical, right_canonical, chain_dims,  # noqa: F401
                    theta_random, canonical_chain)
