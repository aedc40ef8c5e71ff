"""O-U0: closed form for the U=0 Neel quench by single-particle propagation.

TEST INFRASTRUCTURE (see oracle/__init__.py).

At U=0 Eq. (1) is quadratic, so the Neel state Eq. (2) stays a
product of an up- and a down-Slater determinant and

    <n_{i,sigma}>(t) = sum_{j in occ_sigma} |G_ij(t)|^2,     G(t) = exp(-i h t),
    h_ij = -t_h (delta_{i,j+1} + delta_{i+1,j})             (open chain, textbook result),

with the closed-form OBC propagator (i, j = 1..L, k = 1..L)

    G_ij(t) = 2/(L+1) sum_k sin(k pi i/(L+1)) sin(k pi j/(L+1)) exp(+2 i t_h t cos(k pi/(L+1))).

occ_up = sites 0,2,4,... (0-based), occ_dn = sites 1,3,5,...; <n_up n_dn>_i = <n_up><n_dn>
(Wick, the two species are uncorrelated).
"""
import numpy as np


def propagator(L, t_h, t):
    k = np.arange(1, L + 1)
    x = np.arange(1, L + 1)
    S = np.sin(np.outer(x, k) * np.pi / (L + 1))
    phase = np.exp(2j * t_h * t * np.cos(k * np.pi / (L + 1)))
    return (2.0 / (L + 1)) * (S * phase) @ S.T


def observables(L, t_h, t):
    G = propagator(L, t_h, t)
    P = np.abs(G) ** 2
    n_up = P[:, 0::2].sum(axis=1)
    n_dn = P[:, 1::2].sum(axis=1)
    return dict(n_up=n_up, n_dn=n_dn, docc=n_up * n_dn, sz=0.5 * (n_up - n_dn))
