"""O-S driver: two-site TDVP in the symmetric block-sparse format, plus measurements.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Same algorithm as oracle/dense_tdvp.py
(readings A-4..A-7 of DESIGN.md) with every tensor in the reduced
format of oracle/symm.py.  Lanczos runs on the flattened vector scaled by
sqrt(2 j_b + 1) per block, in which the weighted inner product F-6 is Euclidean and the
effective Hamiltonian is Hermitian; the routine itself is dense_tdvp.lanczos_exp.
"""
from math import sqrt

import numpy as np

from . import symm
from .dense_tdvp import lanczos_exp


def flatten(x):
    """dict of blocks -> one vector, each block scaled by sqrt(2 j_last + 1) (F-6)."""
    return np.concatenate([sqrt(k[-1][1] + 1) * v.ravel() for k, v in x.items()])


def unflatten(vec, like):
    out, n = {}, 0
    for k, v in like.items():
        out[k] = (vec[n:n + v.size] / sqrt(k[-1][1] + 1)).reshape(v.shape)
        n += v.size
    return out


def neel_mps(L):
    """Eq. (2) PAPER.md:38 in the reduced format: chi = 1, one block per site (F-2)."""
    A, dims = [], [{(0, 0): 1}]
    q = 0
    for i in range(L):
        s = 0 if i % 2 == 0 else 1
        qn = q + symm.SITE[s][0]
        A.append({((q, 0), s, (qn, 0)): np.ones((1, 1), dtype=complex)})
        dims.append({(qn, 0): 1})
        q = qn
    return A, dims


class SymmTDVP:
    def __init__(self, L, t_h, U, krylov_dim=10, chi_max_full=10 ** 9, eps_trunc=-1.0,
                 A=None, dims=None, krylov_adapt_tol=0.0):
        self.L, self.m = L, krylov_dim
        self.adapt_tol = krylov_adapt_tol     # A-15; 0 = fixed m
        self.krylov_used = []                 # vectors used by every exponential so far
        self.chi_max, self.eps = chi_max_full, eps_trunc
        self.W = [symm.mpo_reduced(i, t_h, U) for i in range(L)]
        if A is None:
            A, dims = neel_mps(L)
        self.A, self.dims = A, dims
        self.Lenv = [None] * (L + 1)
        self.Renv = [None] * (L + 1)
        self.Lenv[0] = symm.boundary_left()
        self.Renv[L] = symm.boundary_right()
        for i in range(L - 1, 0, -1):
            self.Renv[i] = symm.env_update_right(self.Renv[i + 1], self.A[i], self.W[i])
        self.max_discarded = 0.0
        self.svals = [None] * (L + 1)     # kept singular values of the last split per bond

    # ---- local solvers
    def _evolve2(self, i, theta, tau):
        Le, Re = self.Lenv[i], self.Renv[i + 2]
        st1, st2 = symm.heff2_tasks(sorted(Le), sorted(Re), sorted(theta), self.W[i], self.W[i + 1])

        def apply_h(vec):
            th = unflatten(vec, theta)
            Z = symm.run_stage(st1, Le, th)
            out = symm.run_stage(st2, Z, Re, "n", "t")
            for k, v in th.items():
                if k not in out:
                    out[k] = np.zeros_like(v)
            return flatten({k: out[k] for k in theta})

        return unflatten(lanczos_exp(apply_h, flatten(theta), tau, self.m, adapt_tol=self.adapt_tol, stats=self.krylov_used), theta)

    def _evolve1(self, i, Ac, Le, Re, tau):
        st1, st2 = symm.heff1_tasks(sorted(Le), sorted(Re), sorted(Ac), self.W[i])

        def apply_h(vec):
            a = unflatten(vec, Ac)
            X = symm.run_stage(st1, Le, a)
            out = symm.run_stage(st2, X, Re, "n", "t")
            for k, v in a.items():
                if k not in out:
                    out[k] = np.zeros_like(v)
            return flatten({k: out[k] for k in Ac})

        return unflatten(lanczos_exp(apply_h, flatten(Ac), tau, self.m, adapt_tol=self.adapt_tol, stats=self.krylov_used), Ac)

    def _theta(self, i):
        dl, dr = self.dims[i], self.dims[i + 2]
        th = symm.merge(self.A[i], self.A[i + 1])
        full = {}
        for k in symm.theta_keys(dl, dr):
            full[k] = th[k] if k in th else np.zeros((dl[k[0]], dr[k[4]]), dtype=complex)
        return full

    def step(self, dt):
        L = self.L
        tau = dt / 2
        for i in range(L - 1):
            theta = self._evolve2(i, self._theta(i), tau)
            A1, A2, dm, info = symm.svd_split(theta, self.dims[i], self.dims[i + 2],
                                              self.chi_max, self.eps, "right")
            self.max_discarded = max(self.max_discarded, info["discarded"])
            self.A[i], self.A[i + 1], self.dims[i + 1] = A1, A2, dm
            self.svals[i + 1] = {c: info["svals"][c][:k] for c, k in info["keep"].items() if k > 0}
            self.Lenv[i + 1] = symm.env_update_left(self.Lenv[i], A1, self.W[i])
            if i < L - 2:
                self.A[i + 1] = self._evolve1(i + 1, A2, self.Lenv[i + 1], self.Renv[i + 2], -tau)
        for i in range(L - 2, -1, -1):
            theta = self._evolve2(i, self._theta(i), tau)
            A1, A2, dm, info = symm.svd_split(theta, self.dims[i], self.dims[i + 2],
                                              self.chi_max, self.eps, "left")
            self.max_discarded = max(self.max_discarded, info["discarded"])
            self.A[i], self.A[i + 1], self.dims[i + 1] = A1, A2, dm
            self.svals[i + 1] = {c: info["svals"][c][:k] for c, k in info["keep"].items() if k > 0}
            self.Renv[i + 1] = symm.env_update_right(self.Renv[i + 2], A2, self.W[i + 1])
            if i > 0:
                self.A[i] = self._evolve1(i, A1, self.Lenv[i], self.Renv[i + 1], -tau)

    # ---- one-site TDVP (NEXT-1)
    def _evolve0(self, C, Le, Re, tau):
        """Backward zero-site step on the bond matrix C; weight 2j_c+1 per sector block (F-6)."""
        st1, st2 = symm.heff0_tasks(sorted(Le), sorted(Re), sorted(C))
        keys = list(C)

        def flat(x):
            return np.concatenate([sqrt(c[1] + 1) * x[c].ravel() for c in keys])

        def unflat(vec):
            out, n = {}, 0
            for c in keys:
                out[c] = (vec[n:n + C[c].size] / sqrt(c[1] + 1)).reshape(C[c].shape)
                n += C[c].size
            return out

        def apply_h(vec):
            x = unflat(vec)
            X = symm.run_stage(st1, Le, x)
            out = symm.run_stage(st2, X, Re, "n", "t")
            for c in keys:
                if c not in out:
                    out[c] = np.zeros_like(x[c])
            return flat(out)

        return unflat(lanczos_exp(apply_h, flat(C), tau, self.m, adapt_tol=self.adapt_tol, stats=self.krylov_used))

    def step1(self, dt):
        """One-site TDVP step: L->R (forward one-site tau = dt/2, split, backward zero-site) then R->L.
        Starts and ends with the centre on site 0, like `step`; bond dimensions can only shrink (when a
        sector has fewer stacked rows than columns), never grow."""
        L = self.L
        tau = dt / 2
        for i in range(L):
            self.A[i] = self._evolve1(i, self.A[i], self.Lenv[i], self.Renv[i + 1], tau)
            if i < L - 1:
                Q, C, dn = symm.split_site_right_moving(self.A[i], self.dims[i], self.dims[i + 1])
                self.A[i] = Q
                self.Lenv[i + 1] = symm.env_update_left(self.Lenv[i], Q, self.W[i])
                C = self._evolve0(C, self.Lenv[i + 1], self.Renv[i + 1], -tau)
                self.dims[i + 1] = dn
                self.A[i + 1] = symm.absorb_left(C, self.A[i + 1])
        for i in range(L - 1, -1, -1):
            self.A[i] = self._evolve1(i, self.A[i], self.Lenv[i], self.Renv[i + 1], tau)
            if i > 0:
                Q, C, dn = symm.split_site_left_moving(self.A[i], self.dims[i], self.dims[i + 1])
                self.A[i] = Q
                self.Renv[i] = symm.env_update_right(self.Renv[i + 1], Q, self.W[i])
                C = self._evolve0(C, self.Lenv[i], self.Renv[i], -tau)
                self.dims[i] = dn
                self.A[i - 1] = symm.absorb_right(self.A[i - 1], C)

    # ---- measurements (H10; reading A-12)
    def measure_local(self):
        """<1>, <S^z_i>, <P_D,i>/2 per site through left norm-environments
        N_{i+1}[c] = sum_{a,s} A[a,s,c]^dagger N_i[a] A[a,s,c]; valid when all sites to the
        right of the measured one are right-canonical (true after step())."""
        L = self.L
        red_sz = np.array([0.5, -0.5, 0.0])
        red_pd = np.array([0.0, 0.0, 1.0])
        N = {(0, 0): np.ones((1, 1), dtype=complex)}
        n_i, sz_i, docc_i = np.zeros(L), np.zeros(L), np.zeros(L)
        for i in range(L):
            one = sz = pd = 0.0
            Nn = {}
            for (a, s, c), x in self.A[i].items():
                t = x.conj().T @ (N[a] @ x)
                w = (c[1] + 1) * np.trace(t).real
                one += w
                sz += red_sz[s] * w
                pd += red_pd[s] * w
                Nn[c] = Nn.get(c, 0) + t
            n_i[i] = one / one        # <n_i> = 1 identically in a T_tot = 0 state (A-12)
            sz_i[i] = sz / one
            docc_i[i] = 0.5 * pd / one
            N = Nn
        return dict(n=n_i, sz=sz_i, docc=docc_i)

    def measure_global(self):
        """norm^2 and energy from the full left contraction: L_L[(0,0),S,(0,0)] = <psi|psi>,
        L_L[(0,0),F,(0,0)] = <psi|H_sym|psi>."""
        Le = symm.boundary_left()
        for i in range(self.L):
            Le = symm.env_update_left(Le, self.A[i], self.W[i])
        n2 = Le[((0, 0), 0, (0, 0))][0, 0].real
        e = Le[((0, 0), 3, (0, 0))][0, 0].real
        return dict(norm2=n2, energy=e / n2)

    def to_state(self):
        """Dense 4^L state vector through the embedding (small L only)."""
        psi = None
        for i in range(self.L):
            a = symm.embed_site(self.A[i], self.dims[i], self.dims[i + 1], i)
            psi = a.reshape(4, -1) if psi is None else (psi @ a.reshape(a.shape[0], -1)).reshape(-1, a.shape[2])
        return psi.ravel()

    def chi(self):
        return [symm.chi_full(d) for d in self.dims]

    def step_auto(self, dt):
        """Reading A-16 of PAPER.md:53, 250 ("switch from the two-site to the one-site update once the bond
        dimension has saturated"): two-site steps until one of them grows no bond's full dimension, one-site
        steps from then on.  Returns 2 or 1."""
        if getattr(self, "saturated", False):
            self.step1(dt)
            return 1
        before = self.chi()
        self.step(dt)
        self.saturated = all(a <= b for a, b in zip(self.chi(), before))
        return 2
