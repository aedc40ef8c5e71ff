"""O-D: dense, non-symmetric two-site TDVP for the Fermi-Hubbard chain (complex128).

TEST INFRASTRUCTURE (see oracle/__init__.py).

Follows the paper's description of the algorithm (S2.2): DMRG-like
sweeps, each local update the Krylov exponential of the effective Hamiltonian of the
two-site block, SVD of the merged two-site tensor, with
the readings A-4 (second-order symmetric sweep, tau = dt/2 each way), A-5 (fixed Krylov
dimension m, full re-orthogonalisation), A-6 (truncation rule) and A-7 (no
renormalisation) of DESIGN.md.

Tensor index conventions: A[i] has shape (chi_l, 4, chi_r); the MPO tensor W has shape
(6, 6, 4, 4) = [w_left, w_right, s_out, s_in]; environments Lenv[i] (left of site i) and
Renv[i] (right of site i-1, i.e. covering sites >= i) have shape (chi_bra, 6, chi_ket).
"""
import numpy as np

from . import fermi


def dense_mpo(t_h, U):
    """Bond-dimension-6 MPO of Eq. (1), identical on every site.

    Rows/cols: 0 = 'nothing yet' (identity), 1..4 = opened hopping term
    (c^dag_up P, c^dag_dn P, c_up P, c_dn P), 5 = 'finished'.
    """
    cu, cd, P = fermi.C_UP, fermi.C_DN, fermi.PAR
    W = np.zeros((6, 6, 4, 4))
    W[0, 0] = fermi.ID4
    W[5, 5] = fermi.ID4
    W[0, 5] = U * fermi.N_UPDN
    W[0, 1] = cu.T @ P
    W[0, 2] = cd.T @ P
    W[0, 3] = cu @ P
    W[0, 4] = cd @ P
    W[1, 5] = -t_h * cu
    W[2, 5] = -t_h * cd
    W[3, 5] = +t_h * cu.T
    W[4, 5] = +t_h * cd.T
    return W


def neel_mps(L):
    """Neel product state Eq. (2): local index 1 (|up>) on even sites, 2 (|dn>) on odd."""
    A = []
    for i in range(L):
        a = np.zeros((1, 4, 1), dtype=complex)
        a[0, 1 if i % 2 == 0 else 2, 0] = 1.0
        A.append(a)
    return A


def update_left(Lenv, A, W):
    """L'[c',w',c] = sum conj(A[a',s',c']) Lenv[a',w,a] W[w,w',s',s] A[a,s,c]."""
    x = np.tensordot(Lenv, A, axes=(2, 0))                  # a' w s c
    x = np.tensordot(x, W, axes=((1, 2), (0, 3)))           # a' c w' s'
    return np.tensordot(A.conj(), x, axes=((0, 1), (0, 3))).transpose(0, 2, 1)  # c' w' c


def update_right(Renv, A, W):
    """R'[c',w,c] = sum conj(A[c',s',b']) W[w,w',s',s] Renv[b',w',b] A[c,s,b]."""
    x = np.tensordot(A, Renv, axes=(2, 2))                  # c s b' w'
    x = np.tensordot(x, W, axes=((1, 3), (3, 1)))           # c b' w s'
    return np.tensordot(A.conj(), x, axes=((1, 2), (3, 1))).transpose(0, 2, 1)  # c' w c


def heff2(Lenv, W, Renv, theta):
    """Two-site H_eff theta = Lenv . W . W . theta . Renv as a reshape + matmul chain."""
    cl, _, _, cr = theta.shape
    clp, crp = Lenv.shape[0], Renv.shape[0]
    t = Lenv.reshape(clp * 6, cl) @ theta.reshape(cl, 16 * cr)       # (a' wl) (s1 s2 b)
    t = t.reshape(clp, 6, 4, 4 * cr).transpose(1, 2, 0, 3).reshape(24, clp * 4 * cr)
    Wm = W.transpose(1, 2, 0, 3).reshape(24, 24)                     # (wm s1') (wl s1)
    t = (Wm @ t).reshape(6, 4, clp, 4, cr)                           # wm s1' a' s2 b
    t = t.transpose(0, 3, 2, 1, 4).reshape(24, clp * 4 * cr)         # (wm s2) (a' s1' b)
    t = (Wm @ t).reshape(6, 4, clp, 4, cr)                           # wr s2' a' s1' b
    t = t.transpose(2, 3, 1, 0, 4).reshape(clp * 16, 6 * cr)         # (a' s1' s2') (wr b)
    Rm = Renv.transpose(1, 2, 0).reshape(6 * cr, crp)                # (wr b) b'
    return (t @ Rm).reshape(clp, 4, 4, crp)


def heff1(Lenv, W, Renv, A):
    """One-site H_eff A = Lenv . W . A . Renv."""
    cl, _, cr = A.shape
    clp, crp = Lenv.shape[0], Renv.shape[0]
    t = Lenv.reshape(clp * 6, cl) @ A.reshape(cl, 4 * cr)
    t = t.reshape(clp, 6, 4, cr).transpose(1, 2, 0, 3).reshape(24, clp * cr)
    Wm = W.transpose(1, 2, 0, 3).reshape(24, 24)
    t = (Wm @ t).reshape(6, 4, clp, cr).transpose(2, 1, 0, 3).reshape(clp * 4, 6 * cr)
    Rm = Renv.transpose(1, 2, 0).reshape(6 * cr, crp)
    return (t @ Rm).reshape(clp, 4, crp)


def krylov_residual_estimate(alpha, beta, b_next, tau):
    """Reading A-15 ("Krylov dimension chosen adaptively (35)").

    After k Lanczos steps y_k(s) = V_k exp(-i s T_k) e_1 solves y' = -i H y up to the residual
    r_k(s) = y_k' + i H y_k = -i b_k [e_k^T exp(-i s T_k) e_1] v_{k+1}   (H V_k = V_k T_k + b_k v_{k+1} e_k^T),
    b_k = b_next the norm of the (k+1)-th unnormalised Lanczos vector.  The error of y_k(tau) is bounded by
    int_0^tau |r_k(s)| ds; the estimate used for stopping is |tau| * |r_k(tau)|.
    """
    k = len(alpha)
    T = np.diag(alpha) + np.diag(beta[:k - 1], 1) + np.diag(beta[:k - 1], -1)
    lam, Q = np.linalg.eigh(T)
    u_last = Q[k - 1, :] @ (np.exp(-1j * tau * lam) * Q[0, :])
    return abs(tau) * b_next * abs(u_last)


def lanczos_exp(apply_h, v, tau, m, breakdown=1e-12, adapt_tol=0.0, stats=None):
    """exp(-i tau H) v by an (at most) m-vector Lanczos process with full re-orthogonalisation (A-5).

    T = tridiag(alpha, beta) is exponentiated through its symmetric eigendecomposition.
    adapt_tol > 0 (A-15): stop after k < m vectors as soon as krylov_residual_estimate <= adapt_tol
    (relative to |v|, the start vector being normalised).  `stats`, if a list, receives k.
    """
    nrm = np.linalg.norm(v)
    if nrm == 0.0:
        if stats is not None:
            stats.append(0)
        return v.copy()
    shape = v.shape
    V = [(v / nrm).ravel()]
    alpha, beta = [], []
    for j in range(m):
        w = apply_h(V[j].reshape(shape)).ravel()
        a = np.vdot(V[j], w).real
        alpha.append(a)
        w = w - a * V[j]
        if j > 0:
            w = w - beta[j - 1] * V[j - 1]
        for u in V:                      # full re-orthogonalisation
            w = w - np.vdot(u, w) * u
        b = np.linalg.norm(w)
        if j == m - 1 or b < breakdown:
            break
        if adapt_tol > 0.0 and krylov_residual_estimate(alpha, beta, b, tau) <= adapt_tol:
            break
        beta.append(b)
        V.append(w / b)
    k = len(alpha)
    if stats is not None:
        stats.append(k)
    T = np.diag(alpha) + np.diag(beta[:k - 1], 1) + np.diag(beta[:k - 1], -1)
    lam, Q = np.linalg.eigh(T)
    c = Q @ (np.exp(-1j * tau * lam) * Q[0, :])
    out = np.zeros_like(V[0])
    for j in range(k):
        out = out + c[j] * V[j]
    return (nrm * out).reshape(shape)


def truncate_rule(svals, mults, chi_max_full, eps_trunc):
    """Reading A-6.  `svals`: list of 1-D descending arrays (one per sector), `mults`: the
    multiplicity 2j+1 of each sector.  Returns the number kept per sector and the
    discarded relative weight.

    Sort all (s, sector, position) by s descending (ties: sector index, then position);
    drop s <= 1e-14 s_max; keep while the cumulative full dimension sum(2j+1) stays
    <= chi_max_full; if eps_trunc >= 0 additionally stop as soon as the remaining tail
    weight sum (2j+1) s^2 / total is <= eps_trunc; keep at least one.
    """
    items = []
    for c, s in enumerate(svals):
        for p, x in enumerate(s):
            items.append((-float(x), c, p))
    items.sort()
    total = sum(mults[c] * x * x for x, c, _ in items)
    smax = -items[0][0] if items else 0.0
    keep = [0] * len(svals)
    dim = 0
    kept_w = 0.0
    nk = 0
    for x, c, p in items:
        s = -x
        if nk >= 1:
            if s <= 1e-14 * smax:
                break
            if dim + mults[c] > chi_max_full:
                break
            if eps_trunc >= 0 and (total - kept_w) <= eps_trunc * total:
                break
        keep[c] += 1
        dim += mults[c]
        kept_w += mults[c] * s * s
        nk += 1
    disc = max(total - kept_w, 0.0) / total if total > 0 else 0.0
    return keep, disc


class DenseTDVP:
    """Two-site TDVP driver (O-D).  One `step(dt)` = L->R half-sweep with tau = dt/2 and
    R->L half-sweep with tau = dt/2 (reading A-4)."""

    def __init__(self, L, t_h, U, krylov_dim=10, chi_max=10 ** 9, eps_trunc=-1.0):
        self.L, self.m = L, krylov_dim
        self.chi_max, self.eps = chi_max, eps_trunc
        self.W = dense_mpo(t_h, U)
        self.A = neel_mps(L)
        e0 = np.zeros((1, 6, 1), dtype=complex)
        e0[0, 0, 0] = 1.0
        e5 = np.zeros((1, 6, 1), dtype=complex)
        e5[0, 5, 0] = 1.0
        self.Lenv = [None] * (L + 1)
        self.Renv = [None] * (L + 1)
        self.Lenv[0] = e0
        self.Renv[L] = e5
        for i in range(L - 1, 0, -1):
            self.Renv[i] = update_right(self.Renv[i + 1], self.A[i], self.W)
        self.disc_weight = 0.0

    def _split(self, theta):
        cl, _, _, cr = theta.shape
        U_, s, Vh = np.linalg.svd(theta.reshape(cl * 4, 4 * cr), full_matrices=False)
        keep, disc = truncate_rule([s], [1], self.chi_max, self.eps)
        k = keep[0]
        self.disc_weight = max(self.disc_weight, disc)
        return U_[:, :k], s[:k], Vh[:k]

    def step(self, dt):
        L, W, m = self.L, self.W, self.m
        tau = dt / 2
        for i in range(L - 1):                                   # left -> right
            theta = np.tensordot(self.A[i], self.A[i + 1], axes=(2, 0))
            Le, Re = self.Lenv[i], self.Renv[i + 2]
            theta = lanczos_exp(lambda x: heff2(Le, W, Re, x), theta, tau, m)
            cl, cr = theta.shape[0], theta.shape[3]
            U_, s, Vh = self._split(theta)
            self.A[i] = U_.reshape(cl, 4, -1)
            self.A[i + 1] = (s[:, None] * Vh).reshape(-1, 4, cr)
            self.Lenv[i + 1] = update_left(Le, self.A[i], W)
            if i < L - 2:
                Ln = self.Lenv[i + 1]
                self.A[i + 1] = lanczos_exp(lambda x: heff1(Ln, W, Re, x), self.A[i + 1], -tau, m)
        for i in range(L - 2, -1, -1):                           # right -> left
            theta = np.tensordot(self.A[i], self.A[i + 1], axes=(2, 0))
            Le, Re = self.Lenv[i], self.Renv[i + 2]
            theta = lanczos_exp(lambda x: heff2(Le, W, Re, x), theta, tau, m)
            cl, cr = theta.shape[0], theta.shape[3]
            U_, s, Vh = self._split(theta)
            self.A[i] = (U_ * s[None, :]).reshape(cl, 4, -1)
            self.A[i + 1] = Vh.reshape(-1, 4, cr)
            self.Renv[i + 1] = update_right(Re, self.A[i + 1], W)
            if i > 0:
                Rn = self.Renv[i + 1]
                self.A[i] = lanczos_exp(lambda x: heff1(Le, W, Rn, x), self.A[i], -tau, m)

    def to_state(self):
        """Contract the MPS to the 4^L state vector (small L only)."""
        psi = self.A[0].reshape(4, -1)
        for i in range(1, self.L):
            a = self.A[i]
            psi = (psi @ a.reshape(a.shape[0], -1)).reshape(-1, a.shape[2])
        return psi.ravel()

    def bond_dims(self):
        return [a.shape[2] for a in self.A[:-1]]

    def observables(self):
        """Measure on the contracted state vector (reading A-12): n_up, n_dn, docc per site."""
        L = self.L
        psi = self.to_state()
        p = np.abs(psi) ** 2
        norm2 = p.sum()
        idx = np.arange(4 ** L)
        n_up = np.zeros(L)
        n_dn = np.zeros(L)
        docc = np.zeros(L)
        x = idx.copy()
        for i in range(L - 1, -1, -1):
            d = x % 4
            x //= 4
            n_up[i] = p[(d == 1) | (d == 3)].sum() / norm2
            n_dn[i] = p[(d == 2) | (d == 3)].sum() / norm2
            docc[i] = p[d == 3].sum() / norm2
        return dict(n_up=n_up, n_dn=n_dn, docc=docc, norm2=norm2)


# ------------------------------------------------------------------ one-site TDVP (NEXT-1)
def heff0(Lenv, Renv, C):
    """Zero-site effective Hamiltonian on the bond matrix C (chi_l x chi_r):
    K C = sum_w L[a',w,a] C[a,b] R[b',w,b]  (backward step of one-site TDVP, refs 8, 9 of the paper)."""
    return np.einsum("xwa,ab,ywb->xy", Lenv, C, Renv, optimize=True)


def tdvp1_step(self, dt):
    """One-site TDVP time step ("switch from the two-site to the one-site TDVP update
    once chi has saturated"): L->R half-sweep (forward one-site step tau = dt/2, QR, backward
    zero-site step) then the mirror R->L half-sweep.  Bond dimensions never change.  Starts and ends
    with the orthogonality centre on site 0, like `step`."""
    L, W, m = self.L, self.W, self.m
    tau = dt / 2
    for i in range(L):                                           # left -> right
        Le, Re = self.Lenv[i], self.Renv[i + 1]
        self.A[i] = lanczos_exp(lambda x: heff1(Le, W, Re, x), self.A[i], tau, m)
        if i < L - 1:
            cl, _, cr = self.A[i].shape
            Q, R = np.linalg.qr(self.A[i].reshape(cl * 4, cr))
            self.A[i] = Q.reshape(cl, 4, -1)
            self.Lenv[i + 1] = update_left(Le, self.A[i], W)
            Ln = self.Lenv[i + 1]
            C = lanczos_exp(lambda x: heff0(Ln, Re, x), R, -tau, m)
            self.A[i + 1] = np.tensordot(C, self.A[i + 1], axes=(1, 0))
    for i in range(L - 1, -1, -1):                               # right -> left
        Le, Re = self.Lenv[i], self.Renv[i + 1]
        self.A[i] = lanczos_exp(lambda x: heff1(Le, W, Re, x), self.A[i], tau, m)
        if i > 0:
            cl, _, cr = self.A[i].shape
            Q, R = np.linalg.qr(self.A[i].reshape(cl, 4 * cr).T)  # A = R^T Q^T
            self.A[i] = Q.T.reshape(-1, 4, cr)
            self.Renv[i] = update_right(Re, self.A[i], W)
            Rn = self.Renv[i]
            C = lanczos_exp(lambda x: heff0(Le, Rn, x), R.T, -tau, m)
            self.A[i - 1] = np.tensordot(self.A[i - 1], C, axes=(2, 0))


DenseTDVP.step1 = tdvp1_step
