"""Jordan-Wigner operators, the Fermi-Hubbard Hamiltonian and exact diagonalisation (O-ED).

TEST INFRASTRUCTURE (see oracle/__init__.py).

Cites: Hamiltonian Eq. (1); Neel state Eq. (2) PAPER.md:36-41;
pseudospin generators Eqs. (4)-(6) PAPER.md:192-206.

Conventions (readings F-2, A-3): local basis |0>, |up>, |dn>, |updn> with
|updn> := c^dag_up c^dag_dn |0>; fermionic mode order 0up,0dn,1up,1dn,...;
sites are 0-based and the sublattice sign is eps_i = (-1)^i.
"""
import numpy as np
import scipy.sparse as sp

# ---- single-site 4x4 matrices (index 0:|0>, 1:|up>, 2:|dn>, 3:|updn>) ----------
C_UP = np.zeros((4, 4))
C_UP[0, 1] = 1.0            # c_up |up>   = |0>
C_UP[2, 3] = 1.0            # c_up |updn> = |dn>
C_DN = np.zeros((4, 4))
C_DN[0, 2] = 1.0            # c_dn |dn>   = |0>
C_DN[1, 3] = -1.0           # c_dn c^dag_up c^dag_dn|0> = -|up>
PAR = np.diag([1.0, -1.0, -1.0, 1.0])   # (-1)^{n_i}
ID4 = np.eye(4)
N_UP = C_UP.T @ C_UP
N_DN = C_DN.T @ C_DN
N_UPDN = N_UP @ N_DN
P_D = np.diag([1.0, 0.0, 0.0, 1.0])     # projector on empty + doubly occupied = (n-1)^2
SZ = 0.5 * (N_UP - N_DN)


def site_op(L, i, op, string=None):
    """Sparse 4^L matrix of a one-site operator at site i; `string` (e.g. PAR) on sites < i."""
    mats = []
    for k in range(L):
        if k < i:
            mats.append(sp.identity(4, format="csr") if string is None else sp.csr_matrix(string))
        elif k == i:
            mats.append(sp.csr_matrix(op))
        else:
            mats.append(sp.identity(4, format="csr"))
    out = mats[0]
    for m in mats[1:]:
        out = sp.kron(out, m, format="csr")
    return out


def annihilators(L):
    """Full-chain c_{i,up}, c_{i,dn} (lists of sparse matrices) with Jordan-Wigner strings."""
    cup = [site_op(L, i, C_UP, PAR) for i in range(L)]
    cdn = [site_op(L, i, C_DN, PAR) for i in range(L)]
    return cup, cdn


def hamiltonian(L, t_h, U, symmetric=False):
    """Eq. (1) on an open chain as a sparse 4^L matrix.

    symmetric=True returns H_sym = hopping + (U/2) sum_i P_D,i  (reading A-2), which
    commutes with the pseudospin generators and equals Eq. (1) on N = L states.
    """
    cup, cdn = annihilators(L)
    dim = 4 ** L
    H = sp.csr_matrix((dim, dim))
    for i in range(L - 1):
        for c in (cup, cdn):
            hop = c[i].T @ c[i + 1]
            H = H - t_h * (hop + hop.T)
    for i in range(L):
        if symmetric:
            H = H + 0.5 * U * site_op(L, i, P_D)
        else:
            H = H + U * site_op(L, i, N_UPDN)
    return H.tocsr()


def pseudospin(L):
    """T^+, T^-, T^z of Eq. (4) with eps_i = (-1)^i, i 0-based."""
    cup, cdn = annihilators(L)
    dim = 4 ** L
    Tp = sp.csr_matrix((dim, dim))
    Ntot = sp.csr_matrix((dim, dim))
    for i in range(L):
        Tp = Tp + ((-1) ** i) * (cup[i].T @ cdn[i].T)
        Ntot = Ntot + cup[i].T @ cup[i] + cdn[i].T @ cdn[i]
    Tz = 0.5 * (Ntot - L * sp.identity(dim, format="csr"))
    return Tp.tocsr(), Tp.T.tocsr(), Tz.tocsr()


def spin_ops(L):
    """S^+, S^-, S^z total-spin generators."""
    cup, cdn = annihilators(L)
    dim = 4 ** L
    Sp = sp.csr_matrix((dim, dim))
    Sz = sp.csr_matrix((dim, dim))
    for i in range(L):
        Sp = Sp + cup[i].T @ cdn[i]
        Sz = Sz + 0.5 * (cup[i].T @ cup[i] - cdn[i].T @ cdn[i])
    return Sp.tocsr(), Sp.T.tocsr(), Sz.tocsr()


def casimir(plus, minus, z):
    """J^2 = (J+J- + J-J+)/2 + Jz^2."""
    return 0.5 * (plus @ minus + minus @ plus) + z @ z


def neel_index(L):
    """Basis index of |up,dn,up,dn,...> (site 0 = most significant base-4 digit)."""
    idx = 0
    for i in range(L):
        idx = idx * 4 + (1 if i % 2 == 0 else 2)
    return idx


def neel_state(L):
    """Eq. (2) as a dense vector.  With the mode order 0up,0dn,1up,... the
    product basis state |up,dn,up,dn,...> differs from Eq. (2)'s operator ordering only
    by a global sign, which no observable sees."""
    v = np.zeros(4 ** L, dtype=complex)
    v[neel_index(L)] = 1.0
    return v


def sector_indices(L, n_up, n_dn):
    """Indices of basis states with (N_up, N_dn) = (n_up, n_dn)."""
    idx = np.arange(4 ** L)
    nu = np.zeros(4 ** L, dtype=int)
    nd = np.zeros(4 ** L, dtype=int)
    x = idx.copy()
    for _ in range(L):
        digit = x % 4
        nu += (digit == 1) | (digit == 3)
        nd += (digit == 2) | (digit == 3)
        x //= 4
    return idx[(nu == n_up) & (nd == n_dn)]


class ExactEvolution:
    """O-ED: exact time evolution of the Neel state under Eq. (1) in the (L/2, L/2) sector."""

    def __init__(self, L, t_h, U):
        self.L = L
        H = hamiltonian(L, t_h, U)
        self.sec = sector_indices(L, L // 2, L // 2)
        Hs = H[self.sec][:, self.sec].toarray()
        assert np.allclose(Hs, Hs.T)
        self.E, self.V = np.linalg.eigh(Hs)
        psi0 = neel_state(L)[self.sec]
        self.c0 = self.V.T @ psi0
        self.Hs = Hs
        # diagonal observables in the sector
        digits = np.zeros((L, len(self.sec)), dtype=int)
        x = self.sec.copy()
        for i in range(L - 1, -1, -1):
            digits[i] = x % 4
            x //= 4
        self.nup = ((digits == 1) | (digits == 3)).astype(float)
        self.ndn = ((digits == 2) | (digits == 3)).astype(float)
        self.docc = (digits == 3).astype(float)

    def state(self, t):
        return self.V @ (np.exp(-1j * self.E * t) * self.c0)

    def observables(self, t):
        psi = self.state(t)
        p = np.abs(psi) ** 2
        return dict(n_up=self.nup @ p, n_dn=self.ndn @ p, docc=self.docc @ p,
                    norm2=p.sum(), energy=float(np.real(np.vdot(psi, self.Hs @ psi))))
