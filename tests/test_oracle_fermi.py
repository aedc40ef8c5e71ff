"""Pins for oracle/fermi.py, oracle/u0.py: algebra the paper states (Eqs. 1-6) and textbook results."""
import numpy as np
import scipy.sparse as sp

from oracle import fermi, u0


def _comm(a, b):
    return a @ b - b @ a


def _max(m):
    return abs(m).max() if m.nnz else 0.0


def test_canonical_anticommutation():
    L = 3
    cup, cdn = fermi.annihilators(L)
    ops = cup + cdn
    eye = sp.identity(4 ** L)
    for i, a in enumerate(ops):
        for j, b in enumerate(ops):
            assert _max(a @ b + b @ a) < 1e-15
            anti = a @ b.T + b.T @ a
            assert _max(anti - (eye if i == j else 0 * eye)) < 1e-15


def test_two_site_spectrum_analytic():
    """L=2 half-filled Hubbard: singlet energies (U -+ sqrt(U^2+16 t^2))/2, triplet 0, and U."""
    t_h, U = 1.0, 4.0
    H = fermi.hamiltonian(2, t_h, U).toarray()
    sec = fermi.sector_indices(2, 1, 1)
    E = np.linalg.eigvalsh(H[np.ix_(sec, sec)])
    ref = sorted([(U - np.sqrt(U * U + 16 * t_h * t_h)) / 2, 0.0, U, (U + np.sqrt(U * U + 16 * t_h * t_h)) / 2])
    assert np.allclose(E, ref, atol=1e-13)


def test_symmetries_of_H():
    """Eqs. (4)-(6) PAPER.md:194-204 with reading A-2: [H_Eq1, T+] = U T+, [H_sym, T+-] = 0."""
    L, t_h, U = 4, 1.0, 4.0
    H = fermi.hamiltonian(L, t_h, U)
    Hs = fermi.hamiltonian(L, t_h, U, symmetric=True)
    Tp, Tm, Tz = fermi.pseudospin(L)
    Sp, Sm, Sz = fermi.spin_ops(L)
    assert _max(H - H.T) < 1e-15
    assert _max(_comm(Tp, Tm) - 2 * Tz) < 1e-14           # Eq. (5)
    assert _max(_comm(Tz, Tp) - Tp) < 1e-14
    assert _max(_comm(Hs, Tp)) < 1e-13 and _max(_comm(Hs, Tz)) < 1e-13
    assert _max(_comm(H, Tp) - U * Tp) < 1e-13            # Eq. (1) literally is not a T-scalar
    assert _max(Hs - (H - U * Tz)) < 1e-13
    for G in (Sp, Sz, fermi.casimir(Sp, Sm, Sz)):
        assert _max(_comm(H, G)) < 1e-12


def test_neel_quantum_numbers():
    """Neel has T_tot = 0, S^z = 0 and no definite S_tot (<S^2> = L/2)."""
    L = 4
    psi = fermi.neel_state(L)
    Tp, Tm, Tz = fermi.pseudospin(L)
    Sp, Sm, Sz = fermi.spin_ops(L)
    assert np.linalg.norm(fermi.casimir(Tp, Tm, Tz) @ psi) < 1e-14
    assert np.linalg.norm(Sz @ psi) < 1e-14
    s2 = np.vdot(psi, fermi.casimir(Sp, Sm, Sz) @ psi).real
    assert abs(s2 - L / 2) < 1e-14
    # Eq. (2): the product state equals the operator string acting on the vacuum up to a sign
    cup, cdn = fermi.annihilators(L)
    vac = np.zeros(4 ** L)
    vac[0] = 1.0
    v = vac
    for j in (3, 1):
        v = cdn[j].T @ v
    for i in (2, 0):
        v = cup[i].T @ v
    assert abs(abs(np.vdot(psi, v)) - 1.0) < 1e-15


def test_u0_closed_form_vs_ed_and_sum_rules():
    L, t_h = 6, 1.0
    ed = fermi.ExactEvolution(L, t_h, 0.0)
    for t in (0.0, 0.3, 1.1):
        e, u = ed.observables(t), u0.observables(L, t_h, t)
        assert np.abs(e["n_up"] - u["n_up"]).max() < 1e-12
        assert np.abs(e["n_dn"] - u["n_dn"]).max() < 1e-12
        assert np.abs(e["docc"] - u["docc"]).max() < 1e-12
        assert abs(u["n_up"].sum() - L / 2) < 1e-12
    G = u0.propagator(60, 1.0, 0.8)
    assert np.abs(G @ G.conj().T - np.eye(60)).max() < 1e-12          # unitary
    h = -(np.eye(60, k=1) + np.eye(60, k=-1))
    lam, V = np.linalg.eigh(h)
    assert np.abs(G - (V * np.exp(-0.8j * lam)) @ V.T).max() < 1e-12   # = exp(-i h t)


def test_ed_conserves():
    ed = fermi.ExactEvolution(4, 1.0, 4.0)
    o0, o1 = ed.observables(0.0), ed.observables(0.9)
    assert abs(o1["norm2"] - 1) < 1e-13 and abs(o1["energy"] - o0["energy"]) < 1e-12
    assert np.allclose(o0["n_up"], [1, 0, 1, 0]) and np.allclose(o0["docc"], 0)
    assert np.allclose(o1["n_up"] + o1["n_dn"], 1.0, atol=1e-12)       # <n_i> = 1 (reading A-12)
