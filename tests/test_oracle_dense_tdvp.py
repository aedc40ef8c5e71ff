"""Pins for oracle/dense_tdvp.py (O-D): MPO = Eq. (1), Lanczos exponential, TDVP vs ED."""
import numpy as np
import scipy.linalg as sla

from oracle import dense_tdvp as dt
from oracle import fermi


def test_dense_mpo_equals_hamiltonian():
    L, t_h, U = 4, 1.0, 4.0
    W = dt.dense_mpo(t_h, U)
    cur = W[0].transpose(1, 2, 0)
    for _ in range(1, L):
        d = cur.shape[0] * 4
        cur = np.einsum("abw,wvcd->acbdv", cur, W).reshape(d, d, 6)
    assert np.abs(cur[:, :, 5] - fermi.hamiltonian(L, t_h, U).toarray()).max() < 1e-13


def test_lanczos_exp_vs_expm():
    rng = np.random.default_rng(3)
    n = 40
    H = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    H = (H + H.conj().T) / 2
    v = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    ref = sla.expm(-0.05j * H) @ v
    out = dt.lanczos_exp(lambda x: H @ x, v, 0.05, 12)
    assert np.linalg.norm(out - ref) / np.linalg.norm(ref) < 1e-12
    # exact when the Krylov space is the whole space
    out = dt.lanczos_exp(lambda x: H @ x, v, 1.0, n)
    assert np.linalg.norm(out - sla.expm(-1j * H) @ v) / np.linalg.norm(v) < 1e-9


def test_heff_matches_einsum():
    rng = np.random.default_rng(5)
    W = dt.dense_mpo(1.0, 4.0)
    cl, cr = 3, 5
    Le = rng.standard_normal((cl, 6, cl)) + 1j * rng.standard_normal((cl, 6, cl))
    Re = rng.standard_normal((cr, 6, cr)) + 1j * rng.standard_normal((cr, 6, cr))
    th = rng.standard_normal((cl, 4, 4, cr)) + 1j * rng.standard_normal((cl, 4, 4, cr))
    ref = np.einsum("xwa,wvps,vuqt,astb,yub->xpqy", Le, W, W, th, Re)
    assert np.abs(dt.heff2(Le, W, Re, th) - ref).max() < 1e-12
    A = rng.standard_normal((cl, 4, cr)) + 1j * rng.standard_normal((cl, 4, cr))
    ref1 = np.einsum("xwa,wvps,asb,yvb->xpy", Le, W, A, Re)
    assert np.abs(dt.heff1(Le, W, Re, A) - ref1).max() < 1e-12
    refL = np.einsum("xps,xwa,wvpq,aqc->svc", A.conj().transpose(0, 1, 2), Le, W, A)
    assert np.abs(dt.update_left(Le, A, W) - refL).max() < 1e-12
    refR = np.einsum("xpy,wvpq,yvb,cqb->xwc", A.conj(), W, Re, A)
    assert np.abs(dt.update_right(Re, A, W) - refR).max() < 1e-12


def test_truncate_rule():
    keep, disc = dt.truncate_rule([np.array([3.0, 2.0, 1.0]), np.array([2.5, 0.5])], [1, 2], 4, -1.0)
    assert keep == [2, 1]                   # order 3.0(1), 2.5(2), 2.0(1) -> dim 4; 1.0 would be 5
    tot = 9 + 4 + 1 + 2 * (6.25 + 0.25)
    assert abs(disc - (1 + 0.5) / tot) < 1e-15
    keep, _ = dt.truncate_rule([np.array([1.0, 1e-15])], [1], 100, -1.0)
    assert keep == [1]                      # relative 1e-14 floor
    keep, disc = dt.truncate_rule([np.array([1.0, 0.1, 0.01])], [1], 100, 1e-3)
    assert keep == [2] and disc < 1e-3      # tail weight 1e-4/1.0101 <= 1e-3 after two
    keep, _ = dt.truncate_rule([np.array([1.0]), np.array([1.0])], [3, 1], 2, -1.0)
    assert keep == [1, 0]                   # keeps at least one even above the cap


def test_tdvp_vs_ed_and_time_step_order():
    """Config-1-like check at L=4: two-site TDVP from the Neel state has an O(dt^2) splitting
    error and conserves norm/energy (E-tol in DESIGN.md)."""
    L, t_h, U = 4, 1.0, 4.0
    ed = fermi.ExactEvolution(L, t_h, U)
    errs = []
    for dtime in (0.1, 0.05):
        td = dt.DenseTDVP(L, t_h, U, krylov_dim=10)
        steps = int(round(1.0 / dtime))
        err = 0.0
        for k in range(1, steps + 1):
            td.step(dtime)
            o, e = td.observables(), ed.observables(dtime * k)
            err = max(err, np.abs(o["n_up"] - e["n_up"]).max(), np.abs(o["docc"] - e["docc"]).max())
            assert abs(o["norm2"] - 1) < 1e-11
            assert np.abs(o["n_up"] + o["n_dn"] - 1).max() < 1e-11
        errs.append(err)
        psi = td.to_state()
        H = fermi.hamiltonian(L, t_h, U)
        assert abs(np.vdot(psi, H @ psi).real) < 1e-5           # Neel energy is 0
    assert errs[1] < 2e-6
    assert 3.5 < errs[0] / errs[1] < 10.0     # at least second order in dt (measured: 8.0)


def test_tdvp1_on_saturated_bonds_vs_ed_and_time_step_order():
    """NEXT-1: one-site TDVP.  On L = 4 three untruncated two-site steps bring every
    bond to its maximal dimension (4, 16, 4); from there the one-site manifold is the whole Hilbert
    space, so TDVP1 must follow the exact evolution up to its O(dt^2) splitting error, with bond
    dimensions frozen, norm and energy conserved.  Halving dt must cut the error ~4x."""
    L, t_h, U = 4, 1.0, 4.0
    ed = fermi.ExactEvolution(L, t_h, U)
    errs = []
    for dt_ in (0.05, 0.025):
        sim = dt.DenseTDVP(L, t_h, U, krylov_dim=16)
        n2 = int(round(0.15 / dt_))
        for _ in range(n2):
            sim.step(dt_)
        assert sim.bond_dims() == [4, 16, 4]
        worst = 0.0
        n1 = int(round(0.5 / dt_))
        for k in range(1, n1 + 1):
            sim.step1(dt_)
            t = (n2 + k) * dt_
            o, e = sim.observables(), ed.observables(t)
            worst = max(worst, max(np.abs(o[q] - e[q]).max() for q in ("n_up", "n_dn", "docc")))
            assert abs(o["norm2"] - 1.0) < 1e-10
        assert sim.bond_dims() == [4, 16, 4]
        errs.append(worst)
    assert errs[0] < 2e-5, errs
    assert 3.0 < errs[0] / errs[1] < 10.0, errs        # at least second order (measured 5.0e-7 -> 6.2e-8)
    # zero-site operator: Hermitian when the environments are (they are, for a mixed-canonical state)
    rng = np.random.default_rng(2)
    Le, Re = sim.Lenv[1], sim.Renv[1]
    C1 = rng.standard_normal((Le.shape[0], Re.shape[0])) + 1j * rng.standard_normal((Le.shape[0], Re.shape[0]))
    C2 = rng.standard_normal(C1.shape) + 1j * rng.standard_normal(C1.shape)
    assert abs(np.vdot(C1, dt.heff0(Le, Re, C2)) - np.conj(np.vdot(C2, dt.heff0(Le, Re, C1)))) < 1e-10


# ---- NEXT-2, reading A-15: adaptive Krylov dimension -------------------------------------------
def _rand_herm(n, scale, seed):
    rng = np.random.default_rng(seed)
    a = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    h = (a + a.conj().T) / 2
    return h * (scale / np.linalg.norm(h, 2))


def test_krylov_residual_is_the_ode_residual():
    """The stopping estimate is |tau| |r_k(tau)| with r_k = y_k' + i H y_k the residual of the Krylov
    approximation in y' = -i H y.  Brute force: build V_k, T_k by plain Lanczos here, evaluate the residual
    vector from its definition and compare its norm with the oracle's estimate / |tau|."""
    n, k, tau = 60, 5, 0.37
    H = _rand_herm(n, 3.0, 11)
    rng = np.random.default_rng(12)
    v = rng.normal(size=n) + 1j * rng.normal(size=n)
    v /= np.linalg.norm(v)
    V = [v]
    alpha, beta = [], []
    for j in range(k):
        w = H @ V[j]
        alpha.append(np.vdot(V[j], w).real)
        w = w - alpha[j] * V[j] - (beta[j - 1] * V[j - 1] if j else 0)
        for u in V:
            w = w - np.vdot(u, w) * u
        b = np.linalg.norm(w)
        if j < k - 1:
            beta.append(b)
            V.append(w / b)
    Vk = np.array(V).T
    Tk = Vk.conj().T @ H @ Vk
    u = sla.expm(-1j * tau * Tk)[:, 0]
    y = Vk @ u
    ydot = Vk @ (-1j * Tk @ u)
    r = ydot + 1j * (H @ y)
    est = dt.krylov_residual_estimate(alpha, beta, b, tau)
    assert abs(np.linalg.norm(r) - est / tau) < 1e-12 * max(1.0, np.linalg.norm(r))


def test_adaptive_krylov_meets_tolerance_and_bounds_error():
    """error(y_k(tau)) <= int_0^tau |r_k| <= estimate whenever |r_k(s)| is increasing on [0, tau] (true for
    tau |H| small against k); so the adaptive result is within adapt_tol of expm, and uses fewer vectors for
    a looser tolerance or a shorter step."""
    n = 120
    H = _rand_herm(n, 4.0, 21)
    rng = np.random.default_rng(22)
    v = rng.normal(size=n) + 1j * rng.normal(size=n)
    used = {}
    for tau in (0.05, 0.2, 0.5):
        exact = sla.expm(-1j * tau * H) @ v
        for tol in (1e-4, 1e-8, 1e-12):
            st = []
            y = dt.lanczos_exp(lambda x: H @ x, v, tau, 30, adapt_tol=tol, stats=st)
            err = np.linalg.norm(y - exact) / np.linalg.norm(v)
            assert err <= tol + 1e-13, (tau, tol, err, st)
            assert 1 <= st[0] < 30
            used[(tau, tol)] = st[0]
    for tau in (0.05, 0.2, 0.5):
        assert used[(tau, 1e-4)] < used[(tau, 1e-8)] < used[(tau, 1e-12)]
    for tol in (1e-4, 1e-8, 1e-12):
        assert used[(0.05, tol)] < used[(0.2, tol)] < used[(0.5, tol)]


def test_adaptive_krylov_off_and_cap():
    """adapt_tol = 0 is the fixed-m process bit for bit; a cap m smaller than the adaptive choice wins."""
    H = _rand_herm(50, 5.0, 31)
    rng = np.random.default_rng(32)
    v = rng.normal(size=50) + 1j * rng.normal(size=50)
    a = dt.lanczos_exp(lambda x: H @ x, v, 0.3, 8)
    b = dt.lanczos_exp(lambda x: H @ x, v, 0.3, 8, adapt_tol=0.0)
    assert np.array_equal(a, b)
    st = []
    c = dt.lanczos_exp(lambda x: H @ x, v, 0.3, 4, adapt_tol=1e-14, stats=st)
    assert st == [4]
    assert np.array_equal(c, dt.lanczos_exp(lambda x: H @ x, v, 0.3, 4))
    # a stop at k gives exactly the fixed-k result
    st = []
    d = dt.lanczos_exp(lambda x: H @ x, v, 0.3, 30, adapt_tol=1e-6, stats=st)
    assert np.allclose(d, dt.lanczos_exp(lambda x: H @ x, v, 0.3, st[0]), rtol=0, atol=1e-14)
