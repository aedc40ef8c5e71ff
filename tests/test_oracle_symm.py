"""Pins for oracle/symm.py and oracle/symm_tdvp.py (O-S): every reduced object is expanded to
its dense tensor ("dense embedding with coefficients expanded") and compared with the dense
contraction of oracle/dense_tdvp.py; plus the numbers the paper prints (W = 4, Table S2)."""
import numpy as np
import pytest

import fh_inputs as fi
from oracle import dense_tdvp as dt
from oracle import fermi, symm
from oracle import symm_tdvp as stv


def _rand(rng, m, n):
    return rng.standard_normal((m, n)) + 1j * rng.standard_normal((m, n))


@pytest.fixture(scope="module", params=[4, 6])
def chain(request):
    """Random symmetric MPS with all reachable sectors: L=4 (2j <= 2, degeneracies 1..3) and L=6 (2j <= 3, so
    that every branch of the recoupling coefficients with j >= 3/2 is embedded too; degeneracies 1..2)."""
    L, t_h, U = request.param, 1.0, 4.0
    rng = np.random.default_rng(1 if L == 4 else 6)
    tabs = fi.reachable_tables(L)
    dims = [{sec: int(rng.integers(1, 4 if L == 4 else 3)) for sec in tabs[k]} for k in range(L + 1)]
    dims[0] = {(0, 0): 1}
    dims[L] = {(0, 0): 1}
    A = [{k: _rand(rng, dims[i][k[0]], dims[i + 1][k[2]]) for k in symm.site_keys(dims[i], dims[i + 1])}
         for i in range(L)]
    Ws = [symm.mpo_reduced(i, t_h, U) for i in range(L)]
    Wd = [symm.embed_mpo(Ws[i], i) for i in range(L)]
    Ad = [symm.embed_site(A[i], dims[i], dims[i + 1], i) for i in range(L)]
    Le = [symm.boundary_left()]
    for i in range(L):
        Le.append(symm.env_update_left(Le[i], A[i], Ws[i]))
    Re = [None] * (L + 1)
    Re[L] = symm.boundary_right()
    for i in range(L - 1, -1, -1):
        Re[i] = symm.env_update_right(Re[i + 1], A[i], Ws[i])
    Ld = [symm.embed_env(Le[0], dims[0], dims[0])]
    for i in range(L):
        Ld.append(dt.update_left(Ld[i], Ad[i], Wd[i]))
    Rd = [None] * (L + 1)
    Rd[L] = symm.embed_env(Re[L], dims[L], dims[L])
    for i in range(L - 1, -1, -1):
        Rd[i] = dt.update_right(Rd[i + 1], Ad[i], Wd[i])
    return dict(L=L, t_h=t_h, U=U, dims=dims, A=A, Ws=Ws, Wd=Wd, Ad=Ad, Le=Le, Re=Re, Ld=Ld, Rd=Rd, rng=rng)


def test_reduced_site_operators_printed_values():
    """Reading F-2: the non-zero reduced matrix elements."""
    for eps in (1, -1):
        o = symm.reduced_site_ops(eps)
        r2 = np.sqrt(2.0)
        ref_p = np.zeros((3, 3)); ref_p[0, 2] = -r2; ref_p[2, 1] = eps
        ref_m = np.zeros((3, 3)); ref_m[1, 2] = -r2; ref_m[2, 0] = -eps
        ref_pp = np.zeros((3, 3)); ref_pp[0, 2] = -r2; ref_pp[2, 1] = -eps
        ref_mp = np.zeros((3, 3)); ref_mp[1, 2] = -r2; ref_mp[2, 0] = eps
        assert np.abs(o["psi_p"] - ref_p).max() < 1e-14 and np.abs(o["psi_m"] - ref_m).max() < 1e-14
        assert np.abs(o["psi_p_par"] - ref_pp).max() < 1e-14 and np.abs(o["psi_m_par"] - ref_mp).max() < 1e-14
        assert np.allclose(o["one"], np.eye(3)) and np.allclose(o["p_d"], np.diag([0, 0, 1.0]))
        assert np.allclose(o["sz"], np.diag([0.5, -0.5, 0]))


def test_mpo_embedding_equals_H_sym_and_W4(chain):
    """Reduced MPO bond dimension W = 4; expanded chain = dense H_sym exactly."""
    L, Wd = chain["L"], chain["Wd"]
    assert len(symm.MPOB) == 4
    cur = Wd[0][0].transpose(1, 2, 0)
    for i in range(1, L):
        d = cur.shape[0] * 4
        cur = np.einsum("abw,wvcd->acbdv", cur, Wd[i]).reshape(d, d, 6)
    Hs = fermi.hamiltonian(L, chain["t_h"], chain["U"], symmetric=True).toarray()
    assert np.abs(cur[:, :, 5] - Hs).max() < 1e-13
    # on half-filled states H_sym = Eq. (1)
    H = fermi.hamiltonian(L, chain["t_h"], chain["U"]).toarray()
    sec = fermi.sector_indices(L, L // 2, L // 2)
    assert np.abs(Hs[np.ix_(sec, sec)] - H[np.ix_(sec, sec)]).max() < 1e-13


def test_symmetric_mps_is_a_T0_Sz0_state(chain):
    L, Ad = chain["L"], chain["Ad"]
    psi = Ad[0].reshape(4, -1)
    for i in range(1, L):
        psi = (psi @ Ad[i].reshape(Ad[i].shape[0], -1)).reshape(-1, Ad[i].shape[2])
    psi = psi.ravel()
    Tp, Tm, Tz = fermi.pseudospin(L)
    _, _, Sz = fermi.spin_ops(L)
    assert np.linalg.norm(fermi.casimir(Tp, Tm, Tz) @ psi) < 1e-12 * np.linalg.norm(psi)
    assert np.linalg.norm(Sz @ psi) < 1e-12 * np.linalg.norm(psi)
    # full contraction: norm and energy
    Hs = fermi.hamiltonian(L, chain["t_h"], chain["U"], symmetric=True)
    LL = chain["Le"][L]
    assert abs(LL[((0, 0), 0, (0, 0))][0, 0] - np.vdot(psi, psi)) < 1e-10 * abs(np.vdot(psi, psi))
    assert abs(LL[((0, 0), 3, (0, 0))][0, 0] - np.vdot(psi, Hs @ psi)) < 1e-10 * abs(np.vdot(psi, psi))


def test_environments_vs_dense(chain):
    L, dims = chain["L"], chain["dims"]
    for i in range(L + 1):
        dl = chain["Ld"][i]
        dr = chain["Rd"][i]
        assert np.abs(symm.embed_env(chain["Le"][i], dims[i], dims[i]) - dl).max() < 1e-12 * max(1, np.abs(dl).max())
        assert np.abs(symm.embed_env(chain["Re"][i], dims[i], dims[i]) - dr).max() < 1e-12 * max(1, np.abs(dr).max())


def test_heff2_vs_dense_hermiticity_inner(chain):
    L, dims, rng = chain["L"], chain["dims"], chain["rng"]
    for i in range(L - 1):
        keys = symm.theta_keys(dims[i], dims[i + 2])
        assert keys == fi.theta_block_keys(dims[i], dims[i + 2])
        th = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]) for k in keys}
        ph = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]) for k in keys}
        out = symm.heff2_apply(chain["Le"][i], chain["Re"][i + 2], th, chain["Ws"][i], chain["Ws"][i + 1])
        thd = symm.embed_theta(th, dims[i], dims[i + 2], i)
        phd = symm.embed_theta(ph, dims[i], dims[i + 2], i)
        # H_eff theta = L . W_i . W_{i+1} . theta . R, one pairwise contraction at a time
        t1 = np.einsum("xwa,astb->xwstb", chain["Ld"][i], thd)
        t2 = np.einsum("wvps,xwstb->xvptb", chain["Wd"][i], t1)
        t3 = np.einsum("vuqt,xvptb->xpqub", chain["Wd"][i + 1], t2)
        ref = np.einsum("xpqub,yub->xpqy", t3, chain["Rd"][i + 2])
        got = symm.embed_theta(out, dims[i], dims[i + 2], i)
        assert np.linalg.norm(got - ref) < 1e-13 * np.linalg.norm(ref)
        assert abs(symm.inner(ph, th) - np.vdot(phd, thd)) < 1e-12 * np.linalg.norm(phd) * np.linalg.norm(thd)
        hph = symm.heff2_apply(chain["Le"][i], chain["Re"][i + 2], ph, chain["Ws"][i], chain["Ws"][i + 1])
        assert abs(symm.inner(ph, out) - np.conj(symm.inner(th, hph))) < 1e-12 * abs(symm.inner(ph, out))


def test_heff1_vs_dense(chain):
    for i in range(chain["L"]):
        dims = chain["dims"]
        assert symm.site_keys(dims[i], dims[i + 1]) == fi.site_block_keys(dims[i], dims[i + 1])
        out = symm.heff1_apply(chain["Le"][i], chain["Re"][i + 1], chain["A"][i], chain["Ws"][i])
        t1 = np.einsum("xwa,asb->xwsb", chain["Ld"][i], chain["Ad"][i])
        t2 = np.einsum("wvps,xwsb->xvpb", chain["Wd"][i], t1)
        ref = np.einsum("xvpb,yvb->xpy", t2, chain["Rd"][i + 1])
        got = symm.embed_site(out, dims[i], dims[i + 1], i)
        assert np.linalg.norm(got - ref) < 1e-13 * np.linalg.norm(ref)


def test_svd_split_vs_dense_svd(chain):
    """F-7: singular values of the dense two-site matrix = those of M_c with multiplicity 2j_c+1;
    nothing dropped -> merge(A1, A2) reconstructs theta; canonical forms F-6."""
    L, dims, rng = chain["L"], chain["dims"], chain["rng"]
    i = 1
    keys = symm.theta_keys(dims[i], dims[i + 2])
    th = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]) for k in keys}
    thd = symm.embed_theta(th, dims[i], dims[i + 2], i)
    sv = np.linalg.svd(thd.reshape(thd.shape[0] * 4, -1), compute_uv=False)
    for direction in ("right", "left"):
        A1, A2, dm, info = symm.svd_split(th, dims[i], dims[i + 2], 10 ** 9, -1.0, direction)
        mine = np.sort(np.concatenate([np.repeat(s, c[1] + 1) for c, s in info["svals"].items()]))[::-1]
        n = min(len(sv), len(mine))
        assert np.abs(sv[:n] - mine[:n]).max() < 1e-12
        assert (sv[n:] < 1e-12).all() and (mine[n:] < 1e-12).all()
        th2 = symm.merge(A1, A2)
        assert max(np.abs(th2[k] - th[k]).max() for k in th) < 1e-12
        if direction == "right":
            chk = {}
            for (a, s, c), x in A1.items():
                chk[c] = chk.get(c, 0) + x.conj().T @ x
        else:
            chk = {}
            for (c, s, b), x in A2.items():
                chk[c] = chk.get(c, 0) + (b[1] + 1) / (c[1] + 1) * (x @ x.conj().T)
        assert max(np.abs(v - np.eye(len(v))).max() for v in chk.values()) < 1e-12
    # truncation: discarded weight equals the dense discarded weight for the same cut
    A1, A2, dm, info = symm.svd_split(th, dims[i], dims[i + 2], 6, -1.0, "right")
    kept_full = symm.chi_full(dm)
    assert kept_full <= 6
    allv = sorted(((s, c) for c, ss in info["svals"].items() for s in ss), key=lambda t: -t[0])
    tot = sum((c[1] + 1) * s * s for s, c in allv)
    kept_w = sum((c[1] + 1) * info["svals"][c][:k] @ info["svals"][c][:k] for c, k in info["keep"].items())
    assert abs(info["discarded"] - (tot - kept_w) / tot) < 1e-14


def test_task_lists_are_canonical_and_consistent(chain):
    i, dims = 1, chain["dims"]
    Lk, Rk = sorted(chain["Le"][i]), sorted(chain["Re"][i + 2])
    assert Lk == [k for k in symm.env_keys(dims[i], dims[i]) if k in chain["Le"][i]]
    tk = symm.theta_keys(dims[i], dims[i + 2])
    st1, st2 = symm.heff2_tasks(Lk, Rk, tk, chain["Ws"][i], chain["Ws"][i + 1])
    assert list(st1) == sorted(st1) and list(st2) == sorted(st2)
    for segs in st1.values():
        ks = [(e[1], e[2], t[1]) for e, t, _ in segs]
        assert ks == sorted(ks) and all(abs(a) >= symm.ALPHA_ZERO for _, _, a in segs)
    tup, al = symm.task_tuples(st1, list(st1), Lk, tk)
    assert tup.dtype == np.int32 and tup.shape == (sum(len(s) for s in st1.values()), 3)
    assert (np.diff(tup[:, 0]) >= 0).all()
    f = symm.heff2_flops(st1, st2, dims[i], dims[i + 2])
    assert f > 0 and f % 8 == 0
    # reading A-17: every intermediate block of the list is read by stage 2
    assert {seg[0] for segs in st2.values() for seg in segs} == set(st1)


class _Counting(np.ndarray):
    """ndarray that counts 8 m n k for every complex matrix product it takes part in."""
    flops = 0

    def __matmul__(self, other):
        a, b = np.asarray(self), np.asarray(other)
        _Counting.flops += 8 * a.shape[0] * a.shape[1] * b.shape[1]
        return (a @ b).view(_Counting)

    def __rmatmul__(self, other):
        a, b = np.asarray(other), np.asarray(self)
        _Counting.flops += 8 * a.shape[0] * a.shape[1] * b.shape[1]
        return (a @ b).view(_Counting)


def test_heff2_flops_hand_worked_and_counted(chain):
    """Pins of heff2_flops (the numerator of the headline GFLOP/s).
    (a) Hand-worked: the only bond of an L=2 chain, boundary environments L[(0,0),S,(0,0)] (2 x 2) and
    R[(0,0),F,(0,0)] (3 x 3), bond degeneracies d_l = 2, d_r = 3.  theta has the three blocks (s1,s2) = (up,dn),
    (dn,up), (pair,pair).  H = hopping + (U/2)(P_D,0 + P_D,1) has six non-zero reduced elements between them:
    P_D on site 0 (w_m = F) and on site 1 (w_m = S) on the pair block, and the four hopping terms pair<->(up,dn),
    pair<->(dn,up) (w_m = P, M).  Each is one stage-1 task (8 * 2*2*3) and one stage-2 task (8 * 2*3*3).
    (b) Counted: the products the oracle's own heff2_apply executes, counted by an instrumented ndarray."""
    dl, dr = {(0, 0): 2}, {(0, 0): 3}
    Lk, Rk = [((0, 0), 0, (0, 0))], [((0, 0), 3, (0, 0))]
    tk = symm.theta_keys(dl, dr)
    assert len(tk) == 3
    st1, st2 = symm.heff2_tasks(Lk, Rk, tk, symm.mpo_reduced(0, 1.0, 4.0), symm.mpo_reduced(1, 1.0, 4.0))
    assert sum(len(v) for v in st1.values()) == 6 and sum(len(v) for v in st2.values()) == 6
    assert symm.heff2_flops(st1, st2, dl, dr) == 8 * (6 * 2 * 2 * 3 + 6 * 2 * 3 * 3) == 1440
    dims, rng = chain["dims"], chain["rng"]
    for i in range(chain["L"] - 1):
        Le = {k: v.view(_Counting) for k, v in chain["Le"][i].items()}
        Re = {k: v.view(_Counting) for k, v in chain["Re"][i + 2].items()}
        th = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]).view(_Counting)
              for k in symm.theta_keys(dims[i], dims[i + 2])}
        _Counting.flops = 0
        symm.heff2_apply(Le, Re, th, chain["Ws"][i], chain["Ws"][i + 1])
        st1, st2 = symm.heff2_tasks(sorted(Le), sorted(Re), sorted(th), chain["Ws"][i], chain["Ws"][i + 1])
        assert _Counting.flops == symm.heff2_flops(st1, st2, dims[i], dims[i + 2]) > 0


def test_symmetric_tdvp_equals_dense_tdvp_and_measurements():
    """O-S driver = O-D to rounding (same m, nothing truncated); H10 formula = dense measurement."""
    L, t_h, U = 4, 1.0, 4.0
    s = stv.SymmTDVP(L, t_h, U, krylov_dim=10)
    d = dt.DenseTDVP(L, t_h, U, krylov_dim=10)
    ed = fermi.ExactEvolution(L, t_h, U)
    for k in range(1, 11):
        s.step(0.05)
        d.step(0.05)
        ms, od = s.measure_local(), d.observables()
        assert np.abs(ms["sz"] - 0.5 * (od["n_up"] - od["n_dn"])).max() < 1e-11
        assert np.abs(ms["docc"] - od["docc"]).max() < 1e-11
        assert np.allclose(ms["n"], 1.0)
    psi = s.to_state()
    assert abs(abs(np.vdot(psi, d.to_state())) - 1.0) < 1e-10       # same state up to a phase
    e = ed.observables(0.5)
    assert np.abs(ms["docc"] - e["docc"]).max() < 2e-6               # time-step error only
    g = s.measure_global()
    assert abs(g["norm2"] - 1) < 1e-11 and abs(g["energy"]) < 1e-5
    assert s.chi() == [1, 4, 16, 4, 1] and s.chi()[1:-1] == d.bond_dims()
    Tp, Tm, Tz = fermi.pseudospin(L)
    assert np.linalg.norm(fermi.casimir(Tp, Tm, Tz) @ psi) < 1e-10


def test_bookkeeping_table_s2_and_profiles():
    """Eqs. (8)-(10) PAPER.md:216-223 on Table S2: 32 sectors,
    chi_SU(2) = 12288, chi ~ 30000, d_max = 1735, parity n + 2j even."""
    d = fi.table_s2_profile()
    assert len(d) == 32 and symm.chi_su2(d) == 12288 and symm.d_max(d) == 1735
    assert symm.chi_full(d) == 30842 and abs(symm.chi_full(d) / 30000 - 1) < 0.05
    assert all((q + tj) % 2 == 0 for q, tj in d)
    assert 2.3 < symm.chi_full(d) / symm.chi_su2(d) < 2.6            # "chi ~ 2.4 chi_SU(2)" PAPER.md:233
    for k in (29, 30, 31):
        p = fi.gaussian_profile(k, 1024)
        assert 1024 - 30 <= symm.chi_full(p) <= 1024
        assert all((q + tj - k) % 2 == 0 for q, tj in p)
    chain = fi.chain_profiles(256, L=12)
    assert chain[0] == {(0, 0): 1} and chain[12] == {(0, 0): 1}
    tabs = fi.reachable_tables(12)
    assert all(set(chain[k]) <= set(tabs[k]) for k in range(13))


def test_one_site_tdvp_pieces_and_driver_vs_dense():
    """NEXT-1: (i) the zero-site apply with coefficient 1 equals the dense einsum of the embedded
    environments and bond matrix; (ii) the one-site splits reproduce the tensor and give canonical
    factors; (iii) the symmetric TDVP1 driver equals the dense one (itself pinned against ED) through
    observables, after a two-site phase that grows the bonds."""
    from oracle import symm_tdvp as stv
    from oracle import dense_tdvp as dtv
    L, t_h, U, dt = 6, 1.0, 4.0, 0.05
    sy = stv.SymmTDVP(L, t_h, U, krylov_dim=12)
    de = dtv.DenseTDVP(L, t_h, U, krylov_dim=12)
    for _ in range(3):
        sy.step(dt)
        de.step(dt)
    # (i) zero-site apply on bond 3 with the driver's own environments (left env needs building)
    Le = symm.boundary_left()
    for i in range(3):
        Le = symm.env_update_left(Le, sy.A[i], sy.W[i])
    Re = sy.Renv[3]
    d3 = sy.dims[3]
    rng = np.random.default_rng(4)
    C = {c: rng.standard_normal((d, d)) + 1j * rng.standard_normal((d, d)) for c, d in d3.items()}
    got = symm.embed_bond(symm.heff0_apply(Le, Re, C), d3, d3)
    ref = np.einsum("xwa,ab,ywb->xy", symm.embed_env(Le, d3, d3), symm.embed_bond(C, d3, d3),
                    symm.embed_env(Re, d3, d3))
    assert np.abs(got - ref).max() < 1e-12 * max(1.0, np.abs(ref).max())
    # (ii) splits
    A = sy.A[2]
    Q, Cm, dn = symm.split_site_right_moving(A, sy.dims[2], sy.dims[3])
    back = symm.absorb_right(Q, Cm)
    assert max(np.abs(back[k] - A[k]).max() for k in A) < 1e-13
    for c in dn:
        g = sum(Q[k].conj().T @ Q[k] for k in Q if k[2] == c)
        assert np.abs(g - np.eye(dn[c])).max() < 1e-12
    Q, Cm, dn = symm.split_site_left_moving(A, sy.dims[2], sy.dims[3])
    back = symm.absorb_left(Cm, Q)
    assert max(np.abs(back[k] - A[k]).max() for k in A) < 1e-13
    for a in dn:
        g = sum((k[2][1] + 1) / (a[1] + 1) * Q[k] @ Q[k].conj().T for k in Q if k[0] == a)
        assert np.abs(g - np.eye(dn[a])).max() < 1e-12
    # (iii) drivers
    worst = 0.0
    for _ in range(4):
        sy.step1(dt)
        de.step1(dt)
        a, b = sy.measure_local(), de.observables()
        worst = max(worst, np.abs(a["sz"] - 0.5 * (b["n_up"] - b["n_dn"])).max(), np.abs(a["docc"] - b["docc"]).max())
    assert worst < 1e-9, worst
    assert abs(sy.measure_global()["norm2"] - b["norm2"]) < 1e-10


def test_auto_switch_reading_A16_vs_ed():
    """Reading A-16: step_auto takes two-site steps until one of them grows no bond, then one-site steps.
    L = 4 untruncated: the bonds reach their maximal dimensions (4, 16, 4); the step after that grows nothing
    and flips the switch; on the saturated manifold one-site TDVP is exact up to the splitting error, so the
    observables keep following exact diagonalisation.  With a cap the switch comes as soon as the cap binds."""
    from oracle import symm_tdvp as stv
    L, t_h, U, dtime = 4, 1.0, 4.0, 0.05
    s = stv.SymmTDVP(L, t_h, U, krylov_dim=10)
    ed = fermi.ExactEvolution(L, t_h, U)
    seq, err = [], 0.0
    for k in range(1, 21):
        chi_before = s.chi()
        n = s.step_auto(dtime)
        seq.append(n)
        if n == 1:
            assert s.chi() == chi_before            # one-site steps never change a bond here
        o, e = s.measure_local(), ed.observables(dtime * k)
        err = max(err, np.abs(o["docc"] - e["docc"]).max(), np.abs(0.5 + o["sz"] - e["n_up"]).max())
    first1 = seq.index(1)
    assert first1 >= 2 and all(x == 2 for x in seq[:first1]) and all(x == 1 for x in seq[first1:])
    assert s.chi() == [1, 4, 16, 4, 1]
    assert err < 5e-6, err                           # splitting error only (dt = 0.05)
    capped = stv.SymmTDVP(6, t_h, U, krylov_dim=10, chi_max_full=12)
    seq = [capped.step_auto(dtime) for _ in range(5)]
    assert seq[0] == 2 and seq[-1] == 1 and max(capped.chi()) <= 12
