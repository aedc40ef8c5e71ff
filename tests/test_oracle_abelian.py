"""Pins of oracle/abelian.py (U(1) x U(1) reference, NEXT-4): embedded block results equal the dense contractions
of oracle/dense_tdvp.py (themselves pinned against five-operand einsums and ED) on a random abelian-symmetric
chain; the MPO respects the charges; the embedded chain state has definite N_up, N_dn; the profile bookkeeping."""
import numpy as np

import fh_inputs.abelian as fab
from oracle import abelian as ab
from oracle import dense_tdvp as dt
from oracle import fermi


def _rand(rng, m, n):
    return rng.standard_normal((m, n)) + 1j * rng.standard_normal((m, n))


def _chain(L=4, seed=2):
    rng = np.random.default_rng(seed)
    dims = [{k: min(v, int(rng.integers(1, 4))) for k, v in d.items()} for d in fab.chain_dims(64, L)]
    A = [{k: _rand(rng, dims[i][k[0]], dims[i + 1][k[2]]) for k in ab.site_keys(dims[i], dims[i + 1])} for i in range(L)]
    return rng, dims, A


def test_labels_and_profile_bookkeeping():
    assert fab.SITE_Q == ab.SITE_Q and fab.MPO_Q == ab.MPO_Q
    assert [fab.unpack(q) for q in ab.SITE_Q] == [(0, -1), (1, 0), (-1, 0), (0, 1)]      # (N_up - N_dn, N - 1)
    assert [fab.unpack(q) for q in ab.MPO_Q] == [(0, 0), (1, 1), (-1, 1), (-1, -1), (1, -1), (0, 0)]
    for k in (29, 30, 31):
        p = fab.profile(k, 4096)
        assert 4096 - 150 <= sum(p.values()) <= 4096
        for (q, z) in p:
            q1, dn = fab.unpack(q)
            assert z == 0 and (k + dn + q1) % 2 == 0
    d = fab.chain_dims(10 ** 6, 6)                     # uncapped: the full Hilbert space sectors of 6 sites
    assert d[0] == {(0, 0): 1} and d[6] == {(0, 0): 1} and sum(d[3].values()) == 64      # all 4^3 states of the left half


def test_mpo_is_eq1_and_respects_charges():
    W = ab.mpo_elements(1.0, 4.0)
    assert len(W) == 11
    L = 4
    Wd = dt.dense_mpo(1.0, 4.0)
    cur = Wd[0].transpose(1, 2, 0)
    for _ in range(1, L):
        d = cur.shape[0] * 4
        cur = np.einsum("abw,wvcd->acbdv", cur, Wd).reshape(d, d, 6)
    assert np.abs(cur[:, :, 5] - fermi.hamiltonian(L, 1.0, 4.0).toarray()).max() < 1e-13


def test_env_and_apply_equal_dense_contractions():
    L = 4
    rng, dims, A = _chain(L)
    W = ab.mpo_elements(1.0, 4.0)
    Wd = dt.dense_mpo(1.0, 4.0)
    Ad = [ab.embed_site(A[i], dims[i], dims[i + 1]) for i in range(L)]
    Le, Re = [ab.boundary_left()], [None] * (L + 1)
    for i in range(L):
        Le.append(ab.env_update_left(Le[i], A[i], W))
    Re[L] = ab.boundary_right()
    for i in range(L - 1, -1, -1):
        Re[i] = ab.env_update_right(Re[i + 1], A[i], W)
    Ld = [ab.embed_env(Le[0], dims[0], dims[0])]
    for i in range(L):
        Ld.append(dt.update_left(Ld[i], Ad[i], Wd))
    Rd = [None] * (L + 1)
    Rd[L] = ab.embed_env(Re[L], dims[L], dims[L])
    for i in range(L - 1, -1, -1):
        Rd[i] = dt.update_right(Rd[i + 1], Ad[i], Wd)
    for i in range(L + 1):
        for E, D in ((Le[i], Ld[i]), (Re[i], Rd[i])):
            assert np.abs(ab.embed_env(E, dims[i], dims[i]) - D).max() < 1e-12 * max(1.0, np.abs(D).max())
            assert set(E) <= set(ab.env_keys(dims[i], dims[i]))
    # the embedded state has N_up = N_dn = L / 2; <psi|H|psi> and <psi|psi> sit in the last left environment
    psi = Ad[0].reshape(4, -1)
    for i in range(1, L):
        psi = (psi @ Ad[i].reshape(Ad[i].shape[0], -1)).reshape(-1, Ad[i].shape[2])
    psi = psi.ravel()
    sec = fermi.sector_indices(L, L // 2, L // 2)
    mask = np.ones(psi.size, dtype=bool)
    mask[sec] = False
    assert np.abs(psi[mask]).max() == 0.0 and np.linalg.norm(psi[sec]) > 0
    H = fermi.hamiltonian(L, 1.0, 4.0)
    assert abs(Le[L][((0, 0), 5, (0, 0))][0, 0] - np.vdot(psi, H @ psi)) < 1e-10 * abs(np.vdot(psi, psi))
    assert abs(Le[L][((0, 0), 0, (0, 0))][0, 0] - np.vdot(psi, psi)) < 1e-10 * abs(np.vdot(psi, psi))
    for i in range(L - 1):
        keys = ab.theta_keys(dims[i], dims[i + 2])
        assert keys == fab.theta_block_keys(dims[i], dims[i + 2])
        th = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]) for k in keys}
        ph = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]) for k in keys}
        out = ab.heff2_apply(Le[i], Re[i + 2], th, W, W)
        ref = dt.heff2(Ld[i], Wd, Rd[i + 2], ab.embed_theta(th, dims[i], dims[i + 2]))
        got = ab.embed_theta(out, dims[i], dims[i + 2])
        assert np.linalg.norm(got - ref) < 1e-13 * np.linalg.norm(ref)
        hph = ab.heff2_apply(Le[i], Re[i + 2], ph, W, W)
        assert abs(ab.inner(ph, out) - np.conj(ab.inner(th, hph))) < 1e-12 * abs(ab.inner(ph, out))
    for i in range(L):
        assert ab.site_keys(dims[i], dims[i + 1]) == fab.site_block_keys(dims[i], dims[i + 1])
        out = ab.heff1_apply(Le[i], Re[i + 1], A[i], W)
        ref = dt.heff1(Ld[i], Wd, Rd[i + 1], Ad[i])
        assert np.linalg.norm(ab.embed_site(out, dims[i], dims[i + 1]) - ref) < 1e-13 * np.linalg.norm(ref)
