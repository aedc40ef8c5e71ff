"""Pins of oracle/vecops.py against things other than itself: the weighted dot against oracle/symm.inner on a
block dictionary; the unnormalised Lanczos recurrence against the textbook normalised three-term recurrence and
against the exact tridiagonalisation property Q^H H Q = T on a random Hermitian matrix."""
import numpy as np

from oracle import symm, vecops


def test_wdot_equals_symm_inner():
    rng = np.random.default_rng(3)
    keys = [((0, 0), 0, (1, 0)), ((0, 0), 2, (0, 1)), ((1, 1), 2, (1, 2)), ((2, 0), 1, (1, 4))]
    x = {k: rng.standard_normal((3, 2)) + 1j * rng.standard_normal((3, 2)) for k in keys}
    y = {k: rng.standard_normal((3, 2)) + 1j * rng.standard_normal((3, 2)) for k in keys}
    bl, bw = [6] * 4, [k[-1][1] + 1 for k in keys]
    fx = np.concatenate([x[k].ravel() for k in keys])
    fy = np.concatenate([y[k].ravel() for k in keys])
    assert abs(vecops.wdot(bl, bw, fx, fy) - symm.inner(x, y)) < 1e-13
    assert bw == [1, 2, 3, 5]


def test_unnormalised_recurrence_is_lanczos():
    rng = np.random.default_rng(4)
    n, m = 40, 8
    Hm = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    Hm = Hm + Hm.conj().T
    bl, bw = [n], [1]
    v0 = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    # textbook: beta_j v_{j+1} = H v_j - alpha_j v_j - beta_{j-1} v_{j-1}
    V = [v0 / np.linalg.norm(v0)]
    alpha, beta = [], []
    for j in range(m):
        w = Hm @ V[j]
        a = np.vdot(V[j], w).real
        w = w - a * V[j] - (beta[j - 1] * V[j - 1] if j > 0 else 0)
        b = np.linalg.norm(w)
        alpha.append(a)
        beta.append(b)
        V.append(w / b)
    # unnormalised form
    U = [v0 / np.linalg.norm(v0)]
    b2 = [1.0]
    al2 = []
    for j in range(m):
        w = Hm @ U[j]
        a_raw = np.vdot(U[j], w).real
        al2.append(a_raw / b2[j])
        u, n2 = vecops.lanczos_update(bl, bw, a_raw, b2[j] if j > 0 else -1.0, b2[j - 1] if j > 1 else -1.0, 1e-300,
                                      U[j], U[j - 1] if j > 0 else None, w)
        U.append(u)
        b2.append(n2)
    assert np.abs(np.array(al2) - np.array(alpha)).max() < 1e-11
    assert np.abs(np.sqrt(np.array(b2[1:])) - np.array(beta)).max() < 1e-11
    for j in range(m + 1):
        assert np.linalg.norm(U[j] / np.sqrt(b2[j]) - V[j]) < 1e-9
    Q = np.array(V[:m]).T
    T = Q.conj().T @ Hm @ Q
    assert np.abs(T - (np.diag(alpha) + np.diag(beta[:m - 1], 1) + np.diag(beta[:m - 1], -1))).max() < 1e-9


def test_lincomb_and_copy_blocks():
    rng = np.random.default_rng(5)
    V = rng.standard_normal((3, 10)) + 1j * rng.standard_normal((3, 10))
    c = np.array([1 + 2j, -0.5, 3j])
    assert np.allclose(vecops.lincomb(c, V), np.tensordot(c, V, axes=1))
    src = np.arange(24, dtype=complex)
    dst = np.zeros(40, dtype=complex)
    vecops.copy_blocks([(2, 5, 2, 3, 6, 4, 0, 2.0), (1, 20, 2, 3, 6, 5, 1, 1.0)], src, dst)
    assert np.allclose(dst[5:8], 2 * src[2:5]) and np.allclose(dst[9:12], 2 * src[8:11])
    M = np.array([src[1:4], src[7:10]])           # 2 x 3 block; transposed copy is 3 x 2 with ld 5
    assert np.allclose(dst[20:22], M[:, 0]) and np.allclose(dst[25:27], M[:, 1]) and np.allclose(dst[30:32], M[:, 2])
