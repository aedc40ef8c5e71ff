"""U(1) x U(1) block-sparse reference ("U(1) x U(1), fp64").

TEST INFRASTRUCTURE (see oracle/__init__.py).  The abelian special case of the symmetric format of oracle/symm.py:
every multiplet is one-dimensional, every Clebsch-Gordan and recoupling coefficient is 1, and a tensor is just the
dense tensor cut into blocks by its conserved charges.  The functions below are therefore the plain definitions
(SURVEY 8(a) H1-H5 with alpha = the MPO element) written as loops over blocks; tests/test_oracle_abelian.py pins
them against the dense contractions of oracle/dense_tdvp.py through the embedding ``embed_*`` (blocks placed at
their sector offsets, nothing else).

Labels: (q, 0) with q = (N_up - N_dn) + 64 (N - k) on bond k (the packing of fh_inputs/abelian.py; the 0 keeps the
key shapes of the SU(2) mode).  Site states 0 |0>, 1 |up>, 2 |dn>, 3 |updn>; MPO bond states 0 I, 1 c+_up P,
2 c+_dn P, 3 c_up P, 4 c_dn P, 5 final: the bond-dimension-6 MPO of Eq. (1), oracle/dense_tdvp.dense_mpo.
"""
import numpy as np

from .dense_tdvp import dense_mpo

SITE_Q = (-64, 1, -1, 64)
MPO_Q = (0, 65, 63, -65, -63, 0)


def fuse(a, s):
    return (a[0] + SITE_Q[s], 0)


def mpo_elements(t_h, U):
    """{(w, w'): 4 x 4 matrix [s', s]} for the non-zero entries of the dense MPO; asserts that every non-zero
    element respects the charges (q_s' - q_s = q_w' - q_w)."""
    W = dense_mpo(t_h, U)
    out = {}
    for w in range(6):
        for wp in range(6):
            if np.any(W[w, wp] != 0.0):
                out[(w, wp)] = W[w, wp].copy()
                for sp in range(4):
                    for s in range(4):
                        if W[w, wp, sp, s] != 0.0:
                            assert SITE_Q[sp] - SITE_Q[s] == MPO_Q[wp] - MPO_Q[w]
    return out


def site_keys(dl, dr):
    return sorted((a, s, fuse(a, s)) for a in dl for s in range(4) if fuse(a, s) in dr)


def theta_keys(dl, dr):
    return sorted((a, s1, fuse(a, s1), s2, fuse(fuse(a, s1), s2)) for a in dl for s1 in range(4) for s2 in range(4)
                  if fuse(fuse(a, s1), s2) in dr)


def env_keys(d_bra, d_ket):
    return sorted((xp, w, x) for xp in d_bra for w in range(6) for x in d_ket if xp[0] == x[0] + MPO_Q[w])


def boundary_left():
    return {((0, 0), 0, (0, 0)): np.ones((1, 1), dtype=complex)}


def boundary_right():
    return {((0, 0), 5, (0, 0)): np.ones((1, 1), dtype=complex)}


def _acc(out, key, val):
    out[key] = val if key not in out else out[key] + val


def env_update_left(Lenv, A, W):
    """H4: L'[c',w',c] = sum W[w,w'][s',s] A[a',s',c']^dagger L[a',w,a] A[a,s,c]."""
    out = {}
    for (ap, w, a), Lb in Lenv.items():
        for (a2, s, c), Ab in A.items():
            if a2 != a:
                continue
            X = Lb @ Ab
            for (w2, wp), M in W.items():
                if w2 != w:
                    continue
                for sp in range(4):
                    if M[sp, s] == 0.0:
                        continue
                    kp = (ap, sp, fuse(ap, sp))
                    if kp in A:
                        _acc(out, (kp[2], wp, c), M[sp, s] * (A[kp].conj().T @ X))
    return dict(sorted(out.items()))


def env_update_right(Renv, A, W):
    """H5: R'[c',w,c] = sum W[w,w'][s',s] conj(A[c',s',b']) R[b',w',b] A[c,s,b]^T."""
    out = {}
    for (bp, wp, b), Rb in Renv.items():
        for (c, s, b2), Ab in A.items():
            if b2 != b:
                continue
            Y = Rb @ Ab.T
            for (w, wp2), M in W.items():
                if wp2 != wp:
                    continue
                for sp in range(4):
                    if M[sp, s] == 0.0:
                        continue
                    for (cp, sp2, bp2), Apb in A.items():
                        if sp2 == sp and bp2 == bp and cp[0] == c[0] + MPO_Q[w]:
                            _acc(out, (cp, w, c), M[sp, s] * (Apb.conj() @ Y))
    return dict(sorted(out.items()))


def heff2_apply(Lenv, Renv, theta, W1, W2):
    """H1 + H2: out[a',s1',c',s2',b'] = sum W1[wl,wm][s1',s1] W2[wm,wr][s2',s2] L[a',wl,a] theta[a,s1,c,s2,b] R[b',wr,b]^T."""
    out = {k: np.zeros_like(v) for k, v in theta.items()}
    for (ap, wl, a), Lb in Lenv.items():
        for (a2, s1, c, s2, b), T in theta.items():
            if a2 != a:
                continue
            X = Lb @ T
            for (w1, wm), M1 in W1.items():
                if w1 != wl:
                    continue
                for s1p in range(4):
                    if M1[s1p, s1] == 0.0:
                        continue
                    for (wm2, wr), M2 in W2.items():
                        if wm2 != wm:
                            continue
                        for s2p in range(4):
                            if M2[s2p, s2] == 0.0:
                                continue
                            cp = fuse(ap, s1p)
                            bp = fuse(cp, s2p)
                            rk = (bp, wr, b)
                            ok = (ap, s1p, cp, s2p, bp)
                            if rk in Renv and ok in out:
                                out[ok] = out[ok] + M1[s1p, s1] * M2[s2p, s2] * (X @ Renv[rk].T)
    return out


def heff1_apply(Lenv, Renv, A, W):
    """H3: out[a',s',c'] = sum W[wl,wr][s',s] L[a',wl,a] A[a,s,c] R[c',wr,c]^T."""
    out = {k: np.zeros_like(v) for k, v in A.items()}
    for (ap, wl, a), Lb in Lenv.items():
        for (a2, s, c), Ab in A.items():
            if a2 != a:
                continue
            X = Lb @ Ab
            for (w1, wr), M in W.items():
                if w1 != wl:
                    continue
                for sp in range(4):
                    if M[sp, s] == 0.0:
                        continue
                    cp = fuse(ap, sp)
                    rk, ok = (cp, wr, c), (ap, sp, cp)
                    if rk in Renv and ok in out:
                        out[ok] = out[ok] + M[sp, s] * (X @ Renv[rk].T)
    return out


def inner(x, y):
    return sum(np.vdot(v, y[k]) for k, v in x.items())


# ------------------------------------------------------------------ dense embedding (pins)
def offsets(dims):
    off, n = {}, 0
    for sec in sorted(dims):
        off[sec] = n
        n += dims[sec]
    return off, n


def embed_site(A, dl, dr):
    ol, nl = offsets(dl)
    orr, nr = offsets(dr)
    out = np.zeros((nl, 4, nr), dtype=complex)
    for (a, s, c), blk in A.items():
        out[ol[a]:ol[a] + dl[a], s, orr[c]:orr[c] + dr[c]] = blk
    return out


def embed_theta(th, dl, dr):
    ol, nl = offsets(dl)
    orr, nr = offsets(dr)
    out = np.zeros((nl, 4, 4, nr), dtype=complex)
    for (a, s1, c, s2, b), blk in th.items():
        out[ol[a]:ol[a] + dl[a], s1, s2, orr[b]:orr[b] + dr[b]] = blk
    return out


def embed_env(E, d_bra, d_ket):
    ob, nb = offsets(d_bra)
    ok, nk = offsets(d_ket)
    out = np.zeros((nb, 6, nk), dtype=complex)
    for (xp, w, x), blk in E.items():
        out[ob[xp]:ob[xp] + d_bra[xp], w, ok[x]:ok[x] + d_ket[x]] = blk
    return out


# ------------------------------------------------------------------ task lists (H0), same canonical order as symm.py
def heff2_tasks(L_keys, R_keys, th_keys, W1, W2):
    """Two-stage task lists of the two-site apply in the order oracle/symm.heff2_tasks defines (O-S step 5):
    stage 1  Z[a',s1',c',w_m; c,s2,b] = sum_{(w_l,a,s1)} W1[w_l,w_m][s1',s1] L[a',w_l,a] theta[a,s1,c,s2,b],
    stage 2  out[a',s1',c',s2',b']    = sum_{(c,s2,b,w_m,w_r)} W2[w_m,w_r][s2',s2] Z[...] R[b',w_r,b]^T,
    intermediates that no stage-2 task reads dropped (reading A-17).  alpha = the MPO element (recoupling
    coefficient 1)."""
    by_a = {}
    for k in th_keys:
        by_a.setdefault(k[0], []).append(k)
    st1 = {}
    for ek in L_keys:
        ap, w, a = ek
        for kk in by_a.get(a, ()):
            s = kk[1]
            for (w1, wp), M in W1.items():
                if w1 != w:
                    continue
                for sp in range(4):
                    if M[sp, s] != 0.0:
                        st1.setdefault((ap, sp, fuse(ap, sp), wp) + tuple(kk[2:]), []).append((ek, kk, float(M[sp, s])))
    for z in st1:
        st1[z].sort(key=lambda t: (t[0][1], t[0][2], t[1][1]))
    st1 = dict(sorted(st1.items()))
    out_set = set(th_keys)
    by_b = {}
    for rk in R_keys:
        by_b.setdefault(rk[2], []).append(rk)
    st2 = {}
    for zkey in st1:
        ap, s1p, cp, wm, c, s2, b = zkey
        for rk in by_b.get(b, ()):
            bp, wr, _ = rk
            if (wm, wr) not in W2:
                continue
            for s2p in range(4):
                okey = (ap, s1p, cp, s2p, bp)
                al = W2[(wm, wr)][s2p, s2]
                if al != 0.0 and okey in out_set:
                    st2.setdefault(okey, []).append((zkey, rk, float(al)))
    for o in st2:
        st2[o].sort(key=lambda t: (t[0][4], t[0][5], t[0][6], t[0][3], t[1][1]))
    used = {seg[0] for segs in st2.values() for seg in segs}
    st1 = {z: segs for z, segs in st1.items() if z in used}
    return st1, dict(sorted(st2.items()))


def heff2_flops(st1, st2, dl, dr):
    f = 0
    for z, segs in st1.items():
        for (ap, w, a), kk, _ in segs:
            f += 8 * dl[ap] * dl[a] * dr[kk[4]]
    for o, segs in st2.items():
        for zk, (bp, wr, b), _ in segs:
            f += 8 * dl[zk[0]] * dr[b] * dr[bp]
    return f
