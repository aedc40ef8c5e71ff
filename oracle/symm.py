"""O-S: symmetric (U(1) x SU(2)) block-sparse reference for the TDVP hot path.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Plain loops over Python dicts keyed by
label tuples; every reduced object can be expanded to a dense tensor with ``embed_*``
("dense embedding with coefficients expanded") and compared with oracle/dense_tdvp.py.

The paper only says that "each multiplet -> one reduced matrix element" via the
Wigner-Eckart theorem and that bond spaces decompose as Eq. (7)
(PAPER.md:210-214); the concrete conventions are the readings F-1..F-7 of DESIGN.md:

 * sector label (q, tj): q = 2 S^z = N_up - N_dn (integer), tj = 2 T (doubled pseudospin)
   -- U(1)_spin x SU(2)_charge, PAPER.md:41, 208 (reading A-1);
 * site multiplets s: 0 = (+1, 0) |up>,  1 = (-1, 0) |dn>,
   2 = (0, 1/2) with m=-1/2 -> |0>, m=+1/2 -> eps_i |updn>   (F-2);
 * MPO bond multiplets w: 0 = S (0,0), 1 = P (+1,1/2), 2 = M (-1,1/2), 3 = F (0,0)
   (reduced bond dimension W = 4);
 * dense structures (F-4):
     A^{sig}[(a m al),(c n ga)]      = A[a,s,c][al,ga]   C(a m, s sig | c n)
     L[(a' m' al'),(w mu),(a m al)]  = L[a',w,a][al',al] C(a m, k_w mu | a' m')
     R[(b' m' be'),(w mu),(b m be)]  = R[b',w,b][be',be] C(b m, k_w mu | b' m')
     W^{sig' sig}[(w mu),(w' mu')]   = W[w,w'][s',s] sum_rho C(s sig, r rho | s' sig') C(k_w mu, r rho | k_w' mu')
     theta = theta[a,s1,c,s2,b][al,be] C(a m, s1 sig1 | c n) C(c n, s2 sig2 | b m_b)   (summed over n)
"""
from math import sqrt

import numpy as np

from . import fermi
from .su2 import cg, coef_left, coef_right

SITE = ((1, 0), (-1, 0), (0, 1))              # (q, tj) of the site multiplets s = 0, 1, 2
MPOB = ((0, 0), (1, 1), (-1, 1), (0, 0))      # (q, tk) of the MPO bond multiplets S, P, M, F
ALPHA_ZERO = 1e-12                            # |alpha| below this counts as "exactly 0" (A-14)


def triangle(t1, t2, t3):
    return abs(t1 - t2) <= t3 <= t1 + t2 and (t1 + t2 + t3) % 2 == 0


def ms(tj):
    return list(range(-tj, tj + 1, 2))


# ------------------------------------------------------------------ site operators (F-2)
def site_vectors(eps):
    """Dense 4-vectors of the reduced-basis states (s, tm): |up>, |dn>, |0>, eps|updn>."""
    e = np.eye(4)
    return {(0, 0): e[1], (1, 0): e[2], (2, -1): e[0], (2, 1): eps * e[3]}


def _reduce(components, tr, eps):
    """Wigner-Eckart extraction: components = {trho: 4x4 matrix}.  Returns the 3x3 reduced
    matrix red[s', s] with <s' sig'|O_rho|s sig> = red[s',s] C(s sig, r rho | s' sig'),
    asserting that the ratio is the same for every component."""
    vec = site_vectors(eps)
    red = np.zeros((3, 3))
    seen = np.zeros((3, 3), dtype=bool)
    for (sp, tsigp), vp in vec.items():
        for (s, tsig), v in vec.items():
            for trho, O in components.items():
                el = vp @ O @ v
                c = cg(SITE[s][1], tsig, tr, trho, SITE[sp][1], tsigp)
                if abs(c) < 1e-14:
                    assert abs(el) < 1e-14, "operator is not a rank-r tensor operator"
                    continue
                r = el / c
                if seen[sp, s]:
                    assert abs(red[sp, s] - r) < 1e-13, "Wigner-Eckart ratio not constant"
                red[sp, s] = r
                seen[sp, s] = True
    return red


def reduced_site_ops(eps):
    """Reduced matrices of the site operators on a site with sublattice sign eps (F-2)."""
    cu, cd, P = fermi.C_UP, fermi.C_DN, fermi.PAR
    psi_p = {1: cu.T, -1: eps * cd}            # Psi^+ (q=+1): mu=+1/2: c^dag_up, mu=-1/2: eps c_dn
    psi_m = {1: cd.T, -1: -eps * cu}           # Psi^- (q=-1): mu=+1/2: c^dag_dn, mu=-1/2: -eps c_up
    return dict(
        psi_p=_reduce(psi_p, 1, eps), psi_m=_reduce(psi_m, 1, eps),
        psi_p_par=_reduce({k: v @ P for k, v in psi_p.items()}, 1, eps),
        psi_m_par=_reduce({k: v @ P for k, v in psi_m.items()}, 1, eps),
        one=_reduce({0: fermi.ID4}, 0, eps), p_d=_reduce({0: fermi.P_D}, 0, eps),
        sz=_reduce({0: fermi.SZ}, 0, eps))


def mpo_reduced(site, t_h, U):
    """Reduced MPO W_i (F-3): dict {(w, w'): (tr, red[s', s])} for 0-based site index.

    H_sym = hopping + (U/2) sum_i P_D,i (reading A-2) with the bond term
    -t_h eps_i sqrt2 { [Psi^+_i P x Psi^-_{i+1}]^0 - [Psi^-_i P x Psi^+_{i+1}]^0 }.
    """
    eps = (-1) ** site
    eps_prev = -eps
    o = reduced_site_ops(eps)
    r2 = sqrt(2.0)
    return {
        (0, 0): (0, o["one"]), (3, 3): (0, o["one"]), (0, 3): (0, 0.5 * U * o["p_d"]),
        (0, 1): (1, o["psi_p_par"]), (0, 2): (1, o["psi_m_par"]),
        (1, 3): (1, -t_h * eps_prev * r2 * o["psi_m"]),
        (2, 3): (1, +t_h * eps_prev * r2 * o["psi_p"]),
    }


# ------------------------------------------------------------------ bookkeeping (Eqs. 8-10)
def chi_full(dims):
    """Eq. (8) PAPER.md:218."""
    return sum(d * (tj + 1) for (q, tj), d in dims.items())


def chi_su2(dims):
    """Eq. (10) PAPER.md:222."""
    return sum(dims.values())


def d_max(dims):
    """Eq. (9) PAPER.md:220."""
    return max(dims.values())


def fuse(a, s):
    """Sectors c with a (x) s -> c."""
    qs, ts = SITE[s]
    return [(a[0] + qs, tc) for tc in range(abs(a[1] - ts), a[1] + ts + 1, 2)]


def theta_keys(dims_l, dims_r):
    """All fusion-allowed two-site keys (a, s1, c, s2, b), canonical (sorted) order."""
    keys = []
    for a in sorted(dims_l):
        for s1 in range(3):
            for c in fuse(a, s1):
                for s2 in range(3):
                    for b in fuse(c, s2):
                        if b in dims_r:
                            keys.append((a, s1, c, s2, b))
    return sorted(keys)


def site_keys(dims_l, dims_r):
    """All fusion-allowed one-site keys (a, s, c)."""
    keys = []
    for a in sorted(dims_l):
        for s in range(3):
            for c in fuse(a, s):
                if c in dims_r:
                    keys.append((a, s, c))
    return sorted(keys)


def env_keys(dims_bra, dims_ket):
    """All allowed environment keys (x', w, x): q_x' = q_x + q_w, triangle(x, k_w, x')."""
    keys = []
    for xp in sorted(dims_bra):
        for w in range(4):
            qw, tk = MPOB[w]
            for x in sorted(dims_ket):
                if xp[0] == x[0] + qw and triangle(x[1], tk, xp[1]):
                    keys.append((xp, w, x))
    return sorted(keys)


# ------------------------------------------------------------------ dense embedding (F-4)
def bond_offsets(dims):
    """Dense bond basis: sectors sorted, then m ascending, then degeneracy index."""
    off, n = {}, 0
    for sec in sorted(dims):
        off[sec] = n
        n += (sec[1] + 1) * dims[sec]
    return off, n


def _rows(off, dims, sec, tm):
    d = dims[sec]
    start = off[sec] + ((tm + sec[1]) // 2) * d
    return slice(start, start + d)


def embed_site(A, dims_l, dims_r, site):
    vec = site_vectors((-1) ** site)
    offl, nl = bond_offsets(dims_l)
    offr, nr = bond_offsets(dims_r)
    out = np.zeros((nl, 4, nr), dtype=complex)
    for (a, s, c), blk in A.items():
        for tm in ms(a[1]):
            for tsig in ms(SITE[s][1]):
                tn = tm + tsig
                x = cg(a[1], tm, SITE[s][1], tsig, c[1], tn)
                if x == 0.0:
                    continue
                v = vec[(s, tsig)]
                for p in range(4):
                    if v[p] != 0.0:
                        out[_rows(offl, dims_l, a, tm), p, _rows(offr, dims_r, c, tn)] += x * v[p] * blk
    return out


def embed_theta(theta, dims_l, dims_r, site):
    """Two-site tensor on sites (site, site+1) -> dense (chi_l, 4, 4, chi_r)."""
    v1 = site_vectors((-1) ** site)
    v2 = site_vectors((-1) ** (site + 1))
    offl, nl = bond_offsets(dims_l)
    offr, nr = bond_offsets(dims_r)
    out = np.zeros((nl, 4, 4, nr), dtype=complex)
    for (a, s1, c, s2, b), blk in theta.items():
        for tm in ms(a[1]):
            for t1 in ms(SITE[s1][1]):
                tn = tm + t1
                x1 = cg(a[1], tm, SITE[s1][1], t1, c[1], tn)
                if x1 == 0.0:
                    continue
                for t2 in ms(SITE[s2][1]):
                    tmb = tn + t2
                    x2 = cg(c[1], tn, SITE[s2][1], t2, b[1], tmb)
                    if x2 == 0.0:
                        continue
                    for p1 in range(4):
                        for p2 in range(4):
                            f = x1 * x2 * v1[(s1, t1)][p1] * v2[(s2, t2)][p2]
                            if f != 0.0:
                                out[_rows(offl, dims_l, a, tm), p1, p2,
                                    _rows(offr, dims_r, b, tmb)] += f * blk
    return out


MPO_DENSE_OFF = {0: 0, 1: 1, 2: 3, 3: 5}      # S, P(-1/2,+1/2), M(-1/2,+1/2), F


def _mpo_index(w, tmu):
    return MPO_DENSE_OFF[w] + (tmu + MPOB[w][1]) // 2


def embed_env(E, dims_bra, dims_ket):
    """Environment {(x', w, x)} -> dense (chi', 6, chi)."""
    offb, nb = bond_offsets(dims_bra)
    offk, nk = bond_offsets(dims_ket)
    out = np.zeros((nb, 6, nk), dtype=complex)
    for (xp, w, x), blk in E.items():
        tk = MPOB[w][1]
        for tm in ms(x[1]):
            for tmu in ms(tk):
                tmp = tm + tmu
                c = cg(x[1], tm, tk, tmu, xp[1], tmp)
                if c != 0.0:
                    out[_rows(offb, dims_bra, xp, tmp), _mpo_index(w, tmu),
                        _rows(offk, dims_ket, x, tm)] += c * blk
    return out


def embed_mpo(W, site):
    """Reduced MPO -> dense (6, 6, 4, 4) = [w_left, w_right, s_out, s_in]."""
    vec = site_vectors((-1) ** site)
    out = np.zeros((6, 6, 4, 4))
    for (w, wp), (tr, red) in W.items():
        tk, tkp = MPOB[w][1], MPOB[wp][1]
        for (sp, tsigp), vp in vec.items():
            for (s, tsig), v in vec.items():
                if red[sp, s] == 0.0:
                    continue
                for trho in ms(tr):
                    c1 = cg(SITE[s][1], tsig, tr, trho, SITE[sp][1], tsigp)
                    if c1 == 0.0:
                        continue
                    for tmu in ms(tk):
                        tmup = tmu + trho
                        c2 = cg(tk, tmu, tr, trho, tkp, tmup)
                        if c2 != 0.0:
                            out[_mpo_index(w, tmu), _mpo_index(wp, tmup)] += (
                                red[sp, s] * c1 * c2 * np.outer(vp, v))
    return out


# ------------------------------------------------------------------ task lists (H0)
def _alpha_left(a, s, c, w, wp, ap, sp, cp, W):
    """alpha = coefL(a,s,c; k_w,r,k_w'; a',s',c') * W[w,w'][s',s]  (F-5, H1-H4)."""
    ent = W.get((w, wp))
    if ent is None:
        return 0.0
    tr, red = ent
    if red[sp, s] == 0.0:
        return 0.0
    x = coef_left(a[1], SITE[s][1], c[1], MPOB[w][1], tr, MPOB[wp][1], ap[1], SITE[sp][1], cp[1])
    return x * red[sp, s]


def _alpha_right(c, s, b, w, wp, cp, sp, bp, W):
    """alpha_R = coefR(c,s,b; k_w,r,k_w'; c',s',b') * W[w,w'][s',s]  (F-5, H5)."""
    ent = W.get((w, wp))
    if ent is None:
        return 0.0
    tr, red = ent
    if red[sp, s] == 0.0:
        return 0.0
    x = coef_right(c[1], SITE[s][1], b[1], MPOB[w][1], tr, MPOB[wp][1], cp[1], SITE[sp][1], bp[1])
    return x * red[sp, s]


def left_contraction_tasks(env_keys_, ket_keys, W, dims_out_ok=None):
    """Generic 'stage-1' enumeration used by H1, H3, H4.

    env_keys_: keys (a', w, a) of a left-type environment; ket_keys: keys whose first two
    entries are (a, s) and third entry the fused sector c (one-site keys (a,s,c) or two-site
    keys (a,s1,c,s2,b)).  Returns {zkey: [(env_key, ket_key, alpha), ...]} with
    zkey = (a', s', c', w') + ket_key[2:]  -- i.e. the ket's (a, s) replaced by the bra-side
    (a', s', c') and the outgoing MPO multiplet w', the ket's remaining labels kept.
    Segments sorted by (w, a, s); zero-alpha tasks omitted.
    """
    by_a = {}
    for k in ket_keys:
        by_a.setdefault(k[0], []).append(k)
    out = {}
    for ek in env_keys_:
        ap, w, a = ek
        for kk in by_a.get(a, ()):
            s, c = kk[1], kk[2]
            for wp in range(4):
                if (w, wp) not in W:
                    continue
                for sp in range(3):
                    for cp in fuse(ap, sp):
                        if cp[0] != c[0] + MPOB[wp][0] or not triangle(c[1], MPOB[wp][1], cp[1]):
                            continue
                        al = _alpha_left(a, s, c, w, wp, ap, sp, cp, W)
                        if abs(al) < ALPHA_ZERO:
                            continue
                        zkey = (ap, sp, cp, wp) + tuple(kk[2:])
                        out.setdefault(zkey, []).append((ek, kk, al))
    for z in out:
        out[z].sort(key=lambda t: (t[0][1], t[0][2], t[1][1]))
    return dict(sorted(out.items()))


def heff2_tasks(L_keys, R_keys, th_keys, W1, W2):
    """Task lists of the two-site apply (H1 + H2), canonical order (O-S step 5).

    stage 1: Z[a',s1',c',w_m; c,s2,b] = sum alpha1 L[a',w_l,a] theta[a,s1,c,s2,b]
    stage 2: out[a',s1',c',s2',b']    = sum alpha2 Z[a',s1',c',w_m; c,s2,b] R[b',w_r,b]^T
    """
    st1 = left_contraction_tasks(L_keys, th_keys, W1)
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
            for s2p in range(3):
                okey = (ap, s1p, cp, s2p, bp)
                if okey not in out_set:
                    continue
                al = _alpha_left(c, s2, b, wm, wr, cp, s2p, bp, W2)
                if abs(al) < ALPHA_ZERO:
                    continue
                st2.setdefault(okey, []).append((zkey, rk, al))
    for o in st2:
        st2[o].sort(key=lambda t: (t[0][4], t[0][5], t[0][6], t[0][3], t[1][1]))
    # Reading A-17: an intermediate block Z[a',s1',c',w_m; c,s2,b] that no term of H2 reads
    # (W_{i+1}[w_m, w_r; s2', s2] vanishes for every (w_r, s2'), e.g. w_m = P with s2 = down) contributes
    # nothing to H_eff theta; it is not formed and its tasks are not part of the list (nor of the flop count).
    used = {seg[0] for segs in st2.values() for seg in segs}
    st1 = {z: segs for z, segs in st1.items() if z in used}
    return st1, dict(sorted(st2.items()))


def heff1_tasks(L_keys, R_keys, a_keys, W):
    """One-site apply (H3): stage 1 X[a',s',c',w'; c] = sum alpha L[a',w,a] A[a,s,c];
    stage 2 out[a',s',c'] = sum X[a',s',c',w'; c] R[c',w',c]^T  (alpha carried by stage 1)."""
    st1 = left_contraction_tasks(L_keys, a_keys, W)
    out_set = set(a_keys)
    Rset = set(R_keys)
    st2 = {}
    for xkey in st1:
        ap, sp, cp, wp, c = xkey
        if (cp, wp, c) in Rset and (ap, sp, cp) in out_set:
            st2.setdefault((ap, sp, cp), []).append((xkey, (cp, wp, c), 1.0))
    for o in st2:
        st2[o].sort(key=lambda t: (t[0][4], t[0][3]))
    return st1, dict(sorted(st2.items()))


def env_left_tasks(L_keys, a_keys, W):
    """H4: stage 1 as H3; stage 2 L'[c',w',c] = sum A[a',s',c']^dagger X[a',s',c',w'; c]."""
    st1 = left_contraction_tasks(L_keys, a_keys, W)
    aset = set(a_keys)
    st2 = {}
    for xkey in st1:
        ap, sp, cp, wp, c = xkey
        if (ap, sp, cp) in aset:
            st2.setdefault((cp, wp, c), []).append(((ap, sp, cp), xkey, 1.0))
    for o in st2:
        st2[o].sort(key=lambda t: (t[0][0], t[0][1]))
    return st1, dict(sorted(st2.items()))


def env_right_tasks(R_keys, a_keys, W):
    """H5: stage 1 Y[c',s',w; b',... ] -- written as
         Y[c', s', b', w', b] = conj(A[c',s',b']) R[b',w',b]              (d_c' x d_b)
       stage 2 R'[c',w,c] = sum alpha_R Y[c',s',b',w',b] A[c,s,b]^T.
    """
    by_bp = {}
    for rk in R_keys:
        by_bp.setdefault(rk[0], []).append(rk)
    by_b = {}
    for ak in a_keys:
        by_b.setdefault(ak[2], []).append(ak)
    st1, st2 = {}, {}
    for akp in a_keys:
        cp, sp, bp = akp
        for rk in by_bp.get(bp, ()):
            _, wp, b = rk
            ykey = (cp, sp, bp, wp, b)
            for ak in by_b.get(b, ()):
                c, s, _ = ak
                for w in range(4):
                    if (w, wp) not in W:
                        continue
                    if cp[0] != c[0] + MPOB[w][0] or not triangle(c[1], MPOB[w][1], cp[1]):
                        continue
                    al = _alpha_right(c, s, b, w, wp, cp, sp, bp, W)
                    if abs(al) < ALPHA_ZERO:
                        continue
                    st2.setdefault((cp, w, c), []).append((ykey, ak, al))
                    st1[ykey] = [(akp, rk, 1.0)]
    for o in st2:
        st2[o].sort(key=lambda t: (t[0][1], t[0][2], t[0][3], t[1][1], t[1][2]))
    return dict(sorted(st1.items())), dict(sorted(st2.items()))


# ------------------------------------------------------------------ execution of task lists
def run_stage(tasks, lhs, rhs, op_l="n", op_r="n"):
    """out[key] = sum alpha * op_l(lhs[k1]) @ op_r(rhs[k2]) over the key's segment list."""
    out = {}
    for key, segs in tasks.items():
        acc = None
        for k1, k2, al in segs:
            x = lhs[k1]
            y = rhs[k2]
            x = {"n": x, "c": x.conj(), "h": x.conj().T}[op_l]
            y = {"n": y, "t": y.T}[op_r]
            t = al * (x @ y)
            acc = t if acc is None else acc + t
        out[key] = acc
    return out


def heff2_apply(Lenv, Renv, theta, W1, W2):
    """Two-site H_eff theta (H1 + H2).  Output has theta's key set (zero blocks filled)."""
    st1, st2 = heff2_tasks(sorted(Lenv), sorted(Renv), sorted(theta), W1, W2)
    Z = run_stage(st1, Lenv, theta)
    out = run_stage(st2, Z, Renv, "n", "t")
    for k, v in theta.items():
        if k not in out:
            out[k] = np.zeros_like(v)
    return dict(sorted(out.items()))


def heff1_apply(Lenv, Renv, A, W):
    st1, st2 = heff1_tasks(sorted(Lenv), sorted(Renv), sorted(A), W)
    X = run_stage(st1, Lenv, A)
    out = run_stage(st2, X, Renv, "n", "t")
    for k, v in A.items():
        if k not in out:
            out[k] = np.zeros_like(v)
    return dict(sorted(out.items()))


def env_update_left(Lenv, A, W):
    st1, st2 = env_left_tasks(sorted(Lenv), sorted(A), W)
    X = run_stage(st1, Lenv, A)
    return run_stage(st2, A, X, "h", "n")


def env_update_right(Renv, A, W):
    st1, st2 = env_right_tasks(sorted(Renv), sorted(A), W)
    Y = run_stage(st1, A, Renv, "c", "n")
    return run_stage(st2, Y, A, "n", "t")


def inner(x, y):
    """F-6 weighted inner product; the last label of every key is the right bond sector."""
    tot = 0.0 + 0.0j
    for k, v in x.items():
        tot += (k[-1][1] + 1) * np.vdot(v, y[k])
    return tot


def canonical_weight(c, b):
    """F-6: a site tensor A[c,s,b] is right-canonical when sum_{s,b} w(c,b)^2 A A^dagger = 1 with
    w(c,b)^2 = (2 j_b + 1) / (2 j_c + 1): a multiplet of spin j stands for 2j+1 states (Eq. (8))."""
    return np.sqrt((b[1] + 1) / (c[1] + 1))


def boundary_left():
    return {((0, 0), 0, (0, 0)): np.ones((1, 1), dtype=complex)}


def boundary_right():
    return {((0, 0), 3, (0, 0)): np.ones((1, 1), dtype=complex)}


# ------------------------------------------------------------------ merge / SVD split (H8, H9)
def merge(A1, A2):
    """theta[a,s1,c,s2,b] = A1[a,s1,c] @ A2[c,s2,b]."""
    by_c = {}
    for k in A2:
        by_c.setdefault(k[0], []).append(k)
    th = {}
    for (a, s1, c), x in A1.items():
        for (_, s2, b) in by_c.get(c, ()):
            th[(a, s1, c, s2, b)] = x @ A2[(c, s2, b)]
    return dict(sorted(th.items()))


def pack(theta, dims_l, dims_r):
    """H8: per middle sector c, M_c[(a,s1,al),(s2,b,be)] = theta[a,s1,c,s2,b] sqrt((2j_b+1)/(2j_c+1)).
    Returns {c: (M_c, row_layout, col_layout)} with layouts [(key_part, offset, dim)]."""
    rows, cols = {}, {}
    for (a, s1, c, s2, b) in sorted(theta):
        rows.setdefault(c, [])
        cols.setdefault(c, [])
        if (a, s1) not in rows[c]:
            rows[c].append((a, s1))
        if (s2, b) not in cols[c]:
            cols[c].append((s2, b))
    out = {}
    for c in sorted(rows):
        rl, n = [], 0
        for (a, s1) in sorted(rows[c]):
            rl.append(((a, s1), n, dims_l[a]))
            n += dims_l[a]
        cl, m = [], 0
        for (s2, b) in sorted(cols[c], key=lambda t: (t[0], t[1])):
            cl.append(((s2, b), m, dims_r[b]))
            m += dims_r[b]
        M = np.zeros((n, m), dtype=complex)
        for (a, s1), ro, rd in rl:
            for (s2, b), co, cd in cl:
                blk = theta.get((a, s1, c, s2, b))
                if blk is not None:
                    M[ro:ro + rd, co:co + cd] = blk * sqrt((b[1] + 1) / (c[1] + 1))
        out[c] = (M, rl, cl)
    return out


def svd_split(theta, dims_l, dims_r, chi_max_full, eps_trunc, direction):
    """H9 + F-7: block-wise SVD, truncation by reading A-6, unpack.

    direction 'right': A1 = U (left-canonical), A2 = S V^dagger ...;  'left': A1 = U S,
    A2 = V^dagger ... (right-canonical).  Returns (A1, A2, dims_mid, info).
    """
    from .dense_tdvp import truncate_rule
    packed = pack(theta, dims_l, dims_r)
    secs = sorted(packed)
    usv = {}
    for c in secs:
        M = packed[c][0]
        usv[c] = np.linalg.svd(M, full_matrices=False)
    keep, disc = truncate_rule([usv[c][1] for c in secs], [c[1] + 1 for c in secs],
                               chi_max_full, eps_trunc)
    A1, A2, dims_mid = {}, {}, {}
    for c, k in zip(secs, keep):
        if k == 0:
            continue
        U_, s, Vh = usv[c]
        U_, s, Vh = U_[:, :k], s[:k], Vh[:k]
        dims_mid[c] = k
        if direction == "right":
            Vh = s[:, None] * Vh
        else:
            U_ = U_ * s[None, :]
        for (a, s1), ro, rd in packed[c][1]:
            A1[(a, s1, c)] = U_[ro:ro + rd].copy()
        for (s2, b), co, cd in packed[c][2]:
            A2[(c, s2, b)] = Vh[:, co:co + cd] * sqrt((c[1] + 1) / (b[1] + 1))
    info = dict(discarded=disc, svals={c: usv[c][1] for c in secs}, keep=dict(zip(secs, keep)))
    return dict(sorted(A1.items())), dict(sorted(A2.items())), dims_mid, info


# ------------------------------------------------------------------ one-site TDVP pieces (NEXT-1)
def embed_bond(C, dims_bra, dims_ket):
    """Bond matrix {c: (d'_c x d_c)} (an SU(2) scalar: diagonal in the sector and in m) -> dense."""
    offb, nb = bond_offsets(dims_bra)
    offk, nk = bond_offsets(dims_ket)
    out = np.zeros((nb, nk), dtype=complex)
    for c, blk in C.items():
        for tm in ms(c[1]):
            out[_rows(offb, dims_bra, c, tm), _rows(offk, dims_ket, c, tm)] += blk
    return out


def heff0_tasks(L_keys, R_keys, c_keys):
    """Zero-site apply: out[c'] = sum_{(c, w)} L[c',w,c] C[c] R[c',w,c]^T.  The recoupling coefficient
    is 1: with L = L[c',w,c] C(j_c m, k_w mu | j_c' m') and R likewise (F-4), the sum over m and mu of
    the two Clebsch-Gordan coefficients is delta_{m' n'} (CG orthogonality).  Stage 1: X[c',w,c] =
    L[c',w,c] C[c]; stage 2: out[c'] = sum X[c',w,c] R[c',w,c]^T, segments ordered by (c, w)."""
    Rset = set(R_keys)
    cset = set(c_keys)
    st1, st2 = {}, {}
    for (cp, w, c) in L_keys:
        if c in cset and cp in cset and (cp, w, c) in Rset:
            st1[(cp, w, c)] = [((cp, w, c), c, 1.0)]
            st2.setdefault(cp, []).append(((cp, w, c), (cp, w, c), 1.0))
    for o in st2:
        st2[o].sort(key=lambda t: (t[0][2], t[0][1]))
    return dict(sorted(st1.items())), dict(sorted(st2.items()))


def heff0_apply(Lenv, Renv, C):
    st1, st2 = heff0_tasks(sorted(Lenv), sorted(Renv), sorted(C))
    X = run_stage(st1, Lenv, C)
    out = run_stage(st2, X, Renv, "n", "t")
    for c, v in C.items():
        if c not in out:
            out[c] = np.zeros_like(v)
    return out


def split_site_right_moving(A, dims_l, dims_r):
    """A[a,s,c] = Q[a,s,c'] C[c]: per right sector c the stacked rows (a, s, alpha) are decomposed by
    an SVD, Q = U (left-canonical), C = S V^dagger (k_c x d_c), k_c = min(rows, d_c).  No truncation.
    Returns (Q, C, new dims of the bond between them)."""
    by_c = {}
    for k in sorted(A):
        by_c.setdefault(k[2], []).append(k)
    Q, C, dims_new = {}, {}, {}
    for c, keys in by_c.items():
        M = np.vstack([A[k] for k in keys])
        U_, sv, Vh = np.linalg.svd(M, full_matrices=False)
        dims_new[c] = U_.shape[1]
        C[c] = sv[:, None] * Vh
        ro = 0
        for k in keys:
            Q[k] = U_[ro:ro + A[k].shape[0]].copy()
            ro += A[k].shape[0]
    return dict(sorted(Q.items())), dict(sorted(C.items())), dims_new


def split_site_left_moving(A, dims_l, dims_r):
    """A[a,s,b] = C[a] Q[a',s,b]: per left sector a the blocks are laid side by side with the weight
    sqrt((2j_b+1)/(2j_a+1)) (F-6: right-canonical means sum_{s,b} (2j_b+1)/(2j_a+1) Q Q^dagger = 1),
    SVD, C = U S (d_a x k_a), Q = V^dagger with the weight undone."""
    by_a = {}
    for k in sorted(A):
        by_a.setdefault(k[0], []).append(k)
    Q, C, dims_new = {}, {}, {}
    for a, keys in by_a.items():
        M = np.hstack([A[k] * sqrt((k[2][1] + 1) / (a[1] + 1)) for k in keys])
        U_, sv, Vh = np.linalg.svd(M, full_matrices=False)
        dims_new[a] = Vh.shape[0]
        C[a] = U_ * sv[None, :]
        co = 0
        for k in keys:
            n = A[k].shape[1]
            Q[k] = Vh[:, co:co + n] * sqrt((a[1] + 1) / (k[2][1] + 1))
            co += n
    return dict(sorted(Q.items())), dict(sorted(C.items())), dims_new


def absorb_left(C, A):
    """A'[c,s,b] = C[c] A[c,s,b]."""
    return {k: C[k[0]] @ v for k, v in A.items()}


def absorb_right(A, C):
    """A'[a,s,c] = A[a,s,c] C[c]."""
    return {k: v @ C[k[2]] for k, v in A.items()}


# ------------------------------------------------------------------ integer task tuples (A-14)
def task_tuples(tasks, out_order, lhs_order, rhs_order):
    """Flatten {out_key: [(k1, k2, alpha)]} to int32 tuples (out_id, lhs_id, rhs_id) + alphas,
    ids = positions in the given canonical key orders.  Bit-exact comparison target for the
    CUDA library's host layer."""
    oid = {k: i for i, k in enumerate(out_order)}
    lid = {k: i for i, k in enumerate(lhs_order)}
    rid = {k: i for i, k in enumerate(rhs_order)}
    tup, al = [], []
    for key, segs in tasks.items():
        for k1, k2, a in segs:
            tup.append((oid[key], lid[k1], rid[k2]))
            al.append(a)
    return np.array(tup, dtype=np.int32).reshape(-1, 3), np.array(al, dtype=np.float64)


def heff2_flops(st1, st2, dims_l, dims_r):
    """sum 8 m n k over the two task lists (SURVEY 8(d) 'algorithmic work per unit')."""
    f = 0
    for z, segs in st1.items():
        for (ap, w, a), kk, _ in segs:
            f += 8 * dims_l[ap] * dims_l[a] * dims_r[kk[4]]
    for o, segs in st2.items():
        for zk, (bp, wr, b), _ in segs:
            f += 8 * dims_l[zk[0]] * dims_r[b] * dims_r[bp]
    return f
