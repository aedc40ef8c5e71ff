"""Oracle-side assembly of the synthetic workloads for the parity tests (tests/ only).

Mirrors paper_2606_04771_b200/harness.py, but every contraction is done by ``oracle/`` on the
CPU.  The two sides share only the seeded inputs of ``fh_inputs``.
"""
import numpy as np

import fh_inputs as fi
from oracle import symm


def rel_err(x, y, weighted=True):
    """Relative Frobenius error between two block dicts under the F-6 weighted norm."""
    num = den = 0.0
    for k, v in y.items():
        w = (k[-1][1] + 1) if weighted else 1.0
        num += w * np.linalg.norm(x[k] - v) ** 2
        den += w * np.linalg.norm(v) ** 2
    return np.sqrt(num / den) if den > 0 else np.sqrt(num)


def env_key(row):
    return ((int(row[0]), int(row[1])), int(row[2]), (int(row[3]), int(row[4])))


def central_bond(chi, L=60, seed=fi.SEED, profile="gaussian", table_s2_scale=(1, 1), centre=None,
                 t_h=1.0, U=4.0):
    """Oracle twin of harness.build_central_bond: returns dict(dims, Lenv, Renv, A, W)."""
    centre = L // 2 - 1 if centre is None else centre
    dims = fi.chain_dims(chi, L, profile, table_s2_scale)
    W = [symm.mpo_reduced(i, t_h, U) for i in range(L)]
    Le, Re = symm.boundary_left(), symm.boundary_right()
    A_c = {}
    for i, A, dl, dr in fi.canonical_chain(chi, centre, L, seed, dims=dims, weight=symm.canonical_weight):
        if i < centre:
            Le = symm.env_update_left(Le, A, W[i])
        elif i > centre + 1:
            Re = symm.env_update_right(Re, A, W[i])
        else:
            A_c[i] = A
    return dict(dims=dims, Lenv=Le, Renv=Re, A=A_c, W=W, centre=centre)


def heff2_selected(Lenv, Renv, theta, W1, W2, out_keys):
    """Oracle H_eff theta restricted to the output blocks `out_keys` (each output block is an
    independent sum over its own segments, SURVEY 8(c.4) last row)."""
    st1, st2 = symm.heff2_tasks(sorted(Lenv), sorted(Renv), sorted(theta), W1, W2)
    sub2 = {k: st2[k] for k in out_keys if k in st2}
    need = {seg[0] for segs in sub2.values() for seg in segs}
    sub1 = {z: st1[z] for z in need}
    Z = symm.run_stage(sub1, Lenv, theta)
    out = symm.run_stage(sub2, Z, Renv, "n", "t")
    for k in out_keys:
        if k not in out:
            out[k] = np.zeros_like(theta[k])
    return out
