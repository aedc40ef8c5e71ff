"""Workload assembly for tests and bench.py on the CUDA side: turns the seeded synthetic inputs
of ``fh_inputs`` into calls of the C-ABI library (through ``binding``).  Marshalling only: no
contraction, coefficient or decomposition is computed here, and nothing from ``oracle/`` is
imported.
"""
import numpy as np

import fh_inputs as fi

from . import binding


def site_key(row):
    return ((int(row[0]), int(row[1])), int(row[2]), (int(row[3]), int(row[4])))


def theta_key(row):
    return ((int(row[0]), int(row[1])), int(row[2]), (int(row[3]), int(row[4])), int(row[5]),
            (int(row[6]), int(row[7])))


def flatten(blocks, labels, dims, keyfn):
    """Concatenate dict blocks in the library's planned block order, checking that the
    library's layout (labels, dims) is exactly the key set and the shapes of `blocks`."""
    if len(labels) != len(blocks):
        raise ValueError("block count mismatch: library %d, input %d" % (len(labels), len(blocks)))
    parts = []
    for row, dm in zip(labels, dims):
        k = keyfn(row)
        b = blocks[k]
        if b.shape != (int(dm[0]), int(dm[1])):
            raise ValueError("shape mismatch for block %r" % (k,))
        parts.append(np.ascontiguousarray(b, dtype=np.complex128).ravel())
    return np.concatenate(parts) if parts else np.zeros(0, dtype=np.complex128)


def unflatten(vec, labels, dims, keyfn):
    out, n = {}, 0
    for row, dm in zip(labels, dims):
        sz = int(dm[0]) * int(dm[1])
        out[keyfn(row)] = vec[n:n + sz].reshape(int(dm[0]), int(dm[1]))
        n += sz
    return out


def set_site(ctx, mps, site, A, dims_l, dims_r):
    ctx.mps_set_bond(mps, site, dims_l)
    ctx.mps_set_bond(mps, site + 1, dims_r)
    lab, dm, _ = ctx.mps_site_layout(mps, site)
    ctx.mps_set_site(mps, site, flatten(A, lab, dm, site_key))


def build_central_bond(ctx, mpo, chi, L=60, seed=fi.SEED, profile="gaussian", table_s2_scale=(1, 1),
                       centre=None, keep_sites=False):
    """Config 2/3/5 recipe: stream the random canonical chain through env_update_left/right up to
    the bond (centre, centre+1), set the two centre sites, and return (mps, dims).  Site tensors
    away from the centre are dropped after use unless keep_sites."""
    centre = L // 2 - 1 if centre is None else centre
    mps = ctx.mps_create(L)
    dims = fi.chain_dims(chi, L, profile, table_s2_scale)
    for i, A, dl, dr in fi.canonical_chain(chi, centre, L, seed, dims=dims, weight=binding.fh_canonical_weight):
        set_site(ctx, mps, i, A, dl, dr)
        if i < centre:
            ctx.env_update_left(mpo, mps, i)
        elif i > centre + 1:
            ctx.env_update_right(mpo, mps, i)
        if not keep_sites and (i < centre or i > centre + 1):
            ctx.mps_drop_site(mps, i)
    return mps, dims


def to_planned(ctx, flat):
    """Host vector in the interchange format (blocks back to back in heff_layout order) -> device vector
    in the library's planned layout, converted by the library's own kernel (heff_import)."""
    import torch
    blocks = torch.from_numpy(np.ascontiguousarray(flat, dtype=np.complex128)).to(ctx.device)
    vec = torch.empty_like(blocks)
    ctx.heff_import(blocks, vec)
    return vec


def from_planned(ctx, vec):
    """Planned device vector -> host numpy vector in the interchange format (heff_export)."""
    import torch
    blocks = torch.empty_like(vec)
    ctx.heff_export(vec, blocks)
    return blocks.cpu().numpy()


def theta_vector(ctx, site, dims_l, dims_r, seed=fi.SEED):
    """Random two-site vector in the interchange format of the current plan (host numpy)."""
    lab, dm, ne = ctx.heff_layout(2)
    th = fi.theta_random(seed, site, dims_l, dims_r)
    v = flatten(th, lab, dm, theta_key)
    assert v.size == ne
    return v, lab, dm


__all__ = ["binding", "site_key", "theta_key", "flatten", "unflatten", "set_site", "build_central_bond",
           "theta_vector", "to_planned", "from_planned"]
