"""GPU parity tests (-m gpu): the CUDA path, called through the C-ABI binding, against the CPU
oracle on the same seeded inputs.  Tolerances (north_star): relative Frobenius error <= 1e-11 per
heff_apply in FP64; local observables within 1e-8 at matched chi; task tuples bit-exact."""
import os

import numpy as np
import pytest

import fh_inputs as fi
from oracle import symm, vecops
from oracle import symm_tdvp as stv
from oracle.dense_tdvp import lanczos_exp

from oracle_side import central_bond, env_key, heff2_selected, rel_err

pytestmark = pytest.mark.gpu

TOL_APPLY = 1e-11


@pytest.fixture(scope="module")
def H():
    import paper_2606_04771_b200 as pkg
    pkg.build()
    from paper_2606_04771_b200 import harness
    return harness


@pytest.fixture()
def ctx(H):
    c = H.binding.Context(1 << 30)
    yield c
    c.close()


def _torch():
    import torch
    return torch


def _dev(v):
    torch = _torch()
    return torch.from_numpy(np.ascontiguousarray(v)).cuda()


def _rand(rng, m, n):
    return rng.standard_normal((m, n)) + 1j * rng.standard_normal((m, n))


def _small_chain(rng, L, dmax):
    tabs = fi.reachable_tables(L)
    dims = [{sec: int(rng.integers(1, dmax + 1)) for sec in tabs[k]} for k in range(L + 1)]
    dims[0] = {(0, 0): 1}
    dims[L] = {(0, 0): 1}
    A = [{k: _rand(rng, dims[i][k[0]], dims[i + 1][k[2]]) for k in symm.site_keys(dims[i], dims[i + 1])}
         for i in range(L)]
    return dims, A


def _apply_gpu(H, ctx, vec_blocks, nsite):
    lab, dm, ne = ctx.heff_layout(nsite)
    keyfn = H.theta_key if nsite == 2 else H.site_key
    x = H.to_planned(ctx, H.flatten(vec_blocks, lab, dm, keyfn))
    y = _torch().empty_like(x)
    ctx.heff_apply(x, y)
    return H.unflatten(H.from_planned(ctx, y), lab, dm, keyfn)


# ------------------------------------------------------------------ small chains, every bond
@pytest.mark.parametrize("L,dmax,seed", [(4, 3, 1), (6, 5, 2), (6, 11, 3)])
def test_env_and_apply_parity_small_chain(H, ctx, L, dmax, seed):
    """Ragged tiny blocks (1..11), all reachable sector combinations: environments (H4, H5),
    two-site apply (H1+H2) on every bond and one-site apply (H3) on every site."""
    rng = np.random.default_rng(seed)
    t_h, U = 1.0, 4.0
    dims, A = _small_chain(rng, L, dmax)
    W = [symm.mpo_reduced(i, t_h, U) for i in range(L)]
    Le = [symm.boundary_left()]
    for i in range(L):
        Le.append(symm.env_update_left(Le[i], A[i], W[i]))
    Re = [None] * (L + 1)
    Re[L] = symm.boundary_right()
    for i in range(L - 1, -1, -1):
        Re[i] = symm.env_update_right(Re[i + 1], A[i], W[i])

    mpo = ctx.fh_mpo_build(L, t_h, U)
    mps = ctx.mps_create(L)
    for i in range(L):
        H.set_site(ctx, mps, i, A[i], dims[i], dims[i + 1])
    for i in range(L):
        ctx.env_update_left(mpo, mps, i)
    for i in range(L - 1, -1, -1):
        ctx.env_update_right(mpo, mps, i)
    for which, ref in ((0, Le), (1, Re)):
        for k in range(L + 1):
            lab, dm, flat = ctx.env_get(mps, which, k)
            got = H.unflatten(flat, lab, dm, env_key)
            assert sorted(got) == sorted(ref[k]), (which, k)
            assert rel_err(got, ref[k], weighted=False) < 1e-12, (which, k)
    for i in range(L - 1):
        keys = symm.theta_keys(dims[i], dims[i + 2])
        th = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]) for k in keys}
        ref = symm.heff2_apply(Le[i], Re[i + 2], th, W[i], W[i + 1])
        ctx.heff_plan(mpo, mps, i, 2)
        got = _apply_gpu(H, ctx, th, 2)
        assert rel_err(got, ref) < TOL_APPLY, i
    for i in range(L):
        ref = symm.heff1_apply(Le[i], Re[i + 1], A[i], W[i])
        ctx.heff_plan(mpo, mps, i, 1)
        got = _apply_gpu(H, ctx, A[i], 1)
        assert rel_err(got, ref) < TOL_APPLY, i
    ctx.mps_destroy(mps)


# ------------------------------------------------------------------ BASELINE config 2 at full size
def test_config2_full_size_apply_tasks_and_hermiticity(H, ctx):
    """configs[1]: L=60 central bond, chi=1024, environments contracted from the random canonical
    MPS on both sides independently; heff_apply vs O-S <= 1e-11; task tuples bit-exact; flops equal;
    H_eff Hermitian under the weighted inner product F-6."""
    chi, L = 1024, 60
    o = central_bond(chi, L)
    c = o["centre"]
    dl, dr = o["dims"][c], o["dims"][c + 2]
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps, dims = H.build_central_bond(ctx, mpo, chi, L)
    assert dims[c] == dl and dims[c + 2] == dr
    for which, k, ref in ((0, c, o["Lenv"]), (1, c + 2, o["Renv"])):
        lab, dm, flat = ctx.env_get(mps, which, k)
        got = H.unflatten(flat, lab, dm, env_key)
        assert sorted(got) == sorted(ref)
        assert rel_err(got, ref, weighted=False) < 1e-12
    ctx.heff_plan(mpo, mps, c, 2)
    # bit-exact task lists (A-14)
    Lk, Rk = sorted(o["Lenv"]), sorted(o["Renv"])
    vk = symm.theta_keys(dl, dr)
    st1, st2 = symm.heff2_tasks(Lk, Rk, vk, o["W"][c], o["W"][c + 1])
    o1 = symm.task_tuples(st1, list(st1), Lk, vk)
    o2 = symm.task_tuples(st2, vk, list(st1), Rk)
    t1, a1, n1 = ctx.heff_get_tasks(1)
    t2, a2, n2 = ctx.heff_get_tasks(2)
    assert n1 == len(st1) and n2 == len(vk)
    assert t1.shape == o1[0].shape and (t1 == o1[0]).all()
    assert t2.shape == o2[0].shape and (t2 == o2[0]).all()
    assert np.abs(a1 - o1[1]).max() < 1e-13 and np.abs(a2 - o2[1]).max() < 1e-13
    assert ctx.heff_flops() == symm.heff2_flops(st1, st2, dl, dr)
    # apply
    th = fi.theta_random(fi.SEED, c, dl, dr)
    ref = symm.heff2_apply(o["Lenv"], o["Renv"], th, o["W"][c], o["W"][c + 1])
    got = _apply_gpu(H, ctx, th, 2)
    assert rel_err(got, ref) < TOL_APPLY
    # host-buffer entry point gives the same bits as the device entry point
    lab, dm, ne = ctx.heff_layout(2)
    xin = H.flatten(th, lab, dm, H.theta_key)
    xout = np.zeros_like(xin)
    ctx.heff_apply_host(xin, xout)
    assert np.array_equal(xout, H.flatten(got, lab, dm, H.theta_key))
    # Hermiticity and inner product
    ph = fi.theta_random(fi.SEED + 1, c, dl, dr)
    x, y = H.to_planned(ctx, xin), H.to_planned(ctx, H.flatten(ph, lab, dm, H.theta_key))
    hx, hy = _torch().empty_like(x), _torch().empty_like(y)
    ctx.heff_apply(x, hx)
    ctx.heff_apply(y, hy)
    ip = ctx.heff_inner(y, x)
    assert abs(ip - symm.inner(ph, th)) < 1e-12 * max(1.0, abs(ip))
    a, b = ctx.heff_inner(y, hx), ctx.heff_inner(x, hy)
    scale = np.sqrt(abs(ctx.heff_inner(hx, hx)) * abs(ctx.heff_inner(y, y)))
    assert abs(a - np.conj(b)) < 1e-12 * scale
    ctx.mps_destroy(mps)


# ------------------------------------------------------------------ blocks that span several tiles
@pytest.mark.parametrize("den", [24, 8])
def test_apply_parity_table_s2_shape_random_envs(H, ctx, den):
    """Paper-shaped sectors (Table S2 scaled by 1/den: d_max = 72 / 216, several 64- and 32-tiles
    with ragged tails) with iid random environments given through env_set."""
    L, c = 60, 29
    even = fi.table_s2_profile(1, den)
    dl, dr = fi.neighbour_profile(even, -1), fi.neighbour_profile(even, +1)
    Lk, Rk = fi.env_block_keys(dl, dl), fi.env_block_keys(dr, dr)
    Le = fi.random_blocks(7, 1, Lk, {k: (dl[k[0]], dl[k[2]]) for k in Lk})
    Re = fi.random_blocks(7, 2, Rk, {k: (dr[k[0]], dr[k[2]]) for k in Rk})
    th = fi.theta_random(7, c, dl, dr)
    W1, W2 = symm.mpo_reduced(c, 1.0, 4.0), symm.mpo_reduced(c + 1, 1.0, 4.0)
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_create(L)
    ctx.mps_set_bond(mps, c, dl)
    ctx.mps_set_bond(mps, c + 2, dr)
    for which, bond, keys, E in ((0, c, Lk, Le), (1, c + 2, Rk, Re)):
        labels = [[k[0][0], k[0][1], k[1], k[2][0], k[2][1]] for k in keys]
        flat = np.concatenate([E[k].ravel() for k in keys])
        ctx.env_set(mps, which, bond, labels, flat)
    ctx.heff_plan(mpo, mps, c, 2)
    got = _apply_gpu(H, ctx, th, 2)
    rng = np.random.default_rng(den)
    keys = sorted(th)
    if den >= 24:
        ref = symm.heff2_apply(Le, Re, th, W1, W2)
        assert rel_err(got, ref) < TOL_APPLY
    else:
        big = sorted(keys, key=lambda k: -th[k].size)[:6]
        pick = big + [keys[i] for i in rng.choice(len(keys), 30, replace=False)]
        ref = heff2_selected(Le, Re, th, W1, W2, pick)
        for k in pick:
            den_ = max(np.linalg.norm(ref[k]), 1e-300)
            assert np.linalg.norm(got[k] - ref[k]) / den_ < TOL_APPLY, k
    ctx.mps_destroy(mps)


def _per_block_worst(got, ref):
    worst = 0.0
    for k, v in ref.items():
        worst = max(worst, np.linalg.norm(got[k] - v) / max(np.linalg.norm(v), 1e-300))
    return worst


@pytest.mark.parametrize("chi,path", [(4096, 1), (4096, 2), (1024, 2), (4096, 3)])
def test_config3_full_size_all_blocks_both_gemm_forms(H, chi, path):
    """BASELINE config 3 (chi = 4096: the workload and plan bench.py times) and config 2 (chi = 1024), complete:
    the environments L_29, R_31 are contracted on both sides independently from the seeded canonical chain (29
    chained H4 / H5 updates at full block size: blocks that span several units / tiles), then ALL output blocks of
    the two-site apply (H1 + H2), of the one-site apply on site 30 (H3) and of one more right-environment update
    (H5) are compared with the oracle, per block and globally, relative Frobenius <= 1e-11.  `path` forces the
    form of the grouped ZGEMM heff_apply uses (fh_set_option): 1 = warp units, two launches; 2 = warp-specialised
    single launch with cross-stage dependency counters and k-split tiles; 3 = warp units, both stages in one launch."""
    L, c = 60, 29
    o = central_bond(chi, L)
    dims, W = o["dims"], o["W"]
    ctx = H.binding.Context(int(max(1 << 30, 64.0 * chi * chi)))
    try:
        ctx.fh_set_option(ctx.OPT_GEMM_PATH, path)
        mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
        mps, gdims = H.build_central_bond(ctx, mpo, chi, L)
        assert [gdims[k] for k in (c, c + 1, c + 2)] == [dims[k] for k in (c, c + 1, c + 2)]
        for which, bond, ref in ((0, c, o["Lenv"]), (1, c + 2, o["Renv"])):
            lab, dm, flat = ctx.env_get(mps, which, bond)
            got = H.unflatten(flat, lab, dm, env_key)
            assert sorted(got) == sorted(ref)
            assert rel_err(got, ref, weighted=False) < 1e-11 and _per_block_worst(got, ref) < 1e-10
        # two-site apply, every block
        th = fi.theta_random(fi.SEED, c, dims[c], dims[c + 2])
        ref = symm.heff2_apply(o["Lenv"], o["Renv"], th, W[c], W[c + 1])
        ctx.heff_plan(mpo, mps, c, 2)
        assert ctx.heff_flops() == symm.heff2_flops(*symm.heff2_tasks(sorted(o["Lenv"]), sorted(o["Renv"]), sorted(th),
                                                                       W[c], W[c + 1]), dims[c], dims[c + 2])
        lab, dm, ne = ctx.heff_layout(2)
        x = H.to_planned(ctx, H.flatten(th, lab, dm, H.theta_key))
        y, y2 = _torch().empty_like(x), _torch().empty_like(x)
        ctx.heff_apply(x, y)
        ctx.heff_apply(2.0 * x, y2)
        assert bool((y2 == 2.0 * y).all())                      # exact: scaling by 2 commutes with rounding
        got = H.unflatten(H.from_planned(ctx, y), lab, dm, H.theta_key)
        assert len(got) == len(ref) == len(lab)
        e2, w2 = rel_err(got, ref), _per_block_worst(got, ref)
        # one more right-environment update (site 30) and the one-site apply on site 30
        Re30 = symm.env_update_right(o["Renv"], o["A"][c + 1], W[c + 1])
        ctx.env_update_right(mpo, mps, c + 1)
        lab, dm, flat = ctx.env_get(mps, 1, c + 1)
        gotR = H.unflatten(flat, lab, dm, env_key)
        eR = rel_err(gotR, Re30, weighted=False)
        Le30 = symm.env_update_left(o["Lenv"], o["A"][c], W[c])
        ctx.env_update_left(mpo, mps, c)
        lab, dm, flat = ctx.env_get(mps, 0, c + 1)
        eL = rel_err(H.unflatten(flat, lab, dm, env_key), Le30, weighted=False)
        ref1 = symm.heff1_apply(o["Lenv"], Re30, o["A"][c], W[c])
        ctx.heff_plan(mpo, mps, c, 1)
        got1 = _apply_gpu(H, ctx, o["A"][c], 1)
        e1, w1 = rel_err(got1, ref1), _per_block_worst(got1, ref1)
        print("chi=%d path %d: two-site %d blocks global %.2e worst block %.2e; one-site %d blocks %.2e / %.2e; "
              "env updates %.2e %.2e" % (chi, path, len(ref), e2, w2, len(ref1), e1, w1, eL, eR))
        assert e2 < TOL_APPLY and w2 < TOL_APPLY and e1 < TOL_APPLY and w1 < TOL_APPLY and eL < 1e-11 and eR < 1e-11
        ctx.mps_destroy(mps)
    finally:
        ctx.close()


@pytest.mark.parametrize("chi,nsample", [(16384, 12)])
def test_apply_parity_bench_sizes_sampled_blocks(H, chi, nsample):
    """Config 4's size (chi = 16384; chi = 4096 and 1024 are compared block by block in the test above) in
    the launch configuration of the bench (same sector profile, same plan, same unit lists; iid random
    environments through env_set so that no oracle input comes from the CUDA path).  The oracle computes
    sampled output blocks one by one (each output block is an independent sum over its own segments):
    the six largest blocks plus random ones, relative Frobenius error per block <= 1e-11; plus a
    property that holds at any size and for any environments: H(2 theta) = 2 H(theta) bit for bit
    (scaling by two commutes with every rounding; it fails if any block or k-range were skipped or
    visited twice between the two calls)."""
    L, c = 60, 29
    dims = fi.chain_dims(chi, L, "gaussian", (1, 1))
    dl, dr = dims[c], dims[c + 2]
    Lk, Rk = fi.env_block_keys(dl, dl), fi.env_block_keys(dr, dr)
    Le = fi.random_blocks(9, 1, Lk, {k: (dl[k[0]], dl[k[2]]) for k in Lk})
    Re = fi.random_blocks(9, 2, Rk, {k: (dr[k[0]], dr[k[2]]) for k in Rk})
    th = fi.theta_random(9, c, dl, dr)
    W1, W2 = symm.mpo_reduced(c, 1.0, 4.0), symm.mpo_reduced(c + 1, 1.0, 4.0)
    ctx = H.binding.Context(int(max(1 << 30, 48.0 * chi * chi)))
    try:
        mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
        mps = ctx.mps_create(L)
        ctx.mps_set_bond(mps, c, dl)
        ctx.mps_set_bond(mps, c + 2, dr)
        for which, bond, keys, E in ((0, c, Lk, Le), (1, c + 2, Rk, Re)):
            labels = [[k[0][0], k[0][1], k[1], k[2][0], k[2][1]] for k in keys]
            flat = np.concatenate([E[k].ravel() for k in keys])
            ctx.env_set(mps, which, bond, labels, flat)
        ctx.heff_plan(mpo, mps, c, 2)
        lab, dm, ne = ctx.heff_layout(2)
        x = H.to_planned(ctx, H.flatten(th, lab, dm, H.theta_key))
        y = _torch().empty_like(x)
        ctx.heff_apply(x, y)
        got = H.unflatten(H.from_planned(ctx, y), lab, dm, H.theta_key)
        y2 = _torch().empty_like(x)
        ctx.heff_apply(2.0 * x, y2)
        assert bool((y2 == 2.0 * y).all())                      # exact: scaling by 2 commutes with rounding
        rng = np.random.default_rng(chi)
        keys = sorted(th)
        big = sorted(keys, key=lambda k: -th[k].size)[:6]
        pick = big + [keys[i] for i in rng.choice(len(keys), nsample, replace=False)]
        ref = heff2_selected(Le, Re, th, W1, W2, pick)
        worst = 0.0
        for k in pick:
            den_ = max(np.linalg.norm(ref[k]), 1e-300)
            worst = max(worst, np.linalg.norm(got[k] - ref[k]) / den_)
        print("chi=%d: %d sampled blocks, worst rel. Frobenius error %.2e" % (chi, len(pick), worst))
        assert worst < TOL_APPLY
        ctx.mps_destroy(mps)
    finally:
        ctx.close()


# ------------------------------------------------------------------ Lanczos exponential (H6 + H7)
def test_expm_parity_central_bond(H, ctx):
    """exp(-i tau H_eff) theta with m = 10 on the chi = 256 central bond vs the oracle's Lanczos
    (full re-orthogonalisation) on the sqrt(2j+1)-scaled flat vector; norm conserved."""
    chi, L, tau, m = 256, 60, 0.025, 10
    o = central_bond(chi, L)
    c = o["centre"]
    dl, dr = o["dims"][c], o["dims"][c + 2]
    th = fi.theta_random(fi.SEED, c, dl, dr)
    W1, W2 = o["W"][c], o["W"][c + 1]

    def apply_h(vec):
        t = stv.unflatten(vec, th)
        out = symm.heff2_apply(o["Lenv"], o["Renv"], t, W1, W2)
        return stv.flatten({k: out[k] for k in th})

    ref = stv.unflatten(lanczos_exp(apply_h, stv.flatten(th), tau, m), th)
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps, _ = H.build_central_bond(ctx, mpo, chi, L)
    ctx.heff_plan(mpo, mps, c, 2)
    lab, dm, ne = ctx.heff_layout(2)
    x = H.to_planned(ctx, H.flatten(th, lab, dm, H.theta_key))
    y = _torch().empty_like(x)
    ctx.heff_expm(x, y, tau, m)
    got = H.unflatten(H.from_planned(ctx, y), lab, dm, H.theta_key)
    assert rel_err(got, ref) < 1e-10
    n0, n1 = ctx.heff_inner(x, x).real, ctx.heff_inner(y, y).real
    assert abs(n1 / n0 - 1.0) < 1e-11
    ctx.mps_destroy(mps)


# ------------------------------------------------------------------ BASELINE config 1 end to end
NOISE = 1e-12    # floor, relative to the largest singular value on the bond (reading A-13)
SV_TOL = 1e-11   # |s_gpu - s_oracle| <= SV_TOL * s_max for every singular value above the floor


def _compare_bond(dims_g, sv_g, dims_o, sv_o, where):
    """Sector tables after an SVD split (reading A-13): a two-site tensor of exact rank r has singular values
    that are pure rounding noise (~1e-16 s_max) beyond r, and rule A-6 keeps those that land above 1e-14 s_max --
    a coin toss that differs between two correct SVDs.  What is unique: per sector, the singular values above
    the noise floor (1e-12 s_max; the two sides run different, both valid, Lanczos variants (A-5), whose results
    differ by ~1e-13 relative, and an SVD resolves singular values to that absolute accuracy).  Above the floor
    the values must agree in number and to 1e-11 s_max.  Returns the largest deviation / s_max."""
    smax = max(v.max() for v in sv_o.values())
    worst = 0.0
    for sec in sorted(set(dims_g) | set(dims_o)):
        g = sv_g.get(sec, np.zeros(0))
        o = sv_o.get(sec, np.zeros(0))
        assert len(g) == dims_g.get(sec, 0) and len(o) == dims_o.get(sec, 0), where
        n = max(len(g), len(o))
        gp, op = np.zeros(n), np.zeros(n)
        gp[:len(g)], op[:len(o)] = g, o
        gp[gp < NOISE * smax] = 0.0
        op[op < NOISE * smax] = 0.0
        d = np.abs(gp - op).max() / smax
        worst = max(worst, d)
        assert d < SV_TOL, (where, sec, d)
        assert (gp > 10 * SV_TOL * smax).sum() == (op > 10 * SV_TOL * smax).sum(), (where, sec)
    return worst


def test_config1_neel_quench_L8_vs_oracle(H, ctx):
    """configs[0]: L=8 Neel quench, t_h=1, U=4, dt=0.05 to t=1.0, chi_max 256 (exact), m=10.
    GPU tdvp2_sweep + measure_local/global vs the oracle's symmetric TDVP2 driver at matched chi.
    (a) eps_trunc = -1 (nothing but rounding noise is dropped): observables <= 1e-8, kept singular values of
    every bond after every step equal above the noise floor (see _compare_bond: the sector TABLES are not
    unique here, reading A-13), norm and energy conserved.
    (b) eps_trunc = 1e-12 (the rounding-noise values are cut on both sides, so the tables ARE unique):
    sector tables bit-identical after every step, observables <= 1e-8."""
    L, t_h, U, dt, nstep, m = 8, 1.0, 4.0, 0.05, 20, 10
    ref = stv.SymmTDVP(L, t_h, U, krylov_dim=m, chi_max_full=256, eps_trunc=-1.0)
    mpo = ctx.fh_mpo_build(L, t_h, U)
    mps = ctx.mps_init_neel(mpo, L)
    g0 = ctx.measure_global(mpo, mps)
    assert abs(g0["norm2"] - 1.0) < 1e-14 and abs(g0["energy"]) < 1e-13   # <Neel|H|Neel> = 0
    l0 = ctx.measure_local(mps, L)
    assert np.allclose(l0["sz"], [0.5 if i % 2 == 0 else -0.5 for i in range(L)], atol=1e-14)
    assert np.allclose(l0["docc"], 0.0, atol=1e-14) and np.allclose(l0["n"], 1.0, atol=1e-14)
    worst, worst_sv = 0.0, 0.0
    for step in range(nstep):
        ref.step(dt)
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=256, eps_trunc=-1.0)
        a, b = ref.measure_local(), ctx.measure_local(mps, L)
        for key in ("n", "sz", "docc"):
            worst = max(worst, np.abs(a[key] - b[key]).max())
        ga, gb = ref.measure_global(), ctx.measure_global(mpo, mps)
        assert abs(ga["norm2"] - gb["norm2"]) < 1e-10 and abs(ga["energy"] - gb["energy"]) < 1e-9
        assert abs(gb["norm2"] - 1.0) < 1e-10 and abs(gb["energy"]) < 1e-9
        for k in range(1, L):
            worst_sv = max(worst_sv, _compare_bond(ctx.mps_get_bond(mps, k), ctx.mps_get_svals(mps, k), ref.dims[k],
                                                   ref.svals[k], (step, k)))
    assert worst < 1e-8, worst
    st = ctx.tdvp2_last_stats()
    assert st["max_discarded"] < 1e-20
    ctx.mps_destroy(mps)
    # (b) deterministic tables
    ref = stv.SymmTDVP(L, t_h, U, krylov_dim=m, chi_max_full=256, eps_trunc=1e-12)
    mps = ctx.mps_init_neel(mpo, L)
    worst_b = 0.0
    for step in range(nstep):
        ref.step(dt)
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=256, eps_trunc=1e-12)
        for k in range(L + 1):
            assert ctx.mps_get_bond(mps, k) == ref.dims[k], (step, k)     # bit-exact sector bookkeeping
        a, b = ref.measure_local(), ctx.measure_local(mps, L)
        for key in ("n", "sz", "docc"):
            worst_b = max(worst_b, np.abs(a[key] - b[key]).max())
    assert worst_b < 1e-8, worst_b
    assert ctx.tdvp2_last_stats()["chi_full"] == max(ref.chi())
    print("config 1: observables %.1e (exact run) / %.1e (eps 1e-12), singular values above the floor %.1e s_max"
          % (worst, worst_b, worst_sv))
    ctx.mps_destroy(mps)


@pytest.mark.parametrize("L,chi,route", [(12, 128, "default"), (14, 200, "default"), (12, 128, "mid"), (12, 128, "vendor"),
                                         (12, 128, "gram"), (14, 200, "gram"), (14, 200, "gram1")])
def test_config3_sweep_recipe_reduced_size_vs_oracle(H, ctx, L, chi, route):
    """The second half of BASELINE config 3 -- one tdvp2_sweep(0.05), m = 10, truncation back to chi by block-wise
    SVD, started from the seeded random canonical chain (the recipe bench.py times at L = 60,
    chi = 4096: harness.build_central_bond(centre=0, keep_sites=True)) -- at a size the oracle's symmetric driver
    finishes in seconds, on both sides from the same seeded site tensors.  Every bond is truly truncated here
    (a random two-site tensor has full rank), and the sector matrices go through all SVD routes the library has
    for their sizes.  Compared: sector tables after the sweep bit for bit, kept singular values per bond and
    sector (<= 1e-10 s_max), the largest discarded weight, norm, energy and local observables (<= 1e-8);
    then one tdvp1_sweep on the result (one-site splits by QR) against the oracle's step1.
    `route` sends the sector matrices of this small case through the factorisation routes that large bonds use
    (fh_set_option): "mid" = the global-memory Jacobi kernel and cusolver's geqrf/ungqr, "vendor" = cusolver's
    gesvdp / gesvd and geqrf/ungqr; "default" = the shared-memory Jacobi and Householder kernels; "gram" = the
    Gram-matrix eigenvalue route (G = B^H B, eigendecomposition, U = B V / sigma) for every matrix of at least 8
    columns, the eigenproblems of a bond solved in one batched vendor call on Gram matrices padded to a common size
    ("gram1": one Zheevd call per matrix), with its acceptance test on the kept singular values and the vendor redo of
    the sectors that fail it."""
    if route != "default":
        ctx.fh_set_option(ctx.OPT_SVD_SMALL_MAXN, 0)
        ctx.fh_set_option(ctx.OPT_SVD_MID_MAXN, 128 if route == "mid" else 0)
    ctx.fh_set_option(ctx.OPT_SVD_GRAM_MINN, 8 if route.startswith("gram") else 0)
    if route == "gram1":                                  # one eigensolver call per matrix instead of the batched call
        ctx.fh_set_option(ctx.OPT_SVD_GRAM_BATCH_MAXN, 0)
    dims = fi.chain_dims(chi, L, "gaussian", (1, 1))
    sites = {}
    for i, A, dl, dr in fi.canonical_chain(chi, 0, L, fi.SEED, dims=dims, weight=symm.canonical_weight):
        sites[i] = A
    ref = stv.SymmTDVP(L, 1.0, 4.0, krylov_dim=10, chi_max_full=chi, eps_trunc=-1.0,
                       A=[dict(sites[i]) for i in range(L)], dims=[dict(d) for d in dims])
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps, gdims = H.build_central_bond(ctx, mpo, chi, L, centre=0, keep_sites=True)
    assert gdims == dims
    g0, r0 = ctx.measure_global(mpo, mps), ref.measure_global()
    assert abs(g0["norm2"] / r0["norm2"] - 1) < 1e-11 and abs(g0["energy"] - r0["energy"]) < 1e-9 * abs(r0["energy"])
    f0 = ctx.fh_factorization_stats()
    ref.step(0.05)
    ctx.tdvp2_sweep(mpo, mps, 0.05, krylov_dim=10, chi_max_full=chi, eps_trunc=-1.0)
    f1 = ctx.fh_factorization_stats()
    worst_sv = 0.0
    for k in range(L + 1):
        assert ctx.mps_get_bond(mps, k) == ref.dims[k], k          # bit-exact sector bookkeeping
    for k in range(1, L):
        sg, so = ctx.mps_get_svals(mps, k), ref.svals[k]
        assert sg.keys() == so.keys(), k
        smax = max(v.max() for v in so.values())
        for sec in so:
            worst_sv = max(worst_sv, np.abs(sg[sec] - so[sec]).max() / smax)
    st = ctx.tdvp2_last_stats()
    assert worst_sv < 1e-10, worst_sv
    assert ref.max_discarded > 1e-6 and abs(st["max_discarded"] / ref.max_discarded - 1) < 1e-8
    assert st["chi_full"] == max(ref.chi())
    a, b = ref.measure_local(), ctx.measure_local(mps, L)
    worst = max(np.abs(a[key] - b[key]).max() for key in ("n", "sz", "docc"))
    ga, gb = ref.measure_global(), ctx.measure_global(mpo, mps)
    assert worst < 1e-8 and abs(ga["norm2"] / gb["norm2"] - 1) < 1e-9 and abs(ga["energy"] - gb["energy"]) < 1e-8
    ref.step1(0.05)
    ctx.tdvp1_sweep(mpo, mps, 0.05, krylov_dim=10)
    f2 = ctx.fh_factorization_stats()
    a, b = ref.measure_local(), ctx.measure_local(mps, L)
    worst1 = max(np.abs(a[key] - b[key]).max() for key in ("n", "sz", "docc"))
    for k in range(L + 1):
        assert ctx.mps_get_bond(mps, k) == ref.dims[k], k
    assert worst1 < 1e-8, worst1
    routes = {k: f1[k] - f0[k] for k in f1}
    if route == "mid":
        assert routes["jacobi_mid_kernel"] > 0 and routes["jacobi_kernel"] == 0 and f2["qr"] - f1["qr"] > 0
    if route == "vendor":
        assert routes["gesvdp"] + routes["gesvd"] > 0 and routes["jacobi_kernel"] == routes["jacobi_mid_kernel"] == 0
        assert routes["gram_eig"] == 0
    if route.startswith("gram"):
        assert routes["gram_eig"] > 0 and routes["jacobi_kernel"] == routes["jacobi_mid_kernel"] == 0
        assert routes["gram_redone"] < routes["gram_eig"]          # some sectors pass the acceptance test
    print("L=%d chi=%d sweep: sv %.1e s_max, obs %.1e / one-site %.1e, discarded %.3e (oracle %.3e); SVD routes %s; "
          "QR routes %s" % (L, chi, worst_sv, worst, worst1, st["max_discarded"], ref.max_discarded, routes,
                            {k: f2[k] - f1[k] for k in f2 if k.startswith("qr")}))
    ctx.mps_destroy(mps)


def test_gram_route_redone_when_small_singular_values_are_kept(H, ctx):
    """The Gram-matrix eigenvalue route (FH_OPT_SVD_GRAM_MINN) squares the matrix and is accurate only for singular
    values that are not small; the library accepts its result for a sector only if every KEPT value is >= 3e-3 of
    the sector's largest and redoes the sector by the vendor SVD otherwise.  An UNtruncated quench keeps everything
    (down to rule A-6's floor), so with the route forced on every matrix the redo must fire, and the run must still
    agree with the dense oracle as the default routes do (config 1's problem, 8 steps: observables <= 1e-8,
    norm to 1e-10)."""
    from oracle import dense_tdvp as dtv
    L, dt, m = 8, 0.05, 10
    ctx.fh_set_option(ctx.OPT_SVD_SMALL_MAXN, 0)
    ctx.fh_set_option(ctx.OPT_SVD_MID_MAXN, 0)
    ctx.fh_set_option(ctx.OPT_SVD_GRAM_MINN, 2)
    ref = dtv.DenseTDVP(L, 1.0, 4.0, krylov_dim=m)
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_init_neel(mpo, L)
    worst = 0.0
    for step in range(8):
        ref.step(dt)
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=256, eps_trunc=-1.0)
        o, g = ref.observables(), ctx.measure_local(mps, L)
        worst = max(worst, np.abs(g["sz"] - 0.5 * (o["n_up"] - o["n_dn"])).max(), np.abs(g["docc"] - o["docc"]).max())
    f = ctx.fh_factorization_stats()
    gg = ctx.measure_global(mpo, mps)
    print("Gram route forced, untruncated L=8 quench: obs %.1e, norm^2 - 1 %.1e, routes %s" % (worst, gg["norm2"] - 1, f))
    assert f["gram_eig"] > 0 and f["gram_redone"] > 0 and f["jacobi_kernel"] == 0
    assert worst < 1e-8 and abs(gg["norm2"] - 1) < 1e-10
    ctx.mps_destroy(mps)


def test_config4_L60_U0_quench_vs_closed_form(H, ctx):
    """configs[3] shape at U=0: L=60 Neel quench, dt=0.05, m=10, eps_trunc=1e-12 (chi grows as the
    entanglement demands), against the free-fermion closed form O-U0 (oracle/u0.py: single-particle
    propagator of the open chain) -- a pin of the large-L symmetric code path that does not go
    through the symmetric oracle.  The residual is the TDVP2 splitting error at dt=0.05 (O(dt^2) per
    unit time, measured ~1e-6 at L=8 against ED) plus the 1e-12 truncation; n_i = 1 must hold to
    rounding (reading A-12) and the norm and energy (= 0 for the Neel state at any U) stay put."""
    from oracle import u0
    L, t_h, dt, nstep, m = 60, 1.0, 0.05, 8, 10
    mpo = ctx.fh_mpo_build(L, t_h, 0.0)
    mps = ctx.mps_init_neel(mpo, L)
    worst = 0.0
    for step in range(1, nstep + 1):
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=4096, eps_trunc=1e-12)
        got = ctx.measure_local(mps, L)
        ref = u0.observables(L, t_h, step * dt)
        assert np.abs(got["n"] - 1.0).max() < 1e-10
        worst = max(worst, np.abs(got["sz"] - ref["sz"]).max(), np.abs(got["docc"] - ref["docc"]).max())
        g = ctx.measure_global(mpo, mps)
        assert abs(g["norm2"] - 1.0) < 1e-8 and abs(g["energy"]) < 1e-7
    st = ctx.tdvp2_last_stats()
    print("L=60 U=0: max |obs - closed form| = %.2e, chi reached %d (chi_su2 %d), discarded %.1e"
          % (worst, st["chi_full"], st["chi_su2"], st["max_discarded"]))
    assert worst < 2e-5, worst
    assert st["max_discarded"] < 1e-10
    ctx.mps_destroy(mps)


def test_next1_one_site_tdvp_L8_vs_oracle(H, ctx):
    """NEXT-1: tdvp1_sweep against the oracle's symmetric one-site driver (itself equal to the dense TDVP1
    that is pinned against ED).  L = 8 Neel quench: five two-site steps with eps_trunc = 1e-12 grow the
    bonds, then six one-site steps at frozen bond dimensions; observables <= 1e-8, identical sector
    tables after every step, norm and energy conserved."""
    L, t_h, U, dt, m = 8, 1.0, 4.0, 0.05, 10
    ref = stv.SymmTDVP(L, t_h, U, krylov_dim=m, chi_max_full=256, eps_trunc=1e-12)
    mpo = ctx.fh_mpo_build(L, t_h, U)
    mps = ctx.mps_init_neel(mpo, L)
    for _ in range(5):
        ref.step(dt)
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=256, eps_trunc=1e-12)
    e0 = ctx.measure_global(mpo, mps)["energy"]
    worst = 0.0
    for step in range(6):
        ref.step1(dt)
        ctx.tdvp1_sweep(mpo, mps, dt, krylov_dim=m)
        a, b = ref.measure_local(), ctx.measure_local(mps, L)
        for key in ("n", "sz", "docc"):
            worst = max(worst, np.abs(a[key] - b[key]).max())
        ga, gb = ref.measure_global(), ctx.measure_global(mpo, mps)
        assert abs(ga["norm2"] - gb["norm2"]) < 1e-10 and abs(ga["energy"] - gb["energy"]) < 1e-9
        assert abs(gb["energy"] - e0) < 1e-7          # TDVP conserves the energy
        for k in range(1, L):
            assert ctx.mps_get_bond(mps, k) == ref.dims[k], (step, k)
    print("TDVP1 L=8: max |obs GPU - oracle| = %.2e" % worst)
    assert worst < 1e-8, worst
    ctx.mps_destroy(mps)


def test_next1_one_site_task_list_cache(H, ctx, tmp_path):
    """H0 for the one-site sweeps: tdvp1_sweep keeps its task lists from sweep to sweep (one-site TDVP leaves the
    sector tables alone).  Two copies of the same L = 8 state (via mps_save / mps_load) run four
    one-site sweeps, one with the cache, one with it switched off: every site tensor must agree bit for bit
    (same lists, same launches), the cached run re-emits nothing after its first sweep, the uncached run never
    hits, and a two-site sweep empties the cache."""
    L, dt, m = 8, 0.05, 8
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_init_neel(mpo, L)
    for _ in range(4):
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=60)
    path = str(tmp_path / "s.fhmps")
    ctx.mps_save(mps, path)
    a, b = ctx.mps_load(mpo, path), ctx.mps_load(mpo, path)
    ctx.fh_plan_cache_limit(b, 0)
    ctx.tdvp1_sweep(mpo, a, dt, krylov_dim=m)
    s1 = ctx.fh_plan_cache_stats(a)
    # within the first sweep the right-to-left half already reuses the one-site and zero-site plans of the first half
    assert s1["misses"] > 0 and s1["hits"] > 0 and s1["host_bytes"] > 0
    for _ in range(3):
        ctx.tdvp1_sweep(mpo, a, dt, krylov_dim=m)
    s4 = ctx.fh_plan_cache_stats(a)
    assert s4["misses"] == s1["misses"], (s1, s4)         # nothing re-emitted after the first sweep
    assert s4["hits"] > s1["hits"] and s4["host_bytes"] == s1["host_bytes"]
    # the uncached run also goes without the library's phase events (fh_enable_timers): nothing is recorded,
    # and the results below are still bit-identical (events and the programmatic launch order change no arithmetic)
    ctx.fh_reset_timers()
    ctx.fh_enable_timers(False)
    try:
        for _ in range(4):
            ctx.tdvp1_sweep(mpo, b, dt, krylov_dim=m)
        assert all(v == 0.0 for v in ctx.fh_get_timers().values())
    finally:
        ctx.fh_enable_timers(True)
    sb = ctx.fh_plan_cache_stats(b)
    assert sb["hits"] == 0 and sb["host_bytes"] == 0
    for i in range(L):
        assert np.array_equal(ctx.mps_site_layout(a, i)[0], ctx.mps_site_layout(b, i)[0])
        assert np.array_equal(ctx.mps_get_site(a, i), ctx.mps_get_site(b, i)), i
    # a different Hamiltonian on the same state must not reuse the lists (U enters the coefficients)
    mpo2 = ctx.fh_mpo_build(L, 1.0, 2.0)
    ctx.fh_plan_cache_limit(b, 1 << 30)
    ctx.tdvp1_sweep(mpo2, a, dt, krylov_dim=m)
    ctx.tdvp1_sweep(mpo2, b, dt, krylov_dim=m)
    for i in range(L):
        assert np.array_equal(ctx.mps_get_site(a, i), ctx.mps_get_site(b, i)), i
    ctx.tdvp2_sweep(mpo, a, dt, krylov_dim=m, chi_max_full=60)
    assert ctx.fh_plan_cache_stats(a)["host_bytes"] == 0
    for h in (mps, a, b):
        ctx.mps_destroy(h)


# ------------------------------------------------------------------ NEXT-2: adaptive Krylov dimension (A-15)
def test_next2_adaptive_krylov_expm_and_sweeps(H, ctx):
    """(a) heff_expm_adaptive on the chi = 256 central bond: same number of Krylov vectors as the oracle's
    adaptive Lanczos for each tolerance, result within 1e-10, fewer vectors for the looser tolerance, and
    within ~tol of the fixed m = 20 result.  (b) L = 8 quench driven with krylov_adapt_tol = 1e-10 (two-site
    steps, then one-site steps): observables <= 1e-8 against the oracle running the same rule, and the same
    total number of H_eff applies."""
    chi, L, tau, mmax = 256, 60, 0.025, 20
    o = central_bond(chi, L)
    c = o["centre"]
    dl, dr = o["dims"][c], o["dims"][c + 2]
    th = fi.theta_random(fi.SEED, c, dl, dr)
    W1, W2 = o["W"][c], o["W"][c + 1]

    def apply_h(vec):
        t = stv.unflatten(vec, th)
        out = symm.heff2_apply(o["Lenv"], o["Renv"], t, W1, W2)
        return stv.flatten({k: out[k] for k in th})

    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps, _ = H.build_central_bond(ctx, mpo, chi, L)
    ctx.heff_plan(mpo, mps, c, 2)
    lab, dm, ne = ctx.heff_layout(2)
    x = H.to_planned(ctx, H.flatten(th, lab, dm, H.theta_key))
    y = _torch().empty_like(x)
    yfix = _torch().empty_like(x)
    ctx.heff_expm(x, yfix, tau, mmax)
    nx = float(ctx.heff_inner(x, x).real) ** 0.5
    used = {}
    for tol in (1e-4, 1e-8, 1e-12):
        st = []
        ref = stv.unflatten(lanczos_exp(apply_h, stv.flatten(th), tau, mmax, adapt_tol=tol, stats=st), th)
        k = ctx.heff_expm_adaptive(x, y, tau, mmax, tol)
        assert k == st[0], (tol, k, st)
        used[tol] = k
        got = H.unflatten(H.from_planned(ctx, y), lab, dm, H.theta_key)
        assert rel_err(got, ref) < 1e-10
        d = y - yfix
        assert float(ctx.heff_inner(d, d).real) ** 0.5 / nx < 10 * tol + 1e-12
    assert used[1e-4] < used[1e-8] < used[1e-12] < mmax
    print("adaptive Krylov, chi=256 central bond, tau=0.025: k =", used)
    ctx.mps_destroy(mps)

    L, t_h, U, dt, tol = 8, 1.0, 4.0, 0.05, 1e-10
    ref = stv.SymmTDVP(L, t_h, U, krylov_dim=mmax, chi_max_full=256, eps_trunc=1e-12, krylov_adapt_tol=tol)
    mpo = ctx.fh_mpo_build(L, t_h, U)
    mps = ctx.mps_init_neel(mpo, L)
    e0, v0 = ctx.fh_krylov_stats()
    worst = 0.0
    for step in range(8):
        if step < 5:
            ref.step(dt)
            ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=mmax, chi_max_full=256, eps_trunc=1e-12, krylov_adapt_tol=tol)
        else:
            ref.step1(dt)
            ctx.tdvp1_sweep(mpo, mps, dt, krylov_dim=mmax, krylov_adapt_tol=tol)
        a, b = ref.measure_local(), ctx.measure_local(mps, L)
        for key in ("n", "sz", "docc"):
            worst = max(worst, np.abs(a[key] - b[key]).max())
    e1, v1 = ctx.fh_krylov_stats()
    ku = [k for k in ref.krylov_used if k > 0]
    print("adaptive TDVP L=8: %d exponentials, %d applies (oracle %d, %d; fixed m would use %d); max obs diff %.2e"
          % (e1 - e0, v1 - v0, len(ku), sum(ku), mmax * len(ku), worst))
    assert worst < 1e-8, worst
    assert e1 - e0 == len(ku) and v1 - v0 == sum(ku)
    assert sum(ku) < 0.6 * mmax * len(ku)
    ctx.mps_destroy(mps)


def test_next1_auto_switch_two_site_to_one_site(H, ctx):
    """tdvp_sweep_auto (reading A-16): L = 8 quench with the bond dimension capped at chi_full = 40; the
    two-site steps stop growing any bond after the third step, both sides switch to one-site steps there
    (same 2/1 sequence), observables stay within 1e-8 and the sector tables stay identical."""
    L, t_h, U, dt, m, cap = 8, 1.0, 4.0, 0.05, 10, 40
    ref = stv.SymmTDVP(L, t_h, U, krylov_dim=m, chi_max_full=cap, eps_trunc=-1.0)
    mpo = ctx.fh_mpo_build(L, t_h, U)
    mps = ctx.mps_init_neel(mpo, L)
    seq_o, seq_g, worst = [], [], 0.0
    for step in range(8):
        seq_o.append(ref.step_auto(dt))
        seq_g.append(ctx.tdvp_sweep_auto(mpo, mps, dt, krylov_dim=m, chi_max_full=cap, eps_trunc=-1.0))
        a, b = ref.measure_local(), ctx.measure_local(mps, L)
        for key in ("n", "sz", "docc"):
            worst = max(worst, np.abs(a[key] - b[key]).max())
        for k in range(1, L):
            assert ctx.mps_get_bond(mps, k) == ref.dims[k], (step, k)
    print("auto switch: oracle", seq_o, "GPU", seq_g, "max obs diff %.2e" % worst)
    assert seq_g == seq_o and seq_g[0] == 2 and seq_g[-1] == 1
    assert worst < 1e-8, worst
    ctx.mps_destroy(mps)


@pytest.mark.parametrize("L", [2, 4, 6])
def test_tiny_chains_two_site_one_site_auto(H, ctx, L):
    """Degenerate sizes: the shortest chains (1 x 1 sectors, bonds that reach their exact dimension after one or
    two steps, QR of matrices with fewer rows than columns).  tdvp_sweep_auto against the oracle's step_auto:
    same 2/1 sequence, observables to 1e-12, norm and energy conserved."""
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_init_neel(mpo, L)
    ref = stv.SymmTDVP(L, 1.0, 4.0, krylov_dim=8, chi_max_full=64, eps_trunc=-1.0)
    worst = 0.0
    for step in range(6):
        assert ref.step_auto(0.05) == ctx.tdvp_sweep_auto(mpo, mps, 0.05, krylov_dim=8, chi_max_full=64, eps_trunc=-1.0)
        a, b = ref.measure_local(), ctx.measure_local(mps, L)
        for key in ("n", "sz", "docc"):
            worst = max(worst, np.abs(a[key] - b[key]).max())
    g = ctx.measure_global(mpo, mps)
    assert worst < 1e-12 and abs(g["norm2"] - 1.0) < 1e-11 and abs(g["energy"]) < 1e-11, (worst, g)
    assert getattr(ref, "saturated", False)
    ctx.mps_destroy(mps)


def test_checkpoint_resume(H, ctx, tmp_path):
    """mps_save / mps_load: a run interrupted after three steps and resumed from the file continues exactly like
    the uninterrupted one (the right environments are recomputed from the same tensors by the same kernels, so
    the observables agree to rounding), the auto-switch flag travels with the state, bad files are refused."""
    L, dt, m = 8, 0.05, 10
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_init_neel(mpo, L)
    kw = dict(krylov_dim=m, chi_max_full=40, eps_trunc=-1.0)
    for _ in range(4):
        ctx.tdvp_sweep_auto(mpo, mps, dt, **kw)
    path = str(tmp_path / "state.fhmps")
    ctx.mps_save(mps, path)
    seq_a = [ctx.tdvp_sweep_auto(mpo, mps, dt, **kw) for _ in range(3)]
    a, ga = ctx.measure_local(mps, L), ctx.measure_global(mpo, mps)
    mps2 = ctx.mps_load(mpo, path)
    seq_b = [ctx.tdvp_sweep_auto(mpo, mps2, dt, **kw) for _ in range(3)]
    b, gb = ctx.measure_local(mps2, L), ctx.measure_global(mpo, mps2)
    assert seq_a == seq_b and seq_a[-1] == 1          # saturated flag restored: one-site steps after the reload
    for key in ("n", "sz", "docc"):
        assert np.abs(a[key] - b[key]).max() < 1e-13, key
    assert abs(ga["norm2"] - gb["norm2"]) < 1e-13 and abs(ga["energy"] - gb["energy"]) < 1e-12
    for k in range(L + 1):
        assert ctx.mps_get_bond(mps, k) == ctx.mps_get_bond(mps2, k)
    # refused: missing file, truncated file, wrong chain length
    with pytest.raises(H.binding.FhError):
        ctx.mps_load(mpo, str(tmp_path / "nope.fhmps"))
    blob = open(path, "rb").read()
    open(str(tmp_path / "cut.fhmps"), "wb").write(blob[:len(blob) // 2])
    with pytest.raises(H.binding.FhError):
        ctx.mps_load(mpo, str(tmp_path / "cut.fhmps"))
    mpo6 = ctx.fh_mpo_build(6, 1.0, 4.0)
    with pytest.raises(H.binding.FhError):
        ctx.mps_load(mpo6, path)
    ctx.mps_destroy(mps)
    ctx.mps_destroy(mps2)


# ------------------------------------------------------------------ larger sectors: vendor SVD / QR routes
def test_quench_L24_large_sectors_invariants(H, ctx):
    """The L = 8 cases above keep every sector matrix below 48 columns, i.e. on the library's own Jacobi
    kernel.  This quench (L = 24, U = 4, dt = 0.05, eps_trunc = 1e-10) grows the bonds to several hundred
    states so that the gesvdp route (and, in the one-site steps that follow, Householder QR on the worker
    streams) carries the sweep; the oracle is too slow here, so the checks are what holds at any size:
    norm and energy conservation (E(0) = 0 for the Neel state; truncation 1e-10 per bond), <n_i> = 1 on every
    site (T_tot = 0), total S^z = 0, and the inversion x spin-flip symmetry of the Neel quench on an even
    chain, S^z_i = -S^z_{L-1-i}, docc_i = docc_{L-1-i}."""
    L, t_h, U, dt, m = 24, 1.0, 4.0, 0.05, 10
    mpo = ctx.fh_mpo_build(L, t_h, U)
    mps = ctx.mps_init_neel(mpo, L)
    f0 = ctx.fh_factorization_stats()

    def check(tag, etol):
        g = ctx.measure_global(mpo, mps)
        o = ctx.measure_local(mps, L)
        assert abs(g["norm2"] - 1.0) < 1e-6, (tag, g)
        assert abs(g["energy"]) < etol, (tag, g)
        assert np.abs(o["n"] - 1.0).max() < 1e-9, tag
        assert abs(o["sz"].sum()) < 1e-9, tag
        assert np.abs(o["sz"] + o["sz"][::-1]).max() < 1e-6, tag
        assert np.abs(o["docc"] - o["docc"][::-1]).max() < 1e-6, tag
        return g, o

    for step in range(36):
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=4096, eps_trunc=1e-10)
        if step % 6 == 5:
            check(("two-site", step), 1e-5)
    st = ctx.tdvp2_last_stats()
    g2, o2 = check("end of two-site phase", 1e-5)
    f1 = ctx.fh_factorization_stats()
    assert st["chi_full"] > 300 and st["dmax"] >= 24, st
    # the routes above the shared-memory kernel really ran (own global-memory Jacobi up to 128 columns, vendor beyond)
    assert f1["gesvdp"] + f1["jacobi_mid_kernel"] - f0["gesvdp"] - f0["jacobi_mid_kernel"] > 0, f1
    assert f1["jacobi_kernel"] - f0["jacobi_kernel"] > 0, f1
    dims_before = [ctx.mps_get_bond(mps, k) for k in range(L + 1)]
    for step in range(4):
        ctx.tdvp1_sweep(mpo, mps, dt, krylov_dim=m)
    g1, o1 = check("one-site phase", 1e-5)
    f2 = ctx.fh_factorization_stats()
    assert f2["qr"] + f2["qr_kernel"] - f1["qr"] - f1["qr_kernel"] > 0, f2
    assert [ctx.mps_get_bond(mps, k) for k in range(L + 1)] == dims_before      # one-site steps keep the bonds
    assert abs(g1["energy"] - g2["energy"]) < 1e-8 and abs(g1["norm2"] - g2["norm2"]) < 1e-9   # no truncation
    assert 0.02 < o1["docc"].mean() < 0.25 and np.abs(o1["sz"]).max() < 0.5                # the state has moved
    print("L=24 quench: chi_full %d, d_max %d, factorizations %s, E = %.2e, norm2 - 1 = %.2e"
          % (st["chi_full"], st["dmax"], f2, g1["energy"], g1["norm2"] - 1.0))
    ctx.mps_destroy(mps)


def test_mid_size_jacobi_kernel_vs_vendor_svd(H, ctx, tmp_path):
    """H9: sector matrices above the shared-memory route with at most 128 columns are factorised by the library's
    own global-memory Jacobi kernel (mid_svd_kernel, on a side stream beside the vendor routines).  The same L = 16
    state (grown by an untruncated quench until sector matrices of 90-128 columns exist) takes one two-site sweep
    with that kernel and, from a reloaded copy, one with fh_set_option(FH_OPT_SVD_MID_MAXN, 0) (every such matrix through cusolver's
    gesvdp / gesvd): both routes must have run, the kept singular values of every bond agree to 1e-11 s_max, the
    sector tables are identical and the observables agree to 1e-10."""
    L, dt, m = 16, 0.1, 8
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_init_neel(mpo, L)
    for _ in range(22):
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=1200, eps_trunc=1e-12)
    path = str(tmp_path / "mid.fhmps")
    ctx.mps_save(mps, path)
    a, b = ctx.mps_load(mpo, path), ctx.mps_load(mpo, path)
    f0 = ctx.fh_factorization_stats()
    ctx.tdvp2_sweep(mpo, a, dt, krylov_dim=m, chi_max_full=1200, eps_trunc=1e-12)
    f1 = ctx.fh_factorization_stats()
    ctx.fh_set_option(ctx.OPT_SVD_MID_MAXN, 0)
    try:
        ctx.tdvp2_sweep(mpo, b, dt, krylov_dim=m, chi_max_full=1200, eps_trunc=1e-12)
    finally:
        ctx.fh_set_option(ctx.OPT_SVD_MID_MAXN, 128)
    f2 = ctx.fh_factorization_stats()
    assert f1["jacobi_mid_kernel"] - f0["jacobi_mid_kernel"] > 0, (f0, f1)
    assert f2["jacobi_mid_kernel"] == f1["jacobi_mid_kernel"]
    assert f2["gesvdp"] + f2["gesvd"] - f1["gesvdp"] - f1["gesvd"] >= f1["jacobi_mid_kernel"] - f0["jacobi_mid_kernel"]
    worst = 0.0
    for k in range(1, L):
        assert ctx.mps_get_bond(a, k) == ctx.mps_get_bond(b, k), k
        sa, sb = ctx.mps_get_svals(a, k), ctx.mps_get_svals(b, k)
        assert sa.keys() == sb.keys()
        smax = max(v.max() for v in sa.values())
        for key in sa:
            worst = max(worst, np.abs(sa[key] - sb[key]).max() / smax)
    oa, ob = ctx.measure_local(a, L), ctx.measure_local(b, L)
    dobs = max(np.abs(oa[key] - ob[key]).max() for key in ("n", "sz", "docc"))
    print("mid-size Jacobi vs vendor: %d matrices, max |ds|/s_max = %.2e, max |obs diff| = %.2e"
          % (f1["jacobi_mid_kernel"] - f0["jacobi_mid_kernel"], worst, dobs))
    assert worst < 1e-11 and dobs < 1e-10, (worst, dobs)
    for h in (mps, a, b):
        ctx.mps_destroy(h)


# ------------------------------------------------------------------ NEXT-4: U(1) x U(1) mode
@pytest.fixture()
def actx(H):
    c = H.binding.Context(2 << 30)
    c.fh_set_option(c.OPT_SYMMETRY, 1)
    yield c
    c.close()


def test_next4_abelian_env_and_apply_parity(H, actx):
    """U(1) x U(1) mode (FH_OPT_SYMMETRY = 1): environments (H4, H5) along a random abelian
    chain, the two-site apply on every bond and the one-site apply on every site against oracle/abelian.py
    (pinned against the dense contractions), <= 1e-11; then the central bond of the abelian profile at chi = 4096
    (the small-block stress case: 2012 blocks, d_max 148) on ALL output blocks with random environments."""
    import fh_inputs.abelian as fab
    from oracle import abelian as ab
    ctx = actx
    rng = np.random.default_rng(5)
    L = 6
    dims = [{k: min(v, int(rng.integers(1, 6))) for k, v in d.items()} for d in fab.chain_dims(10 ** 6, L)]
    A = [{k: _rand(rng, dims[i][k[0]], dims[i + 1][k[2]]) for k in ab.site_keys(dims[i], dims[i + 1])} for i in range(L)]
    W = ab.mpo_elements(1.0, 4.0)
    Le, Re = [ab.boundary_left()], [None] * (L + 1)
    for i in range(L):
        Le.append(ab.env_update_left(Le[i], A[i], W))
    Re[L] = ab.boundary_right()
    for i in range(L - 1, -1, -1):
        Re[i] = ab.env_update_right(Re[i + 1], A[i], W)
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    val, rank2 = ctx.fh_mpo_get_site(mpo, 1)
    for (w, wp), M in W.items():
        assert np.array_equal(val[w, wp], M) and rank2[w, wp] == 0          # the library's own W = 6 table
    assert (rank2 >= 0).sum() == len(W)
    mps = ctx.mps_create(L)
    for i in range(L):
        H.set_site(ctx, mps, i, A[i], dims[i], dims[i + 1])
    for i in range(L):
        ctx.env_update_left(mpo, mps, i)
    for i in range(L - 1, -1, -1):
        ctx.env_update_right(mpo, mps, i)
    for which, ref in ((0, Le), (1, Re)):
        for k in range(L + 1):
            lab, dm, flat = ctx.env_get(mps, which, k)
            got = H.unflatten(flat, lab, dm, env_key)
            assert sorted(got) == sorted(ref[k]), (which, k)
            assert rel_err(got, ref[k], weighted=False) < 1e-12, (which, k)
    for i in range(L - 1):
        th = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]) for k in ab.theta_keys(dims[i], dims[i + 2])}
        ctx.heff_plan(mpo, mps, i, 2)
        assert rel_err(_apply_gpu(H, ctx, th, 2), ab.heff2_apply(Le[i], Re[i + 2], th, W, W), weighted=False) < TOL_APPLY
    for i in range(L):
        ctx.heff_plan(mpo, mps, i, 1)
        assert rel_err(_apply_gpu(H, ctx, A[i], 1), ab.heff1_apply(Le[i], Re[i + 1], A[i], W), weighted=False) < TOL_APPLY
    ctx.mps_destroy(mps)
    # central bond at chi = 4096
    Lc, c, chi = 60, 29, 4096
    dl, dr = fab.profile(c, chi), fab.profile(c + 2, chi)
    Lk, Rk = ab.env_keys(dl, dl), ab.env_keys(dr, dr)
    Lenv = fi.random_blocks(9, 1, Lk, {k: (dl[k[0]], dl[k[2]]) for k in Lk})
    Renv = fi.random_blocks(9, 2, Rk, {k: (dr[k[0]], dr[k[2]]) for k in Rk})
    th = fab.theta_random(9, c, dl, dr)
    mpo = ctx.fh_mpo_build(Lc, 1.0, 4.0)
    mps = ctx.mps_create(Lc)
    ctx.mps_set_bond(mps, c, dl)
    ctx.mps_set_bond(mps, c + 2, dr)
    for which, bond, keys, E in ((0, c, Lk, Lenv), (1, c + 2, Rk, Renv)):
        labels = [[k[0][0], k[0][1], k[1], k[2][0], k[2][1]] for k in keys]
        ctx.env_set(mps, which, bond, labels, np.concatenate([E[k].ravel() for k in keys]))
    ctx.heff_plan(mpo, mps, c, 2)
    st1, st2 = ab.heff2_tasks(Lk, Rk, sorted(th), W, W)
    assert ctx.heff_flops() == ab.heff2_flops(st1, st2, dl, dr)
    got = _apply_gpu(H, ctx, th, 2)
    ref = symm.run_stage(st2, symm.run_stage(st1, Lenv, th), Renv, "n", "t")    # the pinned lists, executed
    for k in th:
        ref.setdefault(k, np.zeros_like(th[k]))
    e, w = rel_err(got, ref, weighted=False), _per_block_worst(got, {k: v for k, v in ref.items() if np.any(v)})
    print("abelian chi=4096: %d blocks, %.3g GFLOP, rel. Frobenius %.2e, worst block %.2e" % (len(th), ctx.heff_flops() * 1e-9, e, w))
    assert e < TOL_APPLY and w < TOL_APPLY
    ctx.mps_destroy(mps)


def test_next4_abelian_tdvp_L8_vs_dense_oracle(H, actx):
    """U(1) x U(1) two-site TDVP on the L = 8 Neel quench (config 1's problem) against the DENSE oracle O-D
    (oracle/dense_tdvp.DenseTDVP, pinned against ED): untruncated, the symmetric and the dense algorithm are the
    same computation, so n_up, n_dn, double occupancy agree to <= 1e-8 after every step (<n_i> is computed from
    the occupation numbers of the four site states here, not fixed by the representation; it stays 1 by the
    particle-hole symmetry of the quench); norm and energy (Eq. (1) as it stands) are conserved."""
    from oracle import dense_tdvp as dtv
    ctx = actx
    L, dt, m = 8, 0.05, 10
    ref = dtv.DenseTDVP(L, 1.0, 4.0, krylov_dim=m)
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_init_neel(mpo, L)
    worst = 0.0
    for step in range(12):
        ref.step(dt)
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=256, eps_trunc=-1.0)
        o, g = ref.observables(), ctx.measure_local(mps, L)
        worst = max(worst, np.abs(g["sz"] - 0.5 * (o["n_up"] - o["n_dn"])).max(), np.abs(g["docc"] - o["docc"]).max(),
                    np.abs(g["n"] - (o["n_up"] + o["n_dn"])).max())
        gg = ctx.measure_global(mpo, mps)
        assert abs(gg["norm2"] - 1) < 1e-10 and abs(gg["energy"]) < 1e-9       # <Neel|H|Neel> = 0 for Eq. (1)
    print("abelian TDVP L=8 vs dense oracle: max observable difference %.1e, chi %s" % (worst, ctx.tdvp2_last_stats()["chi_full"]))
    assert worst < 1e-8, worst
    ctx.mps_destroy(mps)


# ------------------------------------------------------------------ H6 / H8 kernels on their own
@pytest.mark.parametrize("n", [300_001, 1_500_003, 4_700_011])
def test_vector_kernels_and_block_copy_vs_oracle(H, ctx, n):
    """H6 / H8 directly (not through a Lanczos run): weighted dot, the unnormalised three-term update with its fused
    norm, the linear combination and the scaled block copy (plain and transposing) against oracle/vecops.py, on
    vectors of 0.3, 1.5 and 4.7 Mi elements -- one in each chunk-length class of the library (1024 / 2048 / 8192) --
    cut into ragged blocks (lengths 1 ... 200 000) with weights 1 ... 5."""
    torch = _torch()
    rng = np.random.default_rng(n)
    lens, left = [], n
    while left > 0:
        k = int(min(left, rng.choice([1, 7, 1023, 1024, 1025, 8191, 8193, 50_000, 200_000])))
        lens.append(k)
        left -= k
    wts = [int(rng.integers(1, 6)) for _ in lens]
    x, y, w = (rng.standard_normal(n) + 1j * rng.standard_normal(n) for _ in range(3))
    dx, dy = _dev(x), _dev(y)
    ref = vecops.wdot(lens, wts, x, y)
    got = ctx.fh_vec_wdot(lens, wts, dx, dy)
    assert abs(got - ref) < 1e-12 * abs(ref) + 1e-9, (got, ref)
    assert ctx.fh_vec_wdot(lens, wts, dx, dy) == got                      # fixed reduction order: same bits
    for (bj2, bjm2, prev) in ((-1.0, -1.0, None), (2.5, -1.0, y), (2.5, 0.7, y)):
        dw = _dev(w)
        ru, rn = vecops.lanczos_update(lens, wts, 1.3, bj2, bjm2, 1e-12, x, prev, w)
        gn = ctx.fh_vec_lanczos_update(lens, wts, 1.3, bj2, bjm2, 1e-12, dx, dy if prev is not None else None, dw)
        assert np.abs(dw.cpu().numpy() - ru).max() < 1e-13 * np.abs(ru).max() and abs(gn / rn - 1) < 1e-12
    m = 7
    V = rng.standard_normal((m, n)) + 1j * rng.standard_normal((m, n))
    coef = rng.standard_normal(m) + 1j * rng.standard_normal(m)
    dV, dz = _dev(V), torch.empty(n, dtype=torch.complex128, device="cuda")
    ctx.fh_vec_lincomb(coef, dV, n, dz)
    rl = vecops.lincomb(coef, V)
    assert np.abs(dz.cpu().numpy() - rl).max() < 1e-13 * np.abs(rl).max()
    # block copies: ragged blocks out of a strided source into a strided destination, plain and transposed
    blocks, so, do = [], 0, 0
    for b in range(40):
        r, c = int(rng.integers(1, 130)), int(rng.integers(1, 130))
        ls, tr = c + int(rng.integers(0, 5)), int(b % 2)
        ld = (r if tr else c) + int(rng.integers(0, 5))
        blocks.append((so, do, r, c, ls, ld, tr, float(rng.uniform(0.5, 2.0))))
        so += r * ls
        do += (c if tr else r) * ld
    assert so <= n and do <= n
    dst_ref = np.zeros(n, dtype=complex)
    vecops.copy_blocks(blocks, x, dst_ref)
    ddst = torch.zeros(n, dtype=torch.complex128, device="cuda")
    cols = list(zip(*blocks))
    ctx.fh_copy_blocks(*cols, dx, ddst)
    assert np.array_equal(ddst.cpu().numpy() == 0, dst_ref == 0)
    assert np.abs(ddst.cpu().numpy() - dst_ref).max() < 1e-15 * np.abs(dst_ref).max() + 1e-300


# ------------------------------------------------------------------ edge cases and errors
def test_edge_cases_and_error_codes(H, ctx):
    B = H.binding
    with pytest.raises(B.FhError):
        ctx.fh_mpo_build(7, 1.0, 4.0)                 # odd L
    with pytest.raises(B.FhError):
        ctx.fh_mpo_build(0, 1.0, 4.0)                 # empty chain
    mpo = ctx.fh_mpo_build(2, 1.0, 4.0)
    x = _torch().zeros(4, dtype=_torch().complex128, device="cuda")
    with pytest.raises(B.FhError):
        ctx.heff_apply(x, x.clone())                  # no plan yet
    # smallest chain: L=2 Neel, one bond, every block 1x1; singlet-sector two-site problem
    mps = ctx.mps_init_neel(mpo, 2)
    ctx.heff_plan(mpo, mps, 0, 2)
    lab, dm, ne = ctx.heff_layout(2)
    ref = stv.SymmTDVP(2, 1.0, 4.0, krylov_dim=4)
    th = ref._theta(0)
    assert ne == sum(v.size for v in th.values())
    want = symm.heff2_apply(ref.Lenv[0], ref.Renv[2], th, ref.W[0], ref.W[1])
    got = _apply_gpu(H, ctx, th, 2)
    assert rel_err(got, want) < TOL_APPLY
    # getters refuse a buffer smaller than the tensor instead of writing past it (capacity argument of the C ABI)
    buf = np.zeros(64, dtype=np.complex128)
    rc = B.lib.mps_get_site(ctx.h, mps, 0, buf.ctypes.data, 0, 0)
    assert rc == -1 and b"smaller" in B.lib.fh_last_error(ctx.h) and not buf.any()
    rc = B.lib.env_get(ctx.h, mps, 1, 1, buf.ctypes.data, 0, 0)
    assert rc == -1 and b"smaller" in B.lib.fh_last_error(ctx.h)
    assert B.lib.mps_get_site(ctx.h, mps, 0, buf.ctypes.data, 64, 0) == 0 and buf.any()
    with pytest.raises(B.FhError):
        ctx.heff_plan(mpo, mps, 1, 2)                 # bond out of range
    with pytest.raises(B.FhError):
        ctx.mps_set_bond(mps, 1, {(0, 0): 1})         # violates the parity rule q + 2j = k (mod 2)
    ctx.mps_destroy(mps)
    # arena exhaustion is reported, not fatal
    small = B.Context(1 << 20)
    mpo2 = small.fh_mpo_build(60, 1.0, 4.0)
    with pytest.raises(B.FhError, match="arena"):
        H.build_central_bond(small, mpo2, 4096, 60)
    small.close()


# ------------------------------------------------------------------ NEXT-3: split precision (3 x TF32 on tcgen05)
def _split_case(rng, M, N, Ks, conj, tA, tB):
    """Segments with every operand orientation the task lists use; returns (binding segments, oracle segments, A, B)."""
    segs, osegs, Abuf, Bbuf, ao, bo = [], [], [], [], 0, 0
    for K in Ks:
        A, Bm = _rand(rng, M, K), _rand(rng, K, N)
        al = float(rng.uniform(0.5, 2.0)) * (1 if rng.random() < 0.5 else -1)
        Abuf.append(np.ascontiguousarray(A.T).ravel() if tA else A.ravel())
        Bbuf.append(np.ascontiguousarray(Bm.T).ravel() if tB else Bm.ravel())
        segs.append((K, al, ao, 1 if tA else K, M if tA else 1, bo, 1 if tB else N, K if tB else 1))
        osegs.append((al, A.conj() if conj else A, Bm))
        ao += M * K
        bo += K * N
    cat = lambda b: np.concatenate(b) if b else np.zeros(1, dtype=np.complex128)
    return segs, osegs, cat(Abuf), cat(Bbuf)


@pytest.mark.parametrize("M,N,Ks,conj,tA,tB", [
    (128, 128, [16], 0, 0, 0), (128, 128, [8], 0, 0, 0), (128, 16, [16], 1, 0, 0), (64, 48, [20], 0, 0, 0),
    (1, 1, [1], 0, 0, 0), (129, 257, [1, 3, 17], 1, 1, 0), (100, 77, [50, 13], 1, 0, 1),
    (300, 500, [129, 64, 200], 0, 1, 1), (57, 33, [], 0, 0, 0), (1000, 1000, [512, 300], 0, 0, 0)])
def test_next3_zgemm_split_vs_oracle(H, ctx, M, N, Ks, conj, tA, tB):
    """fh_zgemm_split (tcgen05.mma kind::tf32, accumulators in tensor memory) against oracle/splitprec.py, element by
    element: |C - zgemm_split| <= the float32-accumulation bound K 2^-23 S, hence |C - exact| <= that + the split
    bound 3.1 2^-22 S; nothing outside the M x N block (leading dimension N + 3) is touched.  Cases: one tile / one
    k-step, ragged tiles and tails in all three dimensions, several segments, every operand orientation of the task
    lists (A as stored / transposed / conjugated, B as stored / transposed), an output without segments, 8 x 8
    tiles with 51 chunks."""
    from oracle import splitprec as sp
    torch = _torch()
    rng = np.random.default_rng(1000 * M + N)
    segs, osegs, A, B = _split_case(rng, M, N, Ks, conj, tA, tB)
    ldc = N + 3
    dC = torch.full((M * ldc,), 7 + 7j, dtype=torch.complex128, device="cuda")
    ctx.fh_zgemm_split(M, N, segs, conj, _dev(A), _dev(B), dC, ldc)
    C = dC.cpu().numpy().reshape(M, ldc)
    assert np.all(C[:, N:] == 7 + 7j)
    C = C[:, :N]
    if not Ks:
        assert not C.any()
        return
    exact = sum(al * (a @ b) for al, a, b in osegs)
    acc, spl = sp.split_bounds(osegs, M, N)
    assert np.all(np.abs(C - sp.zgemm_split(osegs, M, N)) <= acc)
    assert np.all(np.abs(C - exact) <= acc + spl)
    e = np.linalg.norm(C - exact) / np.linalg.norm(exact)
    assert e < 2e-5 and (sum(Ks) < 64 or e > 1e-9)               # single-precision class, and really the split path
    dC2 = torch.empty_like(dC)
    ctx.fh_zgemm_split(M, N, segs, conj, _dev(A), _dev(B), dC2, ldc)
    assert bool((dC2.view(torch.float64).reshape(M, ldc, 2)[:, :N] == dC.view(torch.float64).reshape(M, ldc, 2)[:, :N]).all())


@pytest.mark.parametrize("chi", [1024, 4096])
def test_next3_split_apply_vs_oracle_all_blocks(H, chi):
    """FH_OPT_PRECISION = 1 on the plan bench.py times (chi = 4096) and on config 2: the two-site apply through
    the split-precision kernels (same task lists, layout and intermediate as the FP64 apply) against the FP64
    oracle on ALL output blocks.  Tolerance: two chained stages, each within K_total 2^-23 of its operands'
    absolute sums (oracle/splitprec.py); K_total <= ~900 here, so 1e-4 relative Frobenius bounds it with room;
    measured 2e-6 ... 8e-6.  The FP64 apply of the same plan stays at 1e-11 when the option is switched back."""
    L, c = 60, 29
    o = central_bond(chi, L)
    dims, W = o["dims"], o["W"]
    ctx = H.binding.Context(int(max(1 << 30, 64.0 * chi * chi)))
    try:
        mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
        mps, gdims = H.build_central_bond(ctx, mpo, chi, L)
        th = fi.theta_random(fi.SEED, c, dims[c], dims[c + 2])
        ref = symm.heff2_apply(o["Lenv"], o["Renv"], th, W[c], W[c + 1])
        ctx.heff_plan(mpo, mps, c, 2)
        lab, dm, ne = ctx.heff_layout(2)
        x = H.to_planned(ctx, H.flatten(th, lab, dm, H.theta_key))
        y = _torch().empty_like(x)
        ctx.fh_set_option(ctx.OPT_PRECISION, 1)
        ctx.heff_apply(x, y)
        got = H.unflatten(H.from_planned(ctx, y), lab, dm, H.theta_key)
        e, w = rel_err(got, ref), _per_block_worst(got, ref)
        print("split-precision apply chi=%d: rel. Frobenius %.2e, worst block %.2e" % (chi, e, w))
        assert 1e-9 < e < 1e-4 and w < 1e-3
        ctx.fh_set_option(ctx.OPT_PRECISION, 0)
        ctx.heff_apply(x, y)
        assert rel_err(H.unflatten(H.from_planned(ctx, y), lab, dm, H.theta_key), ref) < TOL_APPLY
    finally:
        ctx.close()


def test_next3_split_tdvp_gate_L8(H, ctx):
    """The paper's acceptance test of reduced precision (abs delta <n_up> < 1e-3) on config 1's
    problem: 20 two-site TDVP steps of the L = 8 Neel quench with every H_eff application of the Lanczos steps in
    split precision, against the dense FP64 oracle."""
    from oracle import dense_tdvp as dtv
    L, dt, m = 8, 0.05, 10
    ref = dtv.DenseTDVP(L, 1.0, 4.0, krylov_dim=m)
    ctx.fh_set_option(ctx.OPT_PRECISION, 1)
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_init_neel(mpo, L)
    worst = 0.0
    for step in range(20):
        ref.step(dt)
        ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=m, chi_max_full=256, eps_trunc=-1.0)
        o, g = ref.observables(), ctx.measure_local(mps, L)
        worst = max(worst, np.abs(g["sz"] - 0.5 * (o["n_up"] - o["n_dn"])).max(), np.abs(g["docc"] - o["docc"]).max())
    gg = ctx.measure_global(mpo, mps)
    print("split-precision TDVP L=8, 20 steps: max |delta <S^z_i>|, |delta <n_up n_dn>| = %.1e, norm^2 - 1 = %.1e" % (worst, gg["norm2"] - 1))
    assert 1e-12 < worst < 1e-3 and abs(gg["norm2"] - 1) < 1e-3
    ctx.mps_destroy(mps)


@pytest.mark.parametrize("mode", ["su2", "u1u1"])
def test_next3_split_apply_small_chains_both_modes(H, mode):
    """FH_OPT_PRECISION = 1 on ragged tiny blocks (1 ... 11 columns: every 128 x 128 tile is mostly padding, many
    outputs have no contribution at the chain ends) in both symmetry modes: the two-site apply on every bond of a
    random L = 6 chain against the FP64 oracle, relative Frobenius <= 1e-5 (K_total <= ~60 here: measured ~1e-6),
    while the one-site apply of the same context stays FP64 (<= 1e-11)."""
    rng = np.random.default_rng(77)
    L = 6
    ctx = H.binding.Context(1 << 28)
    try:
        if mode == "u1u1":
            import fh_inputs.abelian as fab
            from oracle import abelian as ab
            ctx.fh_set_option(ctx.OPT_SYMMETRY, 1)
            dims = [{k: min(v, int(rng.integers(1, 12))) for k, v in d.items()} for d in fab.chain_dims(10 ** 6, L)]
            A = [{k: _rand(rng, dims[i][k[0]], dims[i + 1][k[2]]) for k in ab.site_keys(dims[i], dims[i + 1])} for i in range(L)]
            W = [ab.mpo_elements(1.0, 4.0)] * L
            mod, left0, right0 = ab, ab.boundary_left(), ab.boundary_right()
            tkeys = ab.theta_keys
        else:
            dims, A = _small_chain(rng, L, 11)
            W = [symm.mpo_reduced(i, 1.0, 4.0) for i in range(L)]
            mod, left0, right0 = symm, symm.boundary_left(), symm.boundary_right()
            tkeys = symm.theta_keys
        Le, Re = [left0], [None] * (L + 1)
        for i in range(L):
            Le.append(mod.env_update_left(Le[i], A[i], W[i]))
        Re[L] = right0
        for i in range(L - 1, -1, -1):
            Re[i] = mod.env_update_right(Re[i + 1], A[i], W[i])
        mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
        mps = ctx.mps_create(L)
        for i in range(L):
            H.set_site(ctx, mps, i, A[i], dims[i], dims[i + 1])
        for i in range(L):
            ctx.env_update_left(mpo, mps, i)
        for i in range(L - 1, -1, -1):
            ctx.env_update_right(mpo, mps, i)
        ctx.fh_set_option(ctx.OPT_PRECISION, 1)
        worst = 0.0
        for i in range(L - 1):
            th = {k: _rand(rng, dims[i][k[0]], dims[i + 2][k[4]]) for k in tkeys(dims[i], dims[i + 2])}
            ref = mod.heff2_apply(Le[i], Re[i + 2], th, W[i], W[i + 1])
            ctx.heff_plan(mpo, mps, i, 2)
            e = rel_err(_apply_gpu(H, ctx, th, 2), ref, weighted=(mode == "su2"))
            assert 1e-12 < e < 1e-5, (i, e)
            worst = max(worst, e)
        for i in range(L):
            ref = mod.heff1_apply(Le[i], Re[i + 1], A[i], W[i])
            ctx.heff_plan(mpo, mps, i, 1)
            assert rel_err(_apply_gpu(H, ctx, A[i], 1), ref, weighted=(mode == "su2")) < TOL_APPLY, i
        print("split-precision apply, small chain, %s: worst rel. Frobenius %.1e" % (mode, worst))
    finally:
        ctx.close()
