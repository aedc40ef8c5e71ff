"""CPU tests (-m "not gpu") of the library's host symmetry layer: the shared library loads,
exports every symbol include/fh_b200.h declares, its closed-form recoupling coefficients agree
with the oracle's CG-sum definitions, and its task lists equal the oracle's bit for bit."""
import os
import random
import re

import numpy as np
import pytest

import fh_inputs as fi
from oracle import su2, symm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    import paper_2606_04771_b200 as pkg
    pkg.build()
    return pkg.binding


def test_library_exports_every_declared_symbol(binding):
    hdr = open(os.path.join(ROOT, "include", "fh_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b([a-z_0-9]+)\s*\(", hdr))
    names -= {"defined", "sizeof"}
    decl = {n for n in names if re.search(r"\b(int|void|double|int64_t|const char\*)\s+\*?\s*%s\s*\(" % n, hdr)}
    assert len(decl) >= 38
    for n in sorted(decl):
        assert hasattr(binding.lib, n), n
    assert set(binding.EXPORTS) == decl


def test_closed_form_coefficients_match_oracle(binding):
    rnd = random.Random(5)
    n = 0
    while n < 300:
        ta = rnd.randint(0, 9)
        ts, tsp, tk, tr = (rnd.choice([0, 1]) for _ in range(4))
        tkp = rnd.choice(range(abs(tk - tr), tk + tr + 1, 2))
        tc = rnd.choice(range(abs(ta - ts), ta + ts + 1, 2))
        tap = rnd.choice(range(abs(ta - tk), ta + tk + 1, 2))
        tcp = rnd.choice(range(abs(tap - tsp), tap + tsp + 1, 2))
        t = (ta, ts, tc, tk, tr, tkp, tap, tsp, tcp)
        assert abs(binding.fh_coef_left(*t) - su2.coef_left(*t)) < 1e-13, t
        assert abs(binding.fh_coef_right(*t) - su2.coef_right(*t)) < 1e-13, t
        n += 1


def _compare(binding, site, nsite, dims_l, dims_r, Lk, Rk, t_h=1.0, U=4.0):
    W1, W2 = symm.mpo_reduced(site, t_h, U), symm.mpo_reduced(site + 1, t_h, U)
    if nsite == 2:
        vk = symm.theta_keys(dims_l, dims_r)
        st1, st2 = symm.heff2_tasks(Lk, Rk, vk, W1, W2)
    else:
        vk = symm.site_keys(dims_l, dims_r)
        st1, st2 = symm.heff1_tasks(Lk, Rk, vk, W1)
    o1 = symm.task_tuples(st1, list(st1), Lk, vk)
    o2 = symm.task_tuples(st2, vk, list(st1), Rk)
    (t1, a1, n1, f1), (t2, a2, n2, f2) = binding.fh_host_plan(site, nsite, t_h, U, dims_l, dims_r, Lk, Rk)
    assert n1 == len(st1) and n2 == len(vk)
    assert t1.shape == o1[0].shape and (t1 == o1[0]).all()          # bit-exact integer tuples
    assert t2.shape == o2[0].shape and (t2 == o2[0]).all()
    assert np.abs(a1 - o1[1]).max() < 1e-13 and np.abs(a2 - o2[1]).max() < 1e-13
    if nsite == 2:
        assert f1 + f2 == symm.heff2_flops(st1, st2, dims_l, dims_r)
    return len(a1), len(a2)


def test_task_lists_bit_exact_small_chain(binding):
    rng = np.random.default_rng(2)
    L = 6
    tabs = fi.reachable_tables(L)
    dims = [{sec: int(rng.integers(1, 5)) for sec in tabs[k]} for k in range(L + 1)]
    for site in range(L - 1):
        Lk = symm.env_keys(dims[site], dims[site])
        Rk = symm.env_keys(dims[site + 2], dims[site + 2])
        _compare(binding, site, 2, dims[site], dims[site + 2], Lk, Rk)
    for site in range(L):
        Lk = symm.env_keys(dims[site], dims[site])
        Rk = symm.env_keys(dims[site + 1], dims[site + 1])
        _compare(binding, site, 1, dims[site], dims[site + 1], Lk, Rk)


def test_task_lists_bit_exact_config2_shape(binding):
    """BASELINE config 2's sector structure at reduced chi (central bond of L=60)."""
    dl, dr = fi.gaussian_profile(29, 256), fi.gaussian_profile(31, 256)
    Lk, Rk = symm.env_keys(dl, dl), symm.env_keys(dr, dr)
    n1, n2 = _compare(binding, 29, 2, dl, dr, Lk, Rk)
    assert n1 > 500 and n2 > 500


@pytest.mark.parametrize("chi,profile", [(256, "gaussian"), (1024, "gaussian"), (4096, "gaussian"), (0, "table_s2")])
def test_unit_lists_tile_every_output_exactly_once(binding, chi, profile):
    """The warp-unit decomposition the grouped ZGEMM launches, checked on the host:
    every element of every output block is covered by exactly one unit, units have a compiled shape
    (mt * nt <= 16, mt, nt <= 8), only the last 8-sliver of a block is padded, the launch order is
    heaviest first, and the padded DMMA count is what the units add up to."""
    L, c = 60, 29
    dims = fi.chain_dims(chi, L, profile, (1, 24))
    dl, dr = dims[c], dims[c + 2]
    Lk, Rk = sorted(fi.env_block_keys(dl, dl)), sorted(fi.env_block_keys(dr, dr))
    binding.fh_host_plan(c, 2, 1.0, 4.0, dl, dr, Lk, Rk)
    for stage in (1, 2):
        units, outs, padded = binding.fh_host_get_units(stage)
        assert len(units) > 0 and (units[:, 0] >= 0).all()
        cover = [np.zeros(((m + 7) // 8, (n + 7) // 8), dtype=np.int32) for m, n, _ in outs]
        work, total = [], 0
        for o, m0, n0, mt, nt, steps in units:
            M, N, st = outs[o]
            assert 1 <= mt <= 8 and 1 <= nt <= 8 and mt * nt <= 16
            assert m0 % 8 == 0 and n0 % 8 == 0 and steps == st
            assert m0 + 8 * mt <= (M + 7) // 8 * 8 and n0 + 8 * nt <= (N + 7) // 8 * 8   # padding < 8
            cover[o][m0 // 8:m0 // 8 + mt, n0 // 8:n0 // 8 + nt] += 1
            work.append(mt * nt * max(1, steps))
            total += 4 * mt * nt * steps
        for o, cv in enumerate(cover):
            if outs[o][0] > 0 and outs[o][1] > 0:
                assert (cv == 1).all(), (stage, o)
        assert all(a >= b for a, b in zip(work, work[1:]))          # heaviest first
        assert total == padded
        exact = sum(int(m) * int(n) for m, n, _ in outs)             # sanity: padded area < 2x exact for these profiles
        assert sum(int(cv.size) * 64 for cv in cover) < 4 * exact + 64 * len(outs) * 4


@pytest.mark.parametrize("chi,grid", [(1024, 148), (4096, 148), (4096, 7)])
def test_split_precision_tile_lists_and_panel_images(binding, chi, grid):
    """Host side of the split-precision kernel (zgemm_tc.cu, NEXT-3): the 128 x 128 tiles cover every element of
    every merged output exactly once and carry sum ceil(K / 16) chunks; the CTA ranges partition the list, each
    CTA's tiles are in non-increasing weight order and the dealing is balanced to within one tile's weight of the
    mean; the panel images of the static operand (stage 1: op(A), stage 2: op(B)) lie inside the image buffer, are
    32-KB aligned, no image serves two operand blocks and segments that read the same block share one."""
    L, c = 60, 29
    dims = fi.chain_dims(chi, L, "gaussian", (1, 1))
    dl, dr = dims[c], dims[c + 2]
    Lk, Rk = sorted(fi.env_block_keys(dl, dl)), sorted(fi.env_block_keys(dr, dr))
    binding.fh_host_plan(c, 2, 1.0, 4.0, dl, dr, Lk, Rk)
    for stage in (1, 2):
        _, outs, _ = binding.fh_host_get_units(stage)
        tiles, cb, img, opd, nchunk, nbytes = binding.fh_host_get_tc_tiles(stage, grid, stage)
        assert len(tiles) > 0 and (tiles[:, 0] >= 0).all()
        cover = [np.zeros((m, n), dtype=np.int8) for m, n, _ in outs]
        for o, m0, n0, h, w, ch in tiles:
            M, N, _ = outs[o]
            assert m0 % 128 == 0 and n0 % 128 == 0 and 1 <= h <= 128 and 1 <= w <= 128
            assert h == min(128, M - m0) and w == min(128, N - n0)
            cover[o][m0:m0 + h, n0:n0 + w] += 1
        assert all((cv == 1).all() for cv in cover)
        per_out = {}
        for o, *_rest, ch in tiles:
            per_out.setdefault(o, set()).add(int(ch))
        assert all(len(v) == 1 for v in per_out.values())              # every tile of an output has that output's chunks
        assert cb[0] == 0 and cb[-1] == len(tiles) and (np.diff(cb) >= 0).all() and len(cb) == grid + 1
        wt = tiles[:, 5].astype(np.int64) * (128 + (tiles[:, 4] + 15) // 16 * 16) + 64
        loads = np.array([wt[cb[b]:cb[b + 1]].sum() for b in range(grid)])
        for b in range(grid):
            seg = wt[cb[b]:cb[b + 1]]
            assert (np.diff(seg) <= 0).all()
        assert loads.max() - loads.min() <= wt.max()                   # greedy dealing: spread below one tile
        used = img >= 0                                                  # -1: segment of an output merged into its neighbour
        img, opd = img[used], opd[used]
        assert nbytes == nchunk * 32768 and (img % 32768 == 0).all() and (img < nbytes).all() and used.sum() > 0
        # an image serves one operand block only (segments that read the same block with the same extent share it;
        # a block read as part of a wider merged operand has its own image), and images are shared at all
        by_img = {}
        assert len(img) == len(opd) > 0
        for k, off in zip(opd.tolist(), img.tolist()):
            by_img.setdefault(off, set()).add(k)
        assert all(len(v) == 1 for v in by_img.values())
        assert len(by_img) < len(img)


def test_zero_site_task_lists_match_oracle(binding):
    """NEXT-1: the zero-site apply K C = sum_w L C R^T.  Integer task tuples of both stages equal the
    oracle's (oracle/symm.heff0_tasks) bit for bit, all coefficients are exactly 1, flops agree."""
    dims = fi.chain_dims(256, 60, "gaussian", (1, 1))
    dl = dims[30]
    dr = {k: max(1, v - 1) for k, v in dl.items()}          # ket side slightly smaller: rectangular C blocks
    Lk, Rk = sorted(fi.env_block_keys(dl, dl)), sorted(fi.env_block_keys(dr, dr))
    ck = sorted(dl)
    st1, st2 = symm.heff0_tasks(Lk, Rk, ck)
    o1 = symm.task_tuples(st1, list(st1), Lk, ck)
    o2 = symm.task_tuples(st2, ck, list(st1), Rk)
    (t1, a1, n1, f1), (t2, a2, n2, f2) = binding.fh_host_plan(30, 0, 1.0, 4.0, dl, dr, Lk, Rk)
    assert n1 == len(st1) and n2 == len(ck)
    assert t1.shape == o1[0].shape and (t1 == o1[0]).all()
    assert t2.shape == o2[0].shape and (t2 == o2[0]).all()
    assert (a1 == 1.0).all() and (a2 == 1.0).all()
    fl = sum(8 * dl[xk[0]] * dl[xk[2]] * dr[xk[2]] for xk in st1) + \
        sum(8 * dl[o] * dr[seg[0][2]] * dr[o] for o, segs in st2.items() for seg in segs)
    assert f1 + f2 == fl


def test_abelian_mode_task_lists_bit_exact(binding):
    """NEXT-4, U(1) x U(1) mode of the host layer (fh_host_set_symmetry(1)): W = 6 MPO, four site states, packed
    charges.  Integer task tuples of both stages equal oracle/abelian.heff2_tasks bit for bit on the central bond
    of the abelian profile (chi = 64, 1024), alpha = the MPO elements exactly, flops equal; the unit lists tile
    every output once."""
    import fh_inputs.abelian as fab
    from oracle import abelian as ab
    assert binding.lib.fh_host_set_symmetry(1) == 0
    try:
        for chi in (64, 1024):
            dl, dr = fab.profile(29, chi), fab.profile(31, chi)
            Lk, Rk = ab.env_keys(dl, dl), ab.env_keys(dr, dr)
            assert Lk == fab.env_block_keys(dl, dl)
            W = ab.mpo_elements(1.0, 4.0)
            vk = ab.theta_keys(dl, dr)
            st1, st2 = ab.heff2_tasks(Lk, Rk, vk, W, W)
            o1 = symm.task_tuples(st1, list(st1), Lk, vk)
            o2 = symm.task_tuples(st2, vk, list(st1), Rk)
            (t1, a1, n1, f1), (t2, a2, n2, f2) = binding.fh_host_plan(29, 2, 1.0, 4.0, dl, dr, Lk, Rk)
            assert n1 == len(st1) and n2 == len(vk)
            assert t1.shape == o1[0].shape and (t1 == o1[0]).all() and t2.shape == o2[0].shape and (t2 == o2[0]).all()
            assert (a1 == o1[1]).all() and (a2 == o2[1]).all()
            assert f1 + f2 == ab.heff2_flops(st1, st2, dl, dr)
            for stage in (1, 2):
                units, outs, padded = binding.fh_host_get_units(stage)
                cover = [np.zeros(((m + 7) // 8, (n + 7) // 8), dtype=np.int32) for m, n, _ in outs]
                for o, m0, n0, mt, nt, steps in units:
                    cover[o][m0 // 8:m0 // 8 + mt, n0 // 8:n0 // 8 + nt] += 1
                assert all((cv == 1).all() for cv in cover)
    finally:
        binding.lib.fh_host_set_symmetry(0)


def test_host_only_entry_points_refuse_null_handles(binding):
    """fh_plan_cache_stats / fh_plan_cache_limit / fh_enable_timers are host-only calls: without a GPU they can
    still be reached, and a NULL handle or a negative limit is FH_EINVAL (include/fh_b200.h), never a crash."""
    import ctypes as C
    lib = binding.lib
    a = C.c_int64(7)
    assert lib.fh_plan_cache_stats(None, C.byref(a), None, None) < 0 and a.value == 7
    assert lib.fh_plan_cache_limit(None, 0) < 0
    assert lib.fh_enable_timers(None, 0) < 0
