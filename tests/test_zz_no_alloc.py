"""fh_vec_wdot_static (include/fh_b200.h): the weighted inner product of two block vectors (F-6, the reduction
of H6) for callers that may not call cudaMalloc.  Its scratch is one file-scope device array of
FH_STATIC_SCRATCH_BYTES; the test compares it with the existing path (fh_vec_wdot, which takes its partial sums
from a pool of the context) within the tolerance tests/test_gpu_parity.py uses for that kernel, on two calls in
a row that leave different contents behind in the shared array.

The file name sorts last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def B():
    import paper_2606_04771_b200 as pkg
    pkg.build()
    return pkg.binding


def _case(seed, n, weights_hi):
    rng = np.random.default_rng(seed)
    lens, left = [], n
    while left > 0:
        k = int(min(left, rng.choice([0, 1, 7, 255, 256, 1023, 1024, 1025, 8193, 50_000, 200_000])))
        lens.append(k)
        left -= k
    wts = [int(rng.integers(1, weights_hi)) for _ in lens]
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    y = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    return np.array(lens, dtype=np.int64), np.array(wts, dtype=np.int32), x, y


def test_static_entry_point_rejects_sizes_beyond_the_fixed_array(B):
    """The limits are checked before anything touches a device, so this runs without one."""
    big = B.STATIC_MAX_BLOCKS + 1
    rc = B.lib.fh_vec_wdot_static(1024, big, 8, 8, 8, 8, 8, None)
    assert rc == -1 and b"FH_STATIC_MAX_BLOCKS" in B.lib.fh_static_last_error()
    rc = B.lib.fh_vec_wdot_static(B.STATIC_MAX_ELEMS + 1, 4, 8, 8, 8, 8, 8, None)
    assert rc == -1 and b"FH_STATIC_MAX_ELEMS" in B.lib.fh_static_last_error()
    assert B.lib.fh_vec_wdot_static(0, 4, 8, 8, 8, 8, 8, None) == -1
    assert B.lib.fh_vec_wdot_static(16, 4, None, 8, 8, 8, 8, None) == -1


@pytest.mark.gpu
def test_static_wdot_matches_existing_path_on_two_calls_in_a_row(B):
    import torch
    ctx = B.Context(1 << 28)
    try:
        B.fh_static_setup()
        B.fh_static_setup()                                   # once per device: the second call is a no-op
        res = torch.full((2,), 7.0, dtype=torch.float64, device="cuda")
        stream = torch.cuda.current_stream().cuda_stream
        free_before = None
        # a long vector first (4.7 Mi elements: ranges longer than 1024 per CTA, every CTA slot of the scratch
        # array written), then a short one with another block table: stale prefixes / partials must not leak in
        for call, (seed, n, hi) in enumerate(((11, 4_700_321, 6), (12, 300_007, 4), (13, 1, 3))):
            lens, wts, x, y = _case(seed, n, hi)
            dx, dy = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
            dl, dw = torch.from_numpy(lens).cuda(), torch.from_numpy(wts).cuda()
            want = ctx.fh_vec_wdot(lens, wts, dx, dy)         # the existing path
            torch.cuda.synchronize()
            if call == 1:
                free_before = torch.cuda.mem_get_info()[0]
            B.fh_vec_wdot_static(n, len(lens), dl, dw, dx, dy, res, stream)
            torch.cuda.synchronize()
            if call == 1:                                     # no device memory taken by the call
                assert torch.cuda.mem_get_info()[0] == free_before
            got = complex(*res.cpu().tolist())
            assert abs(got - want) < 1e-12 * abs(want) + 1e-9, (call, got, want)
            B.fh_vec_wdot_static(n, len(lens), dl, dw, dx, dy, res, stream)
            torch.cuda.synchronize()
            assert complex(*res.cpu().tolist()) == got        # fixed summation order: same bits
        # a block table that does not add up to n gives NaN, not a wrong number; the next good call is clean
        lens, wts, x, y = _case(14, 70_001, 5)
        dx, dy = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
        dl, dw = torch.from_numpy(lens).cuda(), torch.from_numpy(wts).cuda()
        bad = dl.clone()
        bad[0] += 1
        B.fh_vec_wdot_static(70_001, len(lens), bad, dw, dx, dy, res, stream)
        torch.cuda.synchronize()
        assert torch.isnan(res).all()
        B.fh_vec_wdot_static(70_001, len(lens), dl, dw, dx, dy, res, stream)
        torch.cuda.synchronize()
        want = ctx.fh_vec_wdot(lens, wts, dx, dy)
        assert abs(complex(*res.cpu().tolist()) - want) < 1e-12 * abs(want) + 1e-9
    finally:
        ctx.close()
