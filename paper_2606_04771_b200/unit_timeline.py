"""Per-unit timeline of one heff_apply (developer tool, not used by tests or bench).

Builds libfh_b200_trace.so (the library compiled with -DFH_UNIT_TRACE: every warp unit of the grouped ZGEMM
stamps globaltimer at entry and exit, its SM and its warp slot), runs the BASELINE heff_apply workload once with
the trace on and prints, per stage: span, DMMA-issue ideal, warp-slot residency and tensor-pipe utilisation over
time, the gaps between consecutive units of a warp slot, and unit durations by size class.

    python -m paper_2606_04771_b200.unit_timeline [chi] [gaussian|table_s2]
"""
import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SM_COUNT, SMSP_PER_SM, DMMA_CYCLES = 148, 4, 16


def capture(chi, profile):
    import importlib
    os.environ["FH_B200_LIB"] = importlib.import_module(".build", __package__).build(trace=True)
    import torch
    import fh_inputs as fi
    from . import harness as H
    lib = H.binding.lib
    lib.fh_debug_unit_trace.argtypes = [C.c_void_p, C.c_size_t]
    lib.fh_debug_unit_trace.restype = None
    lib.fh_debug_unit_trace_used.restype = C.c_size_t
    L, c = 60, 29
    ctx = H.binding.Context(max(16 << 30, 64 * chi * chi))
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps, dims = H.build_central_bond(ctx, mpo, chi, L, profile=profile, table_s2_scale=(1, 6))
    ctx.heff_plan(mpo, mps, c, 2)
    lab, dm, ne = ctx.heff_layout(2)
    th = fi.theta_random(fi.SEED, c, dims[c], dims[c + 2])
    x = torch.from_numpy(H.flatten(th, lab, dm, H.theta_key)).cuda()
    y = torch.empty_like(x)
    for _ in range(5):
        ctx.heff_apply(x, y)
    torch.cuda.synchronize()
    try:
        clock_mhz = float(torch.cuda.clock_rate())      # SM clock right after the warm-up applies, MHz
    except Exception:
        clock_mhz = 1965.0                              # the B200 boost clock bench.py observes under load
    cap = 1 << 20
    buf = torch.zeros(4 * cap, dtype=torch.int64, device="cuda")
    lib.fh_debug_unit_trace(C.c_void_p(buf.data_ptr()), cap)
    ctx.heff_apply(x, y)
    torch.cuda.synchronize()
    n = lib.fh_debug_unit_trace_used()
    lib.fh_debug_unit_trace(None, 0)
    t = buf[:4 * n].cpu().numpy().reshape(n, 4)
    return t, clock_mhz


def report(t, clock_mhz, out=sys.stdout):
    shape, steps = t[:, 3] >> 32, t[:, 3] & 0xffffffff
    dm = 4 * (shape // 16) * (shape % 16) * steps
    # units are listed heaviest first per launch: the second launch starts where the work jumps back up
    n1 = int(np.argmax(np.diff(dm.astype(float)) > 0) + 1)
    t0 = t[:, 0].min()
    for name, sl in (("stage 1 (L x theta -> Z)", slice(0, n1)), ("stage 2 (Z x R^T -> H theta)", slice(n1, None))):
        x = t[sl]
        b, e = (x[:, 0] - t0) / 1e3, (x[:, 1] - t0) / 1e3
        sm, wid = x[:, 2] >> 32, x[:, 2] & 0xffffffff
        d = dm[sl].astype(float)
        slots = SM_COUNT * (int(wid.max()) + 1)
        span0, span1 = b.min(), e.max()
        ideal = d.sum() * DMMA_CYCLES / (SM_COUNT * SMSP_PER_SM) / clock_mhz
        dur = np.maximum(e - b, 1e-3)
        share = d * DMMA_CYCLES / clock_mhz / dur
        print("%s: %d units, %.0f DMMAs, span %.1f us, DMMA-issue ideal %.1f us (%.2f of span)"
              % (name, len(b), d.sum(), span1 - span0, ideal, ideal / (span1 - span0)), file=out)
        print("  pipe share of one unit while it runs: mean %.2f, DMMA-weighted %.2f"
              % (share.mean(), (share * d).sum() / d.sum()), file=out)
        grid = np.linspace(span0, span1, 11)
        for lo, hi in zip(grid[:-1], grid[1:]):
            ov = np.clip(np.minimum(e, hi) - np.maximum(b, lo), 0, None)
            util = (d * ov / dur).sum() * DMMA_CYCLES / clock_mhz / (hi - lo) / (SM_COUNT * SMSP_PER_SM)
            print("  t %6.1f-%6.1f us: resident warps %5.0f of %d, tensor-pipe utilisation %.2f"
                  % (lo, hi, ov.sum() / (hi - lo), slots, util), file=out)
        gaps = []
        for s in range(SM_COUNT):
            on_sm = sm == s
            for w in np.unique(wid[on_sm]):
                sel = np.where(on_sm & (wid == w))[0]
                o = sel[np.argsort(b[sel])]
                gaps.extend(b[o][1:] - e[o][:-1])
        gaps = np.array(gaps) if gaps else np.zeros(1)
        print("  gaps between consecutive units of a warp slot: mean %.2f us, median %.2f, p90 %.2f, max %.2f; "
              "idle share %.3f" % (gaps.mean(), np.median(gaps), np.percentile(gaps, 90), gaps.max(),
                                   gaps.sum() / (slots * (span1 - span0))), file=out)
        for lo, hi in ((0, 64), (64, 512), (512, 2048), (2048, 1 << 30)):
            sel = (d >= lo) & (d < hi)
            if sel.any():
                print("  units with %4d <= DMMAs < %-10d: %5d, mean duration %6.2f us, alone on a pipe %6.2f us"
                      % (lo, hi, sel.sum(), dur[sel].mean(), (d[sel] * DMMA_CYCLES / clock_mhz).mean()), file=out)


def main():
    chi = int(sys.argv[1]) if len(sys.argv) > 1 else 4096
    profile = sys.argv[2] if len(sys.argv) > 2 else "gaussian"
    t, clock_mhz = capture(chi, profile)
    print("heff_apply unit timeline, chi = %d, %s profile, SM clock taken as %.0f MHz" % (chi, profile, clock_mhz))
    report(t, clock_mhz)


if __name__ == "__main__":
    main()
