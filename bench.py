#!/usr/bin/env python
"""bench.py -- heff_apply throughput of the B200-native U(1)xSU(2) two-site TDVP hot path.

Contract: `python bench.py --gpus N --steps K --warmup W` prints ONE JSON line (rank 0).
A step is one heff_apply (stage 1 + stage 2 segmented grouped ZGEMM, SURVEY 8(a) H1+H2) on the
central bond of the L=60 chain of BASELINE.json config 3 (chi = 4096 full dimension, Gaussian
sector profile, seeded random canonical MPS, environments contracted from it by the library's
own env_update_* kernels).  `value` = sum 8mnk over the bit-exact task list / device time.
`--impl reference` times the CPU oracle (oracle/symm.py) on the same workload instead.
Other workloads (--chi, --profile) are for the measurements quoted in DESIGN.md.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

NOMINAL_FP64_TF = 40.0      # B200 dense FP64 (tensor = vector) nominal, HGX B200 data sheet
NOMINAL_BF16_TF = 2250.0    # guide: 2.25 PFLOP/s dense bf16
FALLBACK_BF16_TF = 1590.0   # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
FALLBACK_HBM_GBS = 6650.0


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--chi", type=int, default=4096)
    ap.add_argument("--profile", default="gaussian", choices=["gaussian", "table_s2"])
    ap.add_argument("--s2-scale", default="1/6", help="num/den scale of Table S2 degeneracies")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-flush", action="store_true", help="do not flush L2 between timed applies")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "split"],
                    help="split: run the main line's applies with FH_OPT_PRECISION = 1 (3 x TF32 on tcgen05; NEXT-3). "
                         "Not the headline metric: dtype and config say so; used for the ncu capture of that kernel")
    ap.add_argument("--extra-chi", type=int, nargs="*", default=None,
                    help="replace the default other_configs list by Gaussian-profile applies at these chi (e.g. 32768 49152: "
                         "BASELINE config 5 sizes, minutes of host time to generate the environments)")
    ap.add_argument("--set-option", action="append", default=[], metavar="NAME=VALUE",
                    help="fh_set_option on the main context before anything is planned, e.g. SVD_GRAM_MINN=0, "
                         "SVD_GRAM_BATCH_MAXN=0, SVD_THREADS=6, GEMM_PATH=2 (names: binding.Context.OPT_*); recorded in config")
    ap.add_argument("--no-extra", action="store_true",
                    help="skip the apply-only lines of the other configs (chi = 1024, Table S2 x 1/6, 16384, 24576) and "
                         "the oracle timings on configs 1, 2, 5'")
    ap.add_argument("--no-sweep", action="store_true", help="skip the timed tdvp2_sweep (second half of the metric)")
    ap.add_argument("--sweep", action="store_true", help="(default on) time one full tdvp2_sweep at --sweep-chi")
    ap.add_argument("--sweep-chi", type=int, default=4096)
    ap.add_argument("--config4", action="store_true",
                    help="run BASELINE config 4 instead: L=60 Neel quench, 20 steps of dt=0.05, U=4, chi_max 16384, "
                         "eps_trunc 1e-10; prints one JSON line with per-step observables and time breakdown")
    ap.add_argument("--krylov-adapt-tol", type=float, default=0.0,
                    help="--config4 only: adaptive Krylov dimension (NEXT-2, reading A-15) with this residual "
                         "tolerance and at most 20 vectors instead of the fixed m=10")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(bf16=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained"), hbm=d["hbm_gbs"],
                    source="MEASURED_PEAKS.json")
    return dict(bf16=FALLBACK_BF16_TF, bf16_sustained=None, hbm=FALLBACK_HBM_GBS, source="fallback")


def workload_name(args):
    if args.profile == "gaussian":
        cfg = {1024: "config 2", 4096: "config 3"}.get(args.chi, "config 2/3 recipe")
        return "%s heff_apply: L=60 central bond (29,30), chi=%d, Gaussian sector profile, complex128" % (cfg, args.chi)
    return "heff_apply: L=60 central bond, Table S2 profile x %s, complex128" % args.s2_scale


def s2_scale(args):
    a, b = args.s2_scale.split("/")
    return int(a), int(b)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0]))
                mx.append(float(c[1]))
            except ValueError:
                continue
            for n, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_central_bond(chi, L, c, profile, s2):
    """Oracle-side twin of harness.build_central_bond (same seeded chain, every contraction by oracle/symm.py)."""
    import fh_inputs as fi
    from oracle import symm
    dims = fi.chain_dims(chi, L, profile, s2)
    W = [symm.mpo_reduced(i, 1.0, 4.0) for i in range(L)]
    Le, Re = symm.boundary_left(), symm.boundary_right()
    for i, A, dl, dr in fi.canonical_chain(chi, c, L, fi.SEED, dims=dims, weight=symm.canonical_weight):
        if i < c:
            Le = symm.env_update_left(Le, A, W[i])
        elif i > c + 1:
            Re = symm.env_update_right(Re, A, W[i])
    return dims, Le, Re


def cpu_oracle_setup(args, with_chain=None):
    """Oracle-side workload.  chi <= 4096 (Gaussian profile): the environments are contracted by the oracle from
    the same seeded canonical chain the library uses, so that its H_eff theta can also be compared with the
    library's (the `parity` entry of the line).  Larger workloads: same sector structure and theta, iid random
    environments of the right shapes (timing does not depend on their values) and a bounded sample of output
    blocks."""
    import fh_inputs as fi
    from oracle import symm
    L, c = 60, 29
    if with_chain is None:
        with_chain = args.profile == "gaussian" and args.chi <= 4096
    if with_chain:
        dims, Le, Re = oracle_central_bond(args.chi, L, c, args.profile, s2_scale(args))
        dl, dr = dims[c], dims[c + 2]
    else:
        dims = fi.chain_dims(args.chi, L, args.profile, s2_scale(args))
        dl, dr = dims[c], dims[c + 2]
        Lk, Rk = fi.env_block_keys(dl, dl), fi.env_block_keys(dr, dr)
        Le = fi.random_blocks(11, 1, Lk, {k: (dl[k[0]], dl[k[2]]) for k in Lk})
        Re = fi.random_blocks(11, 2, Rk, {k: (dr[k[0]], dr[k[2]]) for k in Rk})
    th = fi.theta_random(fi.SEED, c, dl, dr)
    W1, W2 = symm.mpo_reduced(c, 1.0, 4.0), symm.mpo_reduced(c + 1, 1.0, 4.0)
    st1, st2 = symm.heff2_tasks(sorted(Le), sorted(Re), sorted(th), W1, W2)
    flops = symm.heff2_flops(st1, st2, dl, dr)
    # bound the sample to ~4 GFLOP of output blocks (whole apply when it is smaller)
    budget, sub2, acc = 4e9, {}, 0
    for k, segs in st2.items():
        sub2[k] = segs
        acc += sum(8 * dl[z[0]] * dr[b] * dr[bp] for z, (bp, wr, b), _ in segs)
        if acc > budget:
            break
    whole = len(sub2) == len(st2)
    need = {seg[0] for segs in sub2.values() for seg in segs}
    sub1 = st1 if whole else {z: st1[z] for z in need}
    f1 = sum(8 * dl[ap] * dl[a] * dr[kk[4]] for z, segs in sub1.items() for (ap, w, a), kk, _ in segs)
    f2 = sum(8 * dl[z[0]] * dr[b] * dr[bp] for segs in sub2.values() for z, (bp, wr, b), _ in segs)
    result = {}

    def step():
        Z = symm.run_stage(sub1, Le, th)
        result["out"] = symm.run_stage(sub2, Z, Re, "n", "t")
        return result["out"]

    sample = ("whole heff_apply" if whole else "%d of %d output blocks" % (len(sub2), len(st2))) + \
        " (%.3g of %.3g GFLOP), task lists prebuilt, %s" % (
            (f1 + f2) * 1e-9, flops * 1e-9,
            "environments contracted by the oracle from the seeded canonical chain" if with_chain
            else "random environments of the same shapes")
    return step, f1 + f2, sample, result, (whole and with_chain), th


def cpu_cores():
    try:
        from threadpoolctl import threadpool_info
        n = max([d.get("num_threads", 1) for d in threadpool_info()] or [1])
    except Exception:
        n = os.cpu_count() or 1
    return int(n)


def time_oracle(args, steps, warmup, with_chain=None):
    step, flops, sample, result, comparable, th = cpu_oracle_setup(args, with_chain)
    for _ in range(warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    dt = (time.perf_counter() - t0) / steps
    cb = dict(value=flops / dt * 1e-9, unit="GFLOP/s", cores=cpu_cores(), kind="oracle", sample=sample)
    return cb, dt, (result.get("out") if comparable else None), th


def parity_vs_oracle(got_blocks, ref_blocks):
    """Relative Frobenius error of the library's H_eff theta against the oracle's under the F-6 weighted norm,
    globally and for the worst single block (north_star: <= 1e-11 per heff_apply)."""
    num = den = worst = 0.0
    for k, v in ref_blocks.items():
        w = k[-1][1] + 1
        d = np.linalg.norm(got_blocks[k] - v)
        num += w * d * d
        den += w * np.linalg.norm(v) ** 2
        worst = max(worst, d / max(np.linalg.norm(v), 1e-300))
    return {"rel_frobenius": float(np.sqrt(num / den)), "worst_block": float(worst), "blocks": len(ref_blocks),
            "tolerance": 1e-11, "against": "oracle/symm.py heff2_apply on the same seeded chain, environments "
            "contracted independently on each side"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cb, dt, _, _ = time_oracle(args, args.steps, args.warmup)
    out = {"impl": "reference", "metric": "heff_apply_gflops", "value": cb["value"], "unit": "GFLOP/s",
           "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "complex128 (f64)",
           "data": "synthetic", "config": {"workload": workload_name(args), "chi": args.chi, "profile": args.profile},
           "cpu_baseline": cb,
           "e2e": {"value": cb["value"], "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def max_over_ranks(values, device, world):
    """Per-phase seconds -> the maximum over all ranks (the contract's max-over-ranks timing).  With
    world == 1 (or no process group) the values come back unchanged.  Replicas only: this all-reduce
    of a few timing scalars is the single collective of the N > 1 path; no data-path collective."""
    import torch
    import torch.distributed as dist
    tt = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if world > 1 and dist.is_available() and dist.is_initialized():
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return [float(v) for v in tt.cpu()]


def aggregate_gflops(flops_per_replica, steps, seconds, world):
    """Whole-job throughput of `world` independent replicas that each did `steps` applies."""
    return world * flops_per_replica * steps / seconds * 1e-9


def profile_traffic():
    """dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/): the line
    'dram_bytes_per_launch: <number>' of the newest r*_heff_apply_ncu.md; None when there is none."""
    import glob
    import re
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_heff_apply_ncu.md")), reverse=True):
        m = re.search(r"dram_bytes_per_launch:\s*([0-9.eE+]+)", open(path).read())
        if m:
            return float(m.group(1)), os.path.relpath(path, ROOT)
    return None, None


def time_apply_random_envs(H, fi, torch, chi, profile, s2, steps, peak_dmma, local):
    """heff_apply on the central bond of the given workload with iid random environments of the right shapes
    (env_set; timing does not depend on their values, and contracting a chi >= 16384 chain on the host would
    take minutes).  Own context, so that `arena_peak_bytes` is this workload's.  profile "u1u1": the U(1) x U(1)
    mode (NEXT-4) on fh_inputs.abelian's profile, the small-block stress case."""
    L, c = 60, 29
    abelian = profile == "u1u1"
    if abelian:
        import fh_inputs.abelian as fab
        dl, dr = fab.profile(c, chi, L), fab.profile(c + 2, chi, L)
        env_keys = fab.env_block_keys
    else:
        dims = fi.chain_dims(chi, L, profile, s2)
        dl, dr = dims[c], dims[c + 2]
        env_keys = fi.env_block_keys
    zest = 40e6 * (sum(dl.values()) / 1274.0) ** 2 * 1.5              # bytes of Z: scales like chi_su2^2 (40 MB at 1274)
    ctx = H.binding.Context(int(min(150e9, max(2 << 30, 4 * zest + (1 << 30)))), device="cuda:%d" % local)
    try:
        if abelian:
            ctx.fh_set_option(ctx.OPT_SYMMETRY, 1)
        mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
        mps = ctx.mps_create(L)
        ctx.mps_set_bond(mps, c, dl)
        ctx.mps_set_bond(mps, c + 2, dr)
        for which, bond, d in ((0, c, dl), (1, c + 2, dr)):
            keys = env_keys(d, d)
            E = fi.random_blocks(11, 1 + which, keys, {k: (d[k[0]], d[k[2]]) for k in keys})
            labels = [[k[0][0], k[0][1], k[1], k[2][0], k[2][1]] for k in keys]
            ctx.env_set(mps, which, bond, labels, np.concatenate([E[k].ravel() for k in keys]))
            del E
        ctx.heff_plan(mpo, mps, c, 2)
        lab, dm, ne = ctx.heff_layout(2)
        flops = ctx.heff_flops()
        x = torch.randn(ne, dtype=torch.complex128, device="cuda:%d" % local) * (1.0 / np.sqrt(2.0 * ne))
        y = torch.empty_like(x)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=x.device)
        for _ in range(3):
            ctx.heff_apply(x, y)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        torch.cuda.synchronize()
        clocks = ClockSampler(local)
        for a, b in ev:
            flush.zero_()
            a.record()
            ctx.heff_apply(x, y)
            b.record()
        torch.cuda.synchronize()
        clk = clocks.stop()
        t = sum(a.elapsed_time(b) for a, b in ev) * 1e-3 / steps
        used, peak = ctx.fh_arena_stats()
        split = None
        if max(max(dl.values()), max(dr.values())) >= 128 and not abelian:
            # NEXT-3: the same apply with FH_OPT_PRECISION = 1 (3 x TF32 on tcgen05, zgemm_tc.cu), L2 flushed as above;
            # the error is taken against the FP64 apply of this run (the oracle comparison lives in tests/)
            y64 = y.clone()
            ctx.fh_set_option(ctx.OPT_PRECISION, 1)
            for _ in range(2):
                ctx.heff_apply(x, y)
            torch.cuda.synchronize()
            for a, b in ev:
                flush.zero_()
                a.record()
                ctx.heff_apply(x, y)
                b.record()
            torch.cuda.synchronize()
            ts = sum(a.elapsed_time(b) for a, b in ev) * 1e-3 / steps
            err = float((torch.linalg.norm(y - y64) / torch.linalg.norm(y64)).item())
            ctx.fh_set_option(ctx.OPT_PRECISION, 0)
            split = {"arithmetic": "3 x TF32 on tcgen05, float32 accumulation in tensor memory (FH_OPT_PRECISION = 1)",
                     "ms_per_apply": ts * 1e3, "gflops_complex128_equivalent": flops / ts * 1e-9,
                     "speedup_vs_fp64": t / ts, "rel_frobenius_vs_fp64_apply": err,
                     "tf32_tflops_issued_lower_bound": 3.0 * flops / ts * 1e-12}
        return {"chi": chi, "profile": profile if profile in ("gaussian", "u1u1") else "table_s2 x %d/%d" % s2,
                "split_precision": split,
                "d_max": max(max(dl.values()), max(dr.values())), "theta_blocks": len(lab), "flop_per_apply": flops,
                "ms_per_apply": t * 1e3, "gflops": flops / t * 1e-9, "frac_of_dmma_peak": flops / t * 1e-12 / peak_dmma,
                "steps": steps, "arena_peak_bytes": int(peak), "theta_bytes": 16 * int(ne), "clocks": clk,
                "environments": "iid random blocks (env_set)"}
    finally:
        ctx.close()


def oracle_extra_timings():
    """the oracle on configs 1, 2 and 5' (reported baselines, host cores)."""
    from oracle import dense_tdvp as dtv
    out = {}
    t0 = time.perf_counter()
    d = dtv.DenseTDVP(8, 1.0, 4.0, krylov_dim=10)
    for _ in range(20):
        d.step(0.05)
    out["config1_dense_tdvp_L8_20_steps_seconds"] = time.perf_counter() - t0

    class A:
        pass
    for tag, chi, prof, s2, chain in (("config2_chi1024", 1024, "gaussian", "1/1", True),
                                      ("config5p_table_s2_x_1_6", 0, "table_s2", "1/6", False)):
        a = A()
        a.chi, a.profile, a.s2_scale = chi, prof, s2
        cb, dt, _, _ = time_oracle(a, 2, 1, with_chain=chain)
        out[tag] = {"gflops": cb["value"], "seconds_per_sample": dt, "sample": cb["sample"]}
    out["cores"] = cpu_cores()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_04771_b200 import harness as H     # fails loudly if the CUDA library is missing
    import fh_inputs as fi

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    pk = peaks()
    L, c = 60, 29
    chi = args.chi
    # replicas only (north_star: one GPU, no sharding, no collectives): every rank runs the same bond
    sweep_need = 0.0 if args.no_sweep else 300.0 * args.sweep_chi * args.sweep_chi
    arena = int(min(160e9, max(16 << 30, 64.0 * chi * chi, sweep_need)))
    ctx = H.binding.Context(arena, device="cuda:%d" % local)
    for kv in args.set_option:
        name, val = kv.split("=")
        ctx.fh_set_option(getattr(ctx, "OPT_" + name.upper()), int(val))
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    t_build = time.perf_counter()
    mps, dims = H.build_central_bond(ctx, mpo, chi, L, profile=args.profile, table_s2_scale=s2_scale(args))
    ctx.heff_plan(mpo, mps, c, 2)
    torch.cuda.synchronize()
    t_build = time.perf_counter() - t_build
    lab, dm, ne = ctx.heff_layout(2)
    th = fi.theta_random(fi.SEED, c, dims[c], dims[c + 2])
    x_host = torch.from_numpy(H.flatten(th, lab, dm, H.theta_key)).pin_memory()
    y_host = torch.empty_like(x_host).pin_memory()
    x = torch.empty_like(x_host, device="cuda:%d" % local)
    ctx.heff_import(x_host.cuda(), x)       # interchange format -> the library's planned layout, once
    y = torch.empty_like(x)
    flops = ctx.heff_flops()
    t1, _, nz = ctx.heff_get_tasks(1)
    t2, _, no = ctx.heff_get_tasks(2)
    flush = None if args.no_flush else torch.empty(256 << 20, dtype=torch.uint8, device=x.device)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    if args.precision == "split":
        ctx.fh_set_option(ctx.OPT_PRECISION, 1)
    for _ in range(max(args.warmup, 3)):
        ctx.heff_apply(x, y)
    peak_dmma = ctx.fh_dmma_peak_tflops(5)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = ctx.fh_launch_count()
    sync_all()
    clocks = ClockSampler(local)
    wall0 = time.perf_counter()
    for a, b in ev:
        if flush is not None:
            flush.zero_()
        a.record()
        ctx.heff_apply(x, y)
        b.record()
    sync_all()
    wall = time.perf_counter() - wall0
    launches = ctx.fh_launch_count() - l0
    ms = [a.elapsed_time(b) for a, b in ev]
    t_dev = sum(ms) * 1e-3
    # L2-warm variant: K applies back to back inside one event pair (what a Lanczos loop sees)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(args.steps):
        ctx.heff_apply(x, y)
    b.record()
    torch.cuda.synchronize()
    t_warm = a.elapsed_time(b) * 1e-3
    clk = clocks.stop()
    # end to end through the host-buffer entry point (pinned host memory, H2D + D2H inside)
    for _ in range(2):
        ctx.heff_apply_host(x_host, y_host)
    sync_all()
    w0 = time.perf_counter()
    for _ in range(args.steps):
        ctx.heff_apply_host(x_host, y_host)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - w0
    t_dev, t_e2e, t_warm = max_over_ranks([t_dev, t_e2e, t_warm], x.device, world)
    if rank != 0:
        return
    y_blocks = torch.empty_like(y)
    ctx.heff_export(y, y_blocks)                     # planned layout -> canonical blocks, for the parity entry
    got_blocks = H.unflatten(y_blocks.cpu().numpy(), lab, dm, H.theta_key)
    gf = aggregate_gflops(flops, args.steps, t_dev, world)
    per_gpu_tf = flops * args.steps / t_dev * 1e-12
    traffic, traffic_src = profile_traffic()
    peak_rule = pk["bf16"] * NOMINAL_FP64_TF / NOMINAL_BF16_TF
    zbytes = 16 * sum(int(a_) * int(b_) for a_, b_ in dm)
    out = {
        "metric": "heff_apply_gflops", "value": gf, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": t_dev / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "complex128 (f64)" if args.precision == "fp64" else "complex128 storage, 3 x TF32 products, f32 accumulation (NOT the headline arithmetic)",
        "data": "synthetic",
        "config": {"workload": workload_name(args), "chi": chi, "profile": args.profile,
                   "chi_su2": [sum(dims[k].values()) for k in (c, c + 1, c + 2)],
                   "d_max": max(max(dims[k].values()) for k in (c, c + 2)), "theta_blocks": len(lab),
                   "z_blocks": nz, "tasks": [len(t1), len(t2)], "flop_per_apply": flops, "theta_bytes": zbytes,
                   "l2": "not flushed" if flush is None else "flushed between timed applies (256 MiB write, outside the event pairs)",
                   "parallelism": "replicas only (one GPU per problem, no collectives)", "setup_seconds": t_build,
                   "options": list(args.set_option)},
        "value_l2_warm": world * flops * args.steps / t_warm * 1e-9,
        "roofline": {"kernel": ("grouped_zgemm_tc_kernel (split precision; the FP64 peak below is NOT its roofline)" if args.precision == "split" else
                                "grouped_zgemm_kernel (stage 1 + stage 2 launches of one apply)" if launches == 2 * args.steps else
                                "grouped_zgemm_ws_kernel (both stages of one apply in one launch)"), "bound": "tensor",
                     "achieved": per_gpu_tf, "peak": peak_dmma, "unit": "TFLOP/s", "frac": per_gpu_tf / peak_dmma,
                     "peak_source": "FP64 DMMA.8x8x4 issue peak measured in this run (fh_dmma_peak_tflops)",
                     "peak_rule": peak_rule, "frac_rule": per_gpu_tf / peak_rule,
                     "peak_rule_source": "%s bf16 %.1f TF x nominal fp64/bf16 %g/%g" % (
                         pk["source"], pk["bf16"], NOMINAL_FP64_TF, NOMINAL_BF16_TF),
                     "frac_l2_warm": flops * args.steps / t_warm * 1e-12 / peak_dmma,
                     "traffic": traffic if (chi == 4096 and args.profile == "gaussian") else None,
                     "traffic_source": ("%s: dram__bytes_read.sum + dram__bytes_write.sum, mean over the two launches of "
                                        "one apply" % traffic_src) if traffic_src else None},
        "e2e": {"value": world * flops * args.steps / t_e2e * 1e-9, "unit": "GFLOP/s",
                "h2d_bytes_per_step": zbytes, "d2h_bytes_per_step": zbytes, "api": "heff_apply_host (pinned host buffers)"},
        "gpu_launches": int(launches), "clocks": clk, "wall_seconds_timed_region": wall,
    }
    # H6 / H8: the HBM-bound vector and pack kernels, in isolation, on a Krylov basis the size of
    # chi = 49152's theta (64 Mi elements = 1 GiB per vector: far beyond L2), against the measured copy peak
    try:
        nvec = 1 << 26 if arena >= (14 << 30) else 1 << 22
        g = ctx.fh_vec_kernels_gbs(nvec, m=10, reps=5)
        out["hbm_kernels"] = {"elements": nvec, "unit": "GB/s", "peak": pk["hbm"], "peak_source": pk["source"],
                              "achieved": g, "frac": {k: v / pk["hbm"] for k, v in g.items()}}
    except H.binding.FhError as e:
        out["hbm_kernels"] = {"error": str(e)}
    # library cross-check of the roofline denominator: cuBLAS FP64 GEMM 8192^3, burst (best of 5)
    # and sustained (back to back for ~3 s)
    try:
        peaks64 = {}
        for nm, cplx_, fl in (("dgemm", 0, 2.0 * 8192 ** 3), ("zgemm", 1, 8.0 * 8192 ** 3)):
            burst = min(ctx.fh_cublas_gemm_seconds(8192, cplx_, 1) for _ in range(5))
            reps = max(2, int(3.0 / burst))
            sust = ctx.fh_cublas_gemm_seconds(8192, cplx_, reps)
            peaks64["cublas_%s_8192_tflops_burst" % nm] = fl / burst * 1e-12
            peaks64["cublas_%s_8192_tflops_sustained" % nm] = fl / sust * 1e-12
        out["roofline"]["peak_cublas"] = peaks64
        out["roofline"]["frac_of_cublas_zgemm_burst"] = per_gpu_tf / peaks64["cublas_zgemm_8192_tflops_burst"]
    except H.binding.FhError as e:
        out["roofline"]["peak_cublas"] = {"error": str(e)}
    if not args.no_sweep and world == 1:
        out["sweep"] = run_sweep(ctx, H, mpo, args)
    ctx.close()
    if not args.no_extra and world == 1:
        extra = []
        todo = ((1024, "gaussian", (1, 1), 20), (4096, "u1u1", (1, 1), 20), (0, "table_s2", (1, 6), 10),
                (16384, "gaussian", (1, 1), 5), (24576, "gaussian", (1, 1), 3))
        if args.extra_chi is not None:
            todo = tuple((cx, "gaussian", (1, 1), 3) for cx in args.extra_chi)
        for chi_x, prof_x, s2_x, st_x in todo:
            try:
                extra.append(time_apply_random_envs(H, fi, torch, chi_x, prof_x, s2_x, st_x, peak_dmma, local))
            except Exception as e:            # report, do not lose the headline line
                extra.append({"chi": chi_x, "profile": prof_x, "error": "%s: %s" % (type(e).__name__, e)})
        out["other_configs"] = extra
    if not args.no_cpu_baseline:
        cb, _, ref_blocks, th_o = time_oracle(args, 3, 1)
        out["cpu_baseline"] = cb
        if ref_blocks is not None:
            assert all(np.array_equal(th[k], th_o[k]) for k in th)      # same seeded theta on both sides
            out["parity"] = parity_vs_oracle(got_blocks, ref_blocks)
        if not args.no_extra:
            out["cpu_baseline_other_configs"] = oracle_extra_timings()
    print(json.dumps(out))


def run_sweep(ctx, H, mpo, args):
    """One full tdvp2_sweep(dt=0.05), m=10, over all 59 bonds of the random right-canonical chain
    at --sweep-chi, with the library's per-phase CUDA-event timers (config 3's second half)."""
    import torch
    chi = args.sweep_chi
    mps, _ = H.build_central_bond(ctx, mpo, chi, 60, centre=0, keep_sites=True,
                                  profile="gaussian")
    # the first sweep of a process also pays the one-time set-up of the factorisation workers (vendor handles,
    # workspaces: 0.2-1.3 s, varies from run to run): it is reported as seconds_first_sweep; `seconds` is the
    # sweep after it, on the same chain (bond dimensions stay at the cap, so the work has the same shape)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ctx.tdvp2_sweep(mpo, mps, 0.05, krylov_dim=10, chi_max_full=chi, eps_trunc=-1.0)
    torch.cuda.synchronize()
    sec_first = time.perf_counter() - t0
    ctx.fh_reset_timers()
    torch.cuda.synchronize()
    l0 = ctx.fh_launch_count()
    t0 = time.perf_counter()
    ctx.tdvp2_sweep(mpo, mps, 0.05, krylov_dim=10, chi_max_full=chi, eps_trunc=-1.0)
    torch.cuda.synchronize()
    sec = time.perf_counter() - t0
    tm = ctx.fh_get_timers()
    tr = ctx.fh_get_traffic()
    st = ctx.tdvp2_last_stats()
    launches2 = ctx.fh_launch_count() - l0
    in_sweep = {"vec_gbs": tr["vec_bytes"] / max(tm["vec"], 1e-12) * 1e-9, "pack_gbs": tr["pack_bytes"] / max(tm["pack"], 1e-12) * 1e-9,
                "vec_bytes": tr["vec_bytes"], "pack_bytes": tr["pack_bytes"],
                "note": "algorithmic bytes of the Lanczos vector kernels (H6) and of pack/unpack (H8) inside this sweep / "
                        "their device seconds: vectors of 0.1-10 MB, launch- and latency-bound, unlike the 1 GiB "
                        "vectors of hbm_kernels"}
    # NEXT-1: the one-site sweep on the same (now chi-saturated) MPS -- the paper's 4-10x lever
    ctx.fh_reset_timers()
    torch.cuda.synchronize()
    l1 = ctx.fh_launch_count()
    t0 = time.perf_counter()
    ctx.tdvp1_sweep(mpo, mps, 0.05, krylov_dim=10)
    torch.cuda.synchronize()
    sec1 = time.perf_counter() - t0
    tm1 = ctx.fh_get_timers()
    st1 = ctx.tdvp2_last_stats()
    launches1 = ctx.fh_launch_count() - l1
    # the sweeps after the first reuse its task lists (fh_plan_cache_stats): the steady state of a long run.
    # Two of them without the library's phase events (fh_enable_timers(0): the production setting), then one
    # with the events for the per-phase breakdown.
    steady = []
    ctx.fh_enable_timers(False)
    for _ in range(2):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.tdvp1_sweep(mpo, mps, 0.05, krylov_dim=10)
        torch.cuda.synchronize()
        steady.append(time.perf_counter() - t0)
    ctx.fh_enable_timers(True)
    ctx.fh_reset_timers()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ctx.tdvp1_sweep(mpo, mps, 0.05, krylov_dim=10)
    torch.cuda.synchronize()
    sec1t = time.perf_counter() - t0
    tm1s = ctx.fh_get_timers()
    cache = ctx.fh_plan_cache_stats(mps)
    ctx.mps_destroy(mps)
    return {"chi": chi, "seconds": sec, "seconds_first_sweep": sec_first, "device_seconds_by_phase": tm, "hbm_kernels_in_sweep": in_sweep, "stats": st,
            "launches": launches2,
            "one_site": {"seconds": sec1, "device_seconds_by_phase": tm1, "chi_full": st1["chi_full"],
                         "launches": launches1, "speedup_vs_two_site": sec / sec1,
                         "seconds_task_lists_cached": steady, "seconds_cached_with_phase_events": sec1t,
                         "device_seconds_by_phase_cached": tm1s,
                         "task_list_cache": cache}}


def run_config4(args):
    """BASELINE config 4: the real quench (no synthetic data).  Reports chi actually reached, per-sweep
    seconds by phase, and the observables the paper plots (n_up = 1/2 + <S^z>, double occupancy)."""
    import torch
    from paper_2606_04771_b200 import harness as H
    L, dt, nstep = 60, 0.05, 20
    ctx = H.binding.Context(8 << 30)
    mpo = ctx.fh_mpo_build(L, 1.0, 4.0)
    mps = ctx.mps_init_neel(mpo, L)
    steps = []
    for k in range(1, nstep + 1):
        ctx.fh_reset_timers()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if args.krylov_adapt_tol > 0:
            ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=20, chi_max_full=16384, eps_trunc=1e-10,
                            krylov_adapt_tol=args.krylov_adapt_tol)
        else:
            ctx.tdvp2_sweep(mpo, mps, dt, krylov_dim=10, chi_max_full=16384, eps_trunc=1e-10)
        torch.cuda.synchronize()
        sec = time.perf_counter() - t0
        obs = ctx.measure_local(mps, L)
        g = ctx.measure_global(mpo, mps)
        st = ctx.tdvp2_last_stats()
        steps.append({"t": k * dt, "seconds": sec, "by_phase": ctx.fh_get_timers(), "chi_full": st["chi_full"],
                      "chi_su2": st["chi_su2"], "d_max": st["dmax"], "max_discarded": st["max_discarded"],
                      "norm2": g["norm2"], "energy": g["energy"],
                      "n_up_site29": 0.5 + float(obs["sz"][29]), "docc_site29": float(obs["docc"][29]),
                      "docc_mean": float(obs["docc"].mean()), "n_minus_1_max": float(abs(obs["n"] - 1).max())})
    nexp, nvec = ctx.fh_krylov_stats()
    krylov = ("adaptive m<=20, tol %g" % args.krylov_adapt_tol) if args.krylov_adapt_tol > 0 else "m=10"
    print(json.dumps({"workload": "config 4: L=60 Neel quench, U=4, dt=0.05, 20 steps, chi_max_full 16384, "
                                  "eps_trunc 1e-10, " + krylov,
                      "total_seconds": sum(x["seconds"] for x in steps),
                      "krylov": {"exponentials": nexp, "heff_applies": nvec, "mean_dim": nvec / max(1, nexp)},
                      "steps": steps}))
    ctx.close()


def main():
    args = parse_args()
    if args.config4:
        return run_config4(args)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
