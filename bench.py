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
    ap.add_argument("--sweep", action="store_true", help="also time one full tdvp2_sweep at --sweep-chi")
    ap.add_argument("--sweep-chi", type=int, default=1024)
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
        return "config3 heff_apply: L=60 central bond (29,30), chi=%d, Gaussian sector profile, complex128" % args.chi
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
