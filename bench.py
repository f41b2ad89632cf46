#!/usr/bin/env python
"""bench.py -- the driver's measurement contract for the OuroborosBEM field-evaluation hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

One "step" is one pass of the whole hot path over the workload:
set_panels + set_charges + evaluation of E and phi at every charge (N-body + panels) + epilogue.
Workload at N=1: BASELINE.json configs[2], the 1M-charge "avalanche snapshot" the metric is quoted on
(1,048,576 charges, 65,536 panels), synthetic and seeded (paper_2110_09214_b200/workloads.py).

N > 1 (torchrun, one rank per GPU): targets are sharded across ranks, sources are replicated; the one
real exchange of a time step -- every rank needs all particle positions -- is an NCCL all-gather of the
ranks' charge slices inside the timed step.  Total work is fixed: "scaling": "strong".

--impl reference times the fp64 CPU oracle (oracle/) on the host cores on a bounded sample of the same
workload (tier framing (4)); rank 0 only.
"""
from __future__ import annotations

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

from paper_2110_09214_b200 import workloads as W  # noqa: E402  (no CUDA needed)

METRIC = "G pairwise interactions/s (1M-charge field eval: E and phi at every charge, N-body + panels)"
UNIT = "Ginteractions/s"
FLOP_PER_INTERACTION = 20.0          # BASELINE.json convention
FP32_LANES_PER_SM = 128              # B200: 4 SMSPs x 32 FP32 lanes, 1 FMA = 2 flop per lane per clock
L2_FLUSH_BYTES = 512 << 20           # > 126 MB L2

_CLOCK_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
                "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")


class ClockSampler:
    """nvidia-smi sampling DURING the timed region (B200_PROFILING.md's clocks line)."""

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="obem_clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + _CLOCK_QUERY, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        sm, smax, power, reasons = [], [], [], set()
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1]))
                    smax.append(float(f[2]))
                    power.append(float(f[3]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"),
                                     f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            # "under load": samples drawing more than half the peak power seen (idle head/tail dropped)
            pmax = max(power)
            load = [s for s, p in zip(sm, power) if p >= 0.5 * pmax] or sm
            out.update(sm_mhz=float(np.median(load)), sm_max_mhz=float(max(smax)), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=pmax)
        return out


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config (1-based); 3 = the metric's workload")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def shard_range(n: int, world: int, rank: int):
    """Contiguous target slice of rank `rank`: sizes differ by at most one."""
    base, rem = divmod(n, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)
