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
from paper_2110_09214_b200.sharding import all_gather_charges, shard_range  # noqa: E402

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

    def __init__(self, gpu_index):
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
    ap.add_argument("--no-next", action="store_true", help="skip the supplementary timings of the adjacent steps")
    ap.add_argument("--dry-run-ranks", action="store_true",
                    help="CPU-only check of the multi-rank plumbing (launcher, gloo all-gather of the charge slices, "
                         "one JSON line from rank 0); no CUDA, no timing claim")
    return ap.parse_args()


def launch_ranks(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun around it: start the N ranks ourselves (one process per
    GPU, rendezvous on 127.0.0.1) and return their exit code.  Fails loudly when fewer than N devices are visible."""
    import socket
    if not args.dry_run_ranks:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            print("bench.py: --gpus %d asked for, %d CUDA device(s) visible -- refusing to run fewer ranks than asked"
                  % (args.gpus, have), file=sys.stderr)
            return 2
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_dry_ranks(args) -> int:
    """The N > 1 host logic without a GPU (tests/test_bench_launcher.py): every rank owns a slice of config 1's
    charges, all-gathers the full array over gloo (the one exchange of a time step), checks it, and rank 0 prints a
    line with the rank count it really ran with."""
    import torch
    import torch.distributed as dist
    rank, world, _ = dist_env()
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE is %d" % (args.gpus, world))
    dist.init_process_group("gloo")
    wl = W.make_workload(1)
    n = wl.n_charges
    first, count = shard_range(n, world, rank)
    full = all_gather_charges(torch.from_numpy(wl.xyzq[first:first + count].copy()), n)
    ok = torch.tensor([1 if np.array_equal(full.numpy(), wl.xyzq) else 0])
    dist.all_reduce(ok, op=dist.ReduceOp.MIN)
    dist.barrier()
    if rank == 0:
        print(json.dumps({"dry_run": True, "metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world,
                          "scaling": "strong", "gather_ok": bool(ok.item()),
                          "config": {"workload": "config 1 charges, gloo on CPU: plumbing only"}}), flush=True)
    dist.destroy_process_group()
    return 0 if ok.item() else 1


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ------------------------------------------------------------------------------------------------------
# the CPU oracle, timed as it stands (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------------
def oracle_sample_rate(wl, seconds: float, seed: int = 123):
    """Time oracle/ (fp64, OpenMP over targets, all host cores) on a bounded seeded sample of the workload's
    targets against ALL its sources.  Returns (interactions_per_s, cores, sample_description, seconds_used)."""
    from oracle import ref  # test infrastructure: allowed here (cpu_baseline / --impl reference only)
    ref.build()
    cores = ref.max_threads()
    rng = np.random.default_rng(seed)
    nt = wl.n_targets
    per_target = (wl.n_charges - (1 if wl.points is None else 0)) + 7 * wl.n_panels
    targets_all = wl.points if wl.points is not None else wl.xyzq

    def run(idx):
        tg = targets_all[idx]
        si = idx.astype(np.int64) if wl.points is None else None
        t0 = time.perf_counter()
        ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=tg, self_index=si,
                       eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
        return time.perf_counter() - t0

    probe = np.sort(rng.choice(nt, min(nt, 4 * cores), replace=False))
    tp = max(run(probe), 1e-6)
    rate = len(probe) * per_target / tp
    for _ in range(2):  # the small probe underestimates the rate (thread start-up): re-size once from a real run
        n_s = int(min(nt, max(len(probe), seconds * rate / per_target)))
        idx = np.sort(rng.choice(nt, n_s, replace=False))
        ts = run(idx)
        rate = n_s * per_target / ts
        if ts >= 0.6 * seconds or n_s == nt:
            break
    desc = "%d seeded targets of %d against all %d charges + %d panels (%.3g interactions, %.1f s)" % (
        n_s, nt, wl.n_charges, wl.n_panels, n_s * per_target, ts)
    return rate, cores, desc, ts


def oracle_one_thread_rate(wl, per_core_rate: float, seconds: float = 3.0, seed: int = 321) -> float:
    """The same oracle on ONE thread (SURVEY.md 8d asks for both), on a sample sized for ~3 s."""
    from oracle import ref
    rng = np.random.default_rng(seed)
    nt = wl.n_targets
    per_target = (wl.n_charges - (1 if wl.points is None else 0)) + 7 * wl.n_panels
    n_s = int(min(nt, max(8, seconds * per_core_rate / per_target)))
    idx = np.sort(rng.choice(nt, n_s, replace=False))
    tg = (wl.points if wl.points is not None else wl.xyzq)[idx]
    t0 = time.perf_counter()
    ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=tg,
                   self_index=idx.astype(np.int64) if wl.points is None else None,
                   eps_pp=wl.eps_pp, eps_panel=wl.eps_panel, n_threads=1)
    return n_s * per_target / max(time.perf_counter() - t0, 1e-9)


def workload_config(wl, args, world):
    return {
        "workload": "BASELINE.json configs[%d] '%s': %d charges (e-/ions), %d triangular panels, Plummer eps %.3g m; "
                    "E and phi at every charge" % (wl.cfg - 1, wl.name, wl.n_charges, wl.n_panels, wl.eps_pp),
        "n_charges": wl.n_charges, "n_panels": wl.n_panels, "n_targets": wl.n_targets,
        "interactions_per_step": wl.interactions()["total"],
        "step": "set_panels + set_charges + eval_at_charges(NBODY|PANELS)" +
                (" with NCCL all-gather of the charge slices" if world > 1 else ""),
        "sharding": "targets sharded over %d rank(s), sources replicated" % world,
        "l2": "flushed between timed steps (%d MiB memset, outside the events)" % (L2_FLUSH_BYTES >> 20),
        "seed": "numpy default_rng([0, %d])" % wl.cfg,
    }


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    wl = W.make_workload(args.config)
    total = wl.interactions()["total"]
    per_step = max(2.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
    vals, cores, desc = [], 1, ""
    for i in range(args.warmup + args.steps):
        rate, cores, desc, _ = oracle_sample_rate(wl, per_step, seed=1000 + i)
        if i >= args.warmup:
            vals.append(rate)
    rate = float(np.mean(vals)) if vals else 0.0
    value = rate / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": (total / rate * 1e3) if rate > 0 else None,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(wl, args, 1),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "each step: " + desc + "; ms_per_step is the full workload extrapolated"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    rank, world, local = dist_env()
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but the launcher started %d rank(s)" % (args.gpus, world))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    from paper_2110_09214_b200 import build as _build
    if rank == 0:
        _build.build_lib()
    if world > 1:
        dist.barrier()
    from paper_2110_09214_b200 import api

    wl = W.make_workload(args.config)           # every rank generates the same seeded inputs
    if wl.points is not None:
        return run_map(args, torch, dist, api, wl, rank, world, local, dev)
    n, npan = wl.n_charges, wl.n_panels
    first, count = shard_range(n, world, rank)
    per_target = (n - 1) + 7 * npan
    total_inter = n * per_target
    my_inter = count * per_target

    ctx = api.Context(local)
    ctx.reserve(n, npan)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    d_verts = torch.from_numpy(wl.verts).to(dev)
    d_sigma = torch.from_numpy(wl.sigma).to(dev)
    d_x = torch.from_numpy(wl.xyzq).to(dev)
    d_slice = d_x[first:first + count].clone()
    d_all = torch.empty_like(d_x)
    out = torch.empty((count, 4), dtype=torch.float32, device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def gather_charges():
        return d_x if world == 1 else all_gather_charges(d_slice, n, out=d_all)

    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731

    def step(timers=None):
        flush.zero_()                                   # L2 flush, outside the events
        if timers is not None:
            timers[0].record(stream)
        ctx.set_panels(d_verts, d_sigma)
        ctx.set_charges(gather_charges())
        if timers is not None:
            timers[1].record(stream)
        ctx.eval_at_charges_range(first, count, out=out, flags=api.NBODY | api.PANELS)
        if timers is not None:
            timers[2].record(stream)

    def sync_all():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        step()
    sync_all()

    uuid = getattr(torch.cuda.get_device_properties(local), "uuid", None)
    sampler = ClockSampler("GPU-%s" % uuid if uuid else str(local))
    if rank == 0:
        sampler.start()
    launches0 = ctx.kernel_launches
    timers = [[ev(), ev(), ev()] for _ in range(args.steps)]
    sync_all()
    wall0 = time.perf_counter()
    for k in range(args.steps):
        step(timers[k])
    sync_all()
    wall = time.perf_counter() - wall0
    launches = ctx.kernel_launches - launches0
    clocks = sampler.stop() if rank == 0 else {}

    step_ms = [t[0].elapsed_time(t[2]) for t in timers]
    eval_ms = [t[1].elapsed_time(t[2]) for t in timers]
    tot_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tot_ms, op=dist.ReduceOp.MAX)     # max over ranks, device-timed
    ms_per_step = float(tot_ms.item()) / max(args.steps, 1)
    value = total_inter / (ms_per_step * 1e-3) / 1e9

    # ---- end to end through host buffers ---------------------------------------------------------
    e2e_steps = max(1, min(args.steps, 3))
    h_x = torch.from_numpy(wl.xyzq).pin_memory()
    h_v = torch.from_numpy(wl.verts).pin_memory()
    h_s = torch.from_numpy(wl.sigma).pin_memory()
    h_out = torch.empty((count, 4), dtype=torch.float32).pin_memory()
    h_slice = h_x[first:first + count]
    h2d = d2h = 0

    def e2e_step():
        nonlocal h2d, d2h
        if world == 1:
            # ONE C-ABI call with host pointers: H2D of every input, set_panels, set_charges, eval, D2H
            ctx.field_at_charges_host(h_x.numpy(), h_v.numpy(), h_s.numpy(), out=h_out.numpy(),
                                      flags=api.NBODY | api.PANELS)
            h2d = h_x.numel() * 4 + h_v.numel() * 4 + h_s.numel() * 4
        else:
            d_slice.copy_(h_slice, non_blocking=True)
            d_verts.copy_(h_v, non_blocking=True)
            d_sigma.copy_(h_s, non_blocking=True)
            ctx.set_panels(d_verts, d_sigma)
            ctx.set_charges(gather_charges())
            ctx.eval_at_charges_range(first, count, out=out, flags=api.NBODY | api.PANELS)
            h_out.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
            h2d = h_slice.numel() * 4 + h_v.numel() * 4 + h_s.numel() * 4
        d2h = h_out.numel() * 4

    e2e_step()
    sync_all()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    sync_all()
    e2e_s = torch.tensor([(time.perf_counter() - t0) / e2e_steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    e2e_value = total_inter / float(e2e_s.item()) / 1e9

    # ---- supplementary, N = 1 only: N-body alone (the north_star's 60 % target) and the FP32 pipe probe ----
    extras = {}
    if world == 1:
        def timed(fn, reps=3):
            fn()
            torch.cuda.synchronize()
            best = 1e30
            for _ in range(reps):
                a, b = ev(), ev()
                flush.zero_()
                a.record(stream)
                fn()
                b.record(stream)
                torch.cuda.synchronize()
                best = min(best, a.elapsed_time(b) * 1e-3)
            return best
        t_nb = timed(lambda: ctx.eval_at_charges(out=out, flags=api.NBODY))
        t_pn = timed(lambda: ctx.eval_at_charges(out=out, flags=api.PANELS))
        fl = [0.0]

        def probe(mode):
            def f():
                fl[0] = ctx.fma_peak_probe(mode, 100000)
            t = timed(f)
            return fl[0] / t / 1e12
        extras = {"nbody_only": {"s": t_nb, "Ginteractions_per_s": n * (n - 1) / t_nb / 1e9},
                  "panels_only": {"s": t_pn, "Ginteractions_per_s": 7 * npan * n / t_pn / 1e9},
                  "fp32_probe_tflops": {"FFMA": probe(0), "FFMA2": probe(1)}}
        # the same charges in the order the method produces them (electron-ion pairs: signs
        # interleaved; workloads.pair_creation_order = a seeded permutation): set_charges + N-body launch
        d_xp = torch.from_numpy(W.pair_creation_order(wl).xyzq).to(dev)
        t_set = timed(lambda: ctx.set_charges(d_xp))
        t_nbp = timed(lambda: ctx.eval_at_charges(out=out, flags=api.NBODY))
        t_eo = timed(lambda: ctx.eval_at_charges(out=out, flags=api.NBODY | api.NO_PHI))
        extras["nbody_only_pair_order"] = {"s": t_nbp, "Ginteractions_per_s": n * (n - 1) / t_nbp / 1e9,
                                           "set_charges_s": t_set, "vs_species_order": t_nbp / t_nb - 1.0}
        extras["nbody_only_E_only"] = {"s": t_eo, "Ginteractions_per_s": n * (n - 1) / t_eo / 1e9,
                                       "what": "OBEM_NBODY | OBEM_NO_PHI on the pair-ordered charges (11 packed "
                                               "instructions per interaction pair instead of 12)"}
        if not args.no_next:
            t_trkp = timed(lambda: ctx.eval_at_charges_partners(flags=api.NBODY))
            extras["nbody_with_partners_pair_order"] = {"s": t_trkp, "overhead_vs_nbody_only_pair_order":
                                                        t_trkp / t_nbp - 1.0}
        ctx.set_charges(d_x)
        del d_xp

    # ---- small configs are launch-latency-bound: the same step replayed from a CUDA graph (no launch gaps) ----
    if world == 1 and n <= 131072:
        side = torch.cuda.Stream()
        side.wait_stream(stream)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            ctx.set_panels(d_verts, d_sigma, stream=side)          # sizes every library-owned buffer before capture
            ctx.set_charges(d_x, stream=side)
            ctx.eval_at_charges_range(first, count, out=out, flags=api.NBODY | api.PANELS, stream=side)
            side.synchronize()
            with torch.cuda.graph(graph, stream=side):
                ctx.set_panels(d_verts, d_sigma, stream=side)
                ctx.set_charges(d_x, stream=side)
                ctx.eval_at_charges_range(first, count, out=out, flags=api.NBODY | api.PANELS, stream=side)
        torch.cuda.synchronize()
        reps = 50
        graph.replay()
        torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record(stream)
        for _ in range(reps):
            graph.replay()
        b.record(stream)
        torch.cuda.synchronize()
        g_ms = a.elapsed_time(b) / reps
        extras["step_cuda_graph"] = {"ms_per_step": g_ms, "Ginteractions_per_s": total_inter / (g_ms * 1e-3) / 1e9,
                                     "what": "the same step (set_panels + set_charges + evaluation) captured once in a "
                                             "CUDA graph and replayed %d times back to back, L2 warm: what is left "
                                             "when the launch gaps are gone" % reps}

    # ---- supplementary, N = 1 only: the adjacent steps, each against its own roofline ----
    if world == 1 and not args.no_next:
        extras["next1"] = bench_next1(torch, api, ctx, wl, timed, dev, extras["panels_only"]["s"])
        extras["next2"] = bench_next2(torch, api, ctx, wl, timed, dev, extras["nbody_only"]["s"])
        extras["next3"] = bench_next3(torch, api, ctx, wl, timed, out, extras["panels_only"]["s"])
        extras["next4"] = bench_next4(torch, api, ctx, wl, timed, dev)
        extras["next4"]["nn_nbody"] = bench_nn(torch, api, ctx, wl, timed, out, extras["nbody_only"]["s"])

    # ---- roofline of the dominant kernel (obem_eval_kernel) -------------------------------------------
    sm_count = ctx.sm_count
    sm_max = (clocks.get("sm_max_mhz") or 1965.0) if rank == 0 else 1965.0
    peak = sm_count * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12           # TFLOP/s
    eval_s = float(np.mean(eval_ms)) * 1e-3
    achieved = FLOP_PER_INTERACTION * my_inter / eval_s / 1e12
    alg_bytes = 16 * n + 128 * npan + 16 * count + 16 * count                 # sources once, targets in, results out
    traffic, traffic_src = recorded_traffic(args.config) if world == 1 else (None, "not recorded for N > 1")
    roofline = {
        "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
        "traffic": traffic, "traffic_source": traffic_src,
        "kernel": "obem_eval_kernel: one evaluation = its two launches (charges, then panels) + fix-up / repair "
                  "(< 0.1 %), between CUDA events on the launch stream",
        "peak_source": "derived: %d SMs x %d FP32 lanes x 2 flop x clocks.max.sm %.0f MHz (DESIGN.md); "
                       "MEASURED_PEAKS.json has no FP32 figure" % (sm_count, FP32_LANES_PER_SM, sm_max),
        "flop_per_interaction": FLOP_PER_INTERACTION, "interactions_per_launch": my_inter,
        "avg_launch_ms": eval_s * 1e3,
        "algorithmic_bytes_per_launch": alg_bytes, "achieved_hbm_gbs": alg_bytes / eval_s / 1e9,
    }
    if extras:
        roofline["nbody_only_frac"] = FLOP_PER_INTERACTION * extras["nbody_only"]["Ginteractions_per_s"] / 1e3 / peak
        roofline["nbody_only_pair_order_frac"] = (FLOP_PER_INTERACTION * extras["nbody_only_pair_order"]
                                                  ["Ginteractions_per_s"] / 1e3 / peak)
        # BASELINE.json north_star: "at least 60 % of B200 FP32 peak on the 1M-charge N-body evaluation"
        roofline["north_star_nbody_target"] = {"frac": 0.60, "met": bool(roofline["nbody_only_frac"] >= 0.60)}
        roofline["frac_of_measured_ffma2_peak"] = (achieved / extras["fp32_probe_tflops"]["FFMA2"]
                                                   if extras["fp32_probe_tflops"]["FFMA2"] else None)

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rate, cores, desc, _ = oracle_sample_rate(wl, args.cpu_seconds)
        cpu_baseline = {"value": rate / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                        "value_1_thread": oracle_one_thread_rate(wl, rate / cores) / 1e9}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(wl, args, world),
            "field_evals_per_s": n / (ms_per_step * 1e-3),
            "pct_fp32_peak": 100.0 * FLOP_PER_INTERACTION * value * 1e9 / 1e12 / (peak * world),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "api": "obem_field_at_charges_host (one C-ABI call, pinned host buffers)" if world == 1 else
                           "per rank: pinned H2D of its slice + panels, all-gather, set_*, eval range, D2H"},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "cpu_baseline": cpu_baseline,
            "wall_s_timed_region": wall,
        }
        line.update(extras)
        print(json.dumps(line), flush=True)
    ctx.destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_map(args, torch, dist, api, wl, rank, world, local, dev):
    """Config 5, the field map (Table 1): panel -> point sums only, E and phi at every grid point.
    A step = set_panels + eval_at_points(OBEM_PANELS) over the rank's contiguous slice of the points (weak in
    nothing: total work fixed, points sharded, panels replicated)."""
    m, npan = wl.n_targets, wl.n_panels
    first, count = shard_range(m, world, rank)
    per_target = 7 * npan
    total_inter, my_inter = m * per_target, count * per_target
    ctx = api.Context(local)
    ctx.reserve(0, npan)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    d_verts = torch.from_numpy(wl.verts).to(dev)
    d_sigma = torch.from_numpy(wl.sigma).to(dev)
    d_pts = torch.from_numpy(wl.points[first:first + count]).to(dev)
    out = torch.empty((count, 4), dtype=torch.float32, device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731

    def step(t=None):
        flush.zero_()
        if t is not None:
            t[0].record(stream)
        ctx.set_panels(d_verts, d_sigma)
        if t is not None:
            t[1].record(stream)
        ctx.eval_at_points(d_pts, out=out, flags=api.PANELS)
        if t is not None:
            t[2].record(stream)

    def sync_all():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        step()
    sync_all()
    uuid = getattr(torch.cuda.get_device_properties(local), "uuid", None)
    sampler = ClockSampler("GPU-%s" % uuid if uuid else str(local))
    if rank == 0:
        sampler.start()
    launches0 = ctx.kernel_launches
    timers = [[ev(), ev(), ev()] for _ in range(args.steps)]
    sync_all()
    wall0 = time.perf_counter()
    for k in range(args.steps):
        step(timers[k])
    sync_all()
    wall = time.perf_counter() - wall0
    launches = ctx.kernel_launches - launches0
    clocks = sampler.stop() if rank == 0 else {}
    tot_ms = torch.tensor([sum(t[0].elapsed_time(t[2]) for t in timers)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tot_ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(tot_ms.item()) / max(args.steps, 1)
    value = total_inter / (ms_per_step * 1e-3) / 1e9
    eval_s = float(np.mean([t[1].elapsed_time(t[2]) for t in timers])) * 1e-3

    # end to end: ONE C-ABI call with host pointers (H2D of points and panels, set_panels, eval, D2H of the map)
    h_p = torch.from_numpy(wl.points[first:first + count]).pin_memory()
    h_v = torch.from_numpy(wl.verts).pin_memory()
    h_s = torch.from_numpy(wl.sigma).pin_memory()
    h_out = torch.empty((count, 4), dtype=torch.float32).pin_memory()

    def e2e_step():
        ctx.field_at_points_host(h_p.numpy(), h_v.numpy(), h_s.numpy(), out=h_out.numpy(), flags=api.PANELS)

    e2e_step()
    sync_all()
    t0 = time.perf_counter()
    e2e_step()
    sync_all()
    e2e_s = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)

    sm_max = (clocks.get("sm_max_mhz") or 1965.0) if rank == 0 else 1965.0
    peak = ctx.sm_count * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    achieved = FLOP_PER_INTERACTION * my_inter / eval_s / 1e12
    alg_bytes = 128 * npan + 32 * count
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rate, cores, desc, _ = oracle_sample_rate(wl, args.cpu_seconds)
        cpu_baseline = {"value": rate / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                        "value_1_thread": oracle_one_thread_rate(wl, rate / cores) / 1e9}
    if rank == 0:
        cfg = workload_config(wl, args, world)
        cfg["workload"] = ("BASELINE.json configs[4] '%s': %d grid points, %d triangular panels; E and phi at every "
                           "point, panel-to-point only" % (wl.name, m, npan))
        cfg["step"] = "set_panels + eval_at_points(PANELS)"
        line = {
            "metric": "G point-source interactions/s (field map: 7 quadrature sources x panels x points)",
            "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": cfg,
            "field_evals_per_s": m / (ms_per_step * 1e-3),
            "pct_fp32_peak": 100.0 * FLOP_PER_INTERACTION * value * 1e9 / 1e12 / (peak * world),
            "clocks": clocks,
            "e2e": {"value": total_inter / float(e2e_s.item()) / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": (h_p.numel() + h_v.numel() + h_s.numel()) * 4,
                    "d2h_bytes_per_step": h_out.numel() * 4,
                    "api": "obem_field_at_points_host (one C-ABI call, pinned host buffers)"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "traffic": None, "kernel": "obem_eval_kernel<panels> (+ fix-up / repair) between CUDA events",
                         "flop_per_interaction": FLOP_PER_INTERACTION, "interactions_per_launch": my_inter,
                         "avg_launch_ms": eval_s * 1e3, "algorithmic_bytes_per_launch": alg_bytes,
                         "achieved_hbm_gbs": alg_bytes / eval_s / 1e9},
            "cpu_baseline": cpu_baseline, "wall_s_timed_region": wall,
        }
        if world == 1 and not args.no_next:
            a, b = ev(), ev()
            ctx.eval_at_points(d_pts, out=out, flags=api.PANELS | api.PANELS_EXACT)   # builds the cell lists
            torch.cuda.synchronize()
            flush.zero_()
            a.record(stream)
            ctx.eval_at_points(d_pts, out=out, flags=api.PANELS | api.PANELS_EXACT)
            b.record(stream)
            torch.cuda.synchronize()
            t_ex = a.elapsed_time(b) * 1e-3
            line["next3"] = {"panels_exact": {"s": t_ex, "overhead_vs_7_point_only": t_ex / eval_s - 1.0,
                                              "cell_list_entries": ctx.near_list_size, "cells": ctx.near_cells}}
        print(json.dumps(line), flush=True)
    ctx.destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0


def hbm_peak_gbs():
    """Measured HBM copy bandwidth of this pool's B200 (MEASURED_PEAKS.json, driver-written), else the fallback
    B200_PROFILING.md states (6.65 TB/s, "of fallback")."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "of fallback (B200_PROFILING.md: 6.65 TB/s)"


def bench_next1(torch, api, ctx, wl, timed, dev, t_panels):
    """Influence of the particles on the cells (Eq 3.3/3.4; FP32-pipe bound like the hot path), sigma = M^-1 b
    (HBM bound: 4 n^2 bytes read once) and the chained dynamic update, on the bench workload."""
    n, npan = wl.n_charges, wl.n_panels
    peak_flops = ctx.sm_count * FP32_LANES_PER_SM * 2 * 1965.0e6 / 1e12
    t_inf = timed(lambda: ctx.influence_on_panels())
    inter = 7 * npan * n
    res = {"influence": {"s": t_inf, "Ginteractions_per_s": inter / t_inf / 1e9,
                         "frac_fp32_peak": FLOP_PER_INTERACTION * inter / t_inf / 1e12 / peak_flops,
                         "bound": "alu"}}
    # weighting fields (Eq 3.13): 4 density vectors on the same cells in one pass, against one single-sigma launch
    gen0 = torch.Generator(device=dev)
    gen0.manual_seed(1)
    sig4 = torch.empty((4, npan), dtype=torch.float32, device=dev).normal_(0.0, 1e-5, generator=gen0)
    pts = torch.from_numpy(wl.xyzq).to(dev)
    out4 = torch.empty((4, n, 4), dtype=torch.float32, device=dev)
    t_m4 = timed(lambda: ctx.eval_panels_multi(sig4, pts, out=out4))
    res["panels_multi_4"] = {"s": t_m4, "vectors": 4, "vs_one_single_sigma_launch": t_m4 / t_panels,
                             "packed_fp32_instr_per_panel_and_target_pair": {"multi_4": 103, "single": 87},
                             "Ginteractions_per_s_per_vector_equivalent": 4 * inter / t_m4 / 1e9,
                             "frac_fp32_peak_of_executed_work": FLOP_PER_INTERACTION * inter * (103.0 / 87.0) / t_m4 / 1e12
                             / peak_flops, "bound": "alu"}
    # Eq (3.13) on that pass's output: the induced currents of the 4 electrodes (HBM-bound, launch-latency scale)
    vel = torch.zeros((n, 4), dtype=torch.float32, device=dev)
    vel[:, 2] = 1.0e5
    t_ramo = timed(lambda: ctx.ramo_current(pts, vel, out4), reps=5)
    peak_hbm, src_hbm = hbm_peak_gbs()
    ramo_bytes = n * (16 * 4 + 32)
    res["ramo_current_4"] = {"s": t_ramo, "bound": "hbm (two launches)",
                             "algorithmic_bytes": ramo_bytes, "achieved": ramo_bytes / t_ramo / 1e9, "peak": peak_hbm,
                             "unit": "GB/s", "frac": ramo_bytes / t_ramo / 1e9 / peak_hbm, "peak_source": src_hbm}
    del sig4, out4, pts, vel
    free, _ = torch.cuda.mem_get_info()
    ng = npan
    while ng > 1024 and 4 * ng * ng > 0.6 * free:
        ng //= 2
    gen = torch.Generator(device=dev)
    gen.manual_seed(0)
    minv = torch.empty((ng, ng), dtype=torch.float32, device=dev)
    minv.normal_(0.0, 1e-10, generator=gen)
    b = torch.randn(ng, dtype=torch.float32, device=dev, generator=gen)
    sig = torch.empty(ng, dtype=torch.float32, device=dev)
    t_mv = timed(lambda: ctx.apply_inverse(minv, b, out=sig), reps=5)
    peak, src = hbm_peak_gbs()
    gbs = 4.0 * ng * ng / t_mv / 1e9
    res["apply_inverse"] = {"n": ng, "s": t_mv, "bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s",
                            "frac": gbs / peak, "peak_source": src,
                            "algorithmic_bytes": 4 * ng * ng + 8 * ng}
    if ng == npan:
        kind = (torch.arange(npan, device=dev) % 3 == 0).to(torch.int32)
        bc = torch.zeros(npan, dtype=torch.float32, device=dev)
        deps = torch.full((npan,), 2.5 * 8.8541878128e-12, dtype=torch.float32, device=dev)
        sigma0 = torch.from_numpy(wl.sigma).to(dev)
        t_dyn = timed(lambda: ctx.update_sigma_dynamic(kind, bc, deps, minv))
        ctx.set_sigma(sigma0)
        res["dynamic_update"] = {"s": t_dyn, "what": "influence + rhs + M^-1 b + set_sigma on one stream"}
    del minv
    return res


def bench_next2(torch, api, ctx, wl, timed, dev, t_nbody):
    """Recombination by-product of the N-body pass and one Euler / PEFRL step on the
    bench workload, N-body + panels."""
    n = wl.n_charges
    peak_flops = ctx.sm_count * FP32_LANES_PER_SM * 2 * 1965.0e6 / 1e12
    t_trk = timed(lambda: ctx.eval_at_charges_partners(flags=api.NBODY))
    res = {"nbody_with_partners": {"s": t_trk, "Ginteractions_per_s": n * (n - 1) / t_trk / 1e9,
                                   "frac_fp32_peak": FLOP_PER_INTERACTION * n * (n - 1) / t_trk / 1e12 / peak_flops,
                                   "overhead_vs_nbody_only": t_trk / t_nbody - 1.0}}
    x = torch.from_numpy(wl.xyzq).to(dev)
    v = torch.zeros_like(x)
    v[:, 3] = 9.1093837015e-31
    per_eval = n * ((n - 1) + 7 * wl.n_panels)
    t_e = timed(lambda: ctx.step_euler(x, v, 25e-15), reps=2)
    res["step_euler"] = {"s": t_e, "field_evaluations": 1, "Ginteractions_per_s": per_eval / t_e / 1e9}
    t_p = timed(lambda: ctx.step_pefrl(x, v, 25e-15), reps=1)
    res["step_pefrl"] = {"s": t_p, "field_evaluations": 4, "Ginteractions_per_s": 4 * per_eval / t_p / 1e9}
    ctx.set_charges(torch.from_numpy(wl.xyzq).to(dev))
    return res


def bench_next3(torch, api, ctx, wl, timed, out, t_panels):
    """Near-field-accurate panels: the panel sum with the closed-form integrals for the panels
    within 3 longest-edges of each charge, against the 7-point sum alone.  The first call builds the cell lists
    (once per geometry) and is timed separately."""
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    ctx.eval_at_charges(out=out, flags=api.PANELS | api.PANELS_EXACT)
    ev1.record()
    torch.cuda.synchronize()
    t_first = ev0.elapsed_time(ev1) * 1e-3
    t_ex = timed(lambda: ctx.eval_at_charges(out=out, flags=api.PANELS | api.PANELS_EXACT))
    return {"panels_exact": {"s": t_ex, "overhead_vs_7_point_only": t_ex / t_panels - 1.0,
                             "first_call_with_list_build_s": t_first, "near_factor": 3.0,
                             "cell_list_entries": ctx.near_list_size, "cells": ctx.near_cells}}


def bench_nn(torch, api, ctx, wl, timed, out, t_nbody):
    """NN approximation of the N-body sum (paper's Table 2: 0.09 s for 1e6 particles on 1 GPU of
    2019) on the bench workload: whole call (k-d order, leaves, lists, sums, scatter) and what it computes."""
    n = wl.n_charges
    peak_flops = ctx.sm_count * FP32_LANES_PER_SM * 2 * 1965.0e6 / 1e12
    res = {}
    for theta in (2.0, 1.0):
        ctx.set_nn_theta(theta)
        t = timed(lambda: ctx.eval_at_charges_nn(out=out, flags=api.NBODY))
        units = ctx.nn_last_units()
        inter = units * 2048 * 256
        res["theta_%g" % theta] = {"s": t, "speedup_vs_exact_sum": t_nbody / t, "units": units,
                                   "pair_interactions": inter, "fraction_of_exact_pairs": inter / (n * (n - 1)),
                                   "Ginteractions_per_s_whole_call": inter / t / 1e9,
                                   "frac_fp32_peak_whole_call": FLOP_PER_INTERACTION * inter / t / 1e12 / peak_flops}
    ctx.set_nn_theta(2.0)
    # the paper's largest Table-2 case: 1e7 particles (synthetic Gaussian electron/ion cloud, seeded on the device)
    free, _ = torch.cuda.mem_get_info()
    if free > 16e9:
        n10 = 10_000_000
        gen = torch.Generator(device=out.device)
        gen.manual_seed(10)
        x10 = torch.randn((n10, 4), dtype=torch.float32, device=out.device, generator=gen)
        x10[:, :3] *= torch.tensor([40e-6, 40e-6, 20e-6], device=out.device)
        x10[:, 3] = torch.where(x10[:, 3] > 0, 1.602176634e-19, -1.602176634e-19)
        out10 = torch.empty_like(x10)
        ctx.set_charges(x10)
        t = timed(lambda: ctx.eval_at_charges_nn(out=out10, flags=api.NBODY), reps=2)
        units = ctx.nn_last_units()
        res["n_1e7_theta_2"] = {"s": t, "units": units, "pair_interactions": units * 2048 * 256,
                                "fraction_of_exact_pairs": units * 2048 * 256 / (n10 * (n10 - 1.0)),
                                "exact_sum_would_take_s": n10 * (n10 - 1.0) / (n * (n - 1.0)) * t_nbody}
        del x10, out10
        ctx.set_charges(torch.from_numpy(wl.xyzq).to(out.device))
    return res


def bench_next4(torch, api, ctx, wl, timed, dev):
    """Static field option: trilinear interpolation in a 256^3 x float4 map (config 5's shape,
    268 MB: larger than L2) at the bench workload's charges (clustered, as an avalanche is) and at as many
    uniformly scattered positions (worst case for the gather).  HBM bound; algorithmic bytes = 16 B position in +
    16 B result out per position + the map read once if every node is touched (scattered: min(map, 8 x 16 B x M))."""
    n = wl.n_charges
    shape = (256, 256, 256)
    origin = (-210e-6, -210e-6, -150e-6)
    spacing = (420e-6 / 255, 420e-6 / 255, 300e-6 / 255)
    gen = torch.Generator(device=dev)
    gen.manual_seed(4)
    fmap = torch.empty(shape + (4,), dtype=torch.float32, device=dev)
    fmap.normal_(0.0, 1.0, generator=gen)
    pts_c = torch.from_numpy(wl.xyzq).to(dev)
    pts_u = torch.rand((n, 4), dtype=torch.float32, device=dev, generator=gen)
    pts_u = pts_u * torch.tensor([420e-6, 420e-6, 300e-6, 0.0], device=dev) + torch.tensor(
        [origin[0], origin[1], origin[2], 0.0], device=dev)
    out = torch.empty((n, 4), dtype=torch.float32, device=dev)
    peak, src = hbm_peak_gbs()
    res = {"map": "256x256x256 float4 (268 MB)", "positions": n, "bound": "hbm", "peak": peak, "unit": "GB/s",
           "peak_source": src}
    map_bytes = fmap.numel() * 4
    for name, pts in (("at_charges", pts_c), ("scattered", pts_u)):
        t = timed(lambda: ctx.interp_map(fmap, origin, spacing, pts, out=out), reps=5)
        stream_b = 32 * n
        touched = min(map_bytes, 8 * 16 * n)
        res[name] = {"s": t, "Mpositions_per_s": n / t / 1e6, "streamed_GBps": stream_b / t / 1e9,
                     "frac_streamed_only": stream_b / t / 1e9 / peak,
                     "GBps_incl_map_upper_bound": (stream_b + touched) / t / 1e9}
    del fmap
    return res


def kernel_source_hash() -> str:
    """sha256 over the sources of the evaluation kernels -- csrc/obem.cu and the device helpers of obem_internal.cuh
    (everything before the host-side context structs): ties a recorded ncu figure to the code it was captured on."""
    import hashlib
    h = hashlib.sha256()
    base = os.path.join(ROOT, "paper_2110_09214_b200", "csrc")
    with open(os.path.join(base, "obem.cu"), "rb") as fh:
        h.update(fh.read())
    with open(os.path.join(base, "obem_internal.cuh"), "rb") as fh:
        h.update(fh.read().split(b"/* obem_nn.cu: buffers of the NN approximation")[0])
    return h.hexdigest()[:16]


def recorded_traffic(cfg: int):
    """`roofline.traffic` cannot be measured inside this process (DRAM counters need ncu), so it is a RECORDED figure:
    profiles/r02_traffic.json holds dram__bytes_read.sum + dram__bytes_write.sum per evaluation from the committed
    `ncu --set full` capture, with the hash of the kernel sources it was taken on.  If the sources changed since,
    the figure is stale and null is reported instead of a wrong number."""
    path = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        with open(path) as f:
            rec = json.load(f)
        ent = rec["configs"].get(str(cfg))
        if ent is None:
            return None, "no capture recorded for config %d in profiles/r02_traffic.json" % cfg
        if rec["kernel_source_hash"] != kernel_source_hash():
            return None, "stale: profiles/r02_traffic.json was captured on kernel sources %s, these are %s" % (
                rec["kernel_source_hash"], kernel_source_hash())
        return ent["bytes_per_evaluation"], "recorded, not measured live: %s (%s)" % (ent["capture"], path[len(ROOT) + 1:])
    except Exception as e:  # noqa: BLE001
        return None, "no record: %s" % e


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)      # rank 0 alone times the oracle; the other ranks of a torchrun exit 0
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return launch_ranks(args)
    if args.dry_run_ranks:
        return run_dry_ranks(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
