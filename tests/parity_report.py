#!/usr/bin/env python
"""Measured GPU-vs-oracle errors of the hot path on the five BASELINE.json configs (run on the GPU box):

    python tests/parity_report.py [--configs 1,2,3,4,5] [--sample 2048] > gpurun_out/parity_report.json

For each config: E rel-L2 and per-target max, phi rel-L2, and the per-target phi error measured against
max(|phi_ref|, floor * rms(phi_ref)) for floor = 1e-3, 1e-2, 1e-1 (DESIGN.md section 7 / reading A6), for the
N-body part, the panel part and their sum.  Configs 1-2: all targets; 3-5: a seeded sample plus adversarial extras
(largest / smallest |E|, largest and smallest |phi| in the GPU output).  Test infrastructure: imports oracle/."""
import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def errors(got, ref):
    got = np.asarray(got, dtype=np.float64)
    dE = np.linalg.norm(got[:, :3] - ref[:, :3], axis=1)
    nE = np.linalg.norm(ref[:, :3], axis=1)
    dphi = np.abs(got[:, 3] - ref[:, 3])
    rms = float(np.sqrt((ref[:, 3] ** 2).mean()))
    out = {"E_rel_l2": float(np.sqrt((dE ** 2).sum() / (nE ** 2).sum())), "E_max_rel": float((dE / nE).max()),
           "phi_rel_l2": float(np.sqrt((dphi ** 2).sum() / (ref[:, 3] ** 2).sum())),
           "phi_abs_err_over_rms_max": float(dphi.max() / rms), "phi_abs_err_over_rms_rms": float(np.sqrt((dphi ** 2).mean()) / rms)}
    for fl in (1e-3, 1e-2, 1e-1):
        out["phi_max_rel_floor_%g" % fl] = float((dphi / np.maximum(np.abs(ref[:, 3]), fl * rms)).max())
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="1,2,3,4,5")
    ap.add_argument("--sample", type=int, default=2048)
    ap.add_argument("--pair-order", action="store_true", help="charges in pair-creation order (interleaved signs)")
    args = ap.parse_args()
    import torch
    from oracle import ref
    from paper_2110_09214_b200 import api, workloads as W
    ref.build()
    report = {}
    for cfg in [int(c) for c in args.configs.split(",")]:
        wl = W.make_workload(cfg)
        if args.pair_order:
            wl = W.pair_creation_order(wl)
        ctx = api.Context(0)
        ctx.set_softening(wl.eps_pp, wl.eps_panel)
        ctx.set_panels(torch.from_numpy(wl.verts).cuda(), torch.from_numpy(wl.sigma).cuda())
        ctx.set_charges(torch.from_numpy(wl.xyzq).cuda())
        tg = wl.points if wl.points is not None else wl.xyzq
        parts = {}
        flags = {"panels": api.PANELS} if wl.points is not None else {"nbody": api.NBODY, "panels": api.PANELS,
                                                                      "both": api.NBODY | api.PANELS}
        for name, fl in flags.items():
            d = torch.from_numpy(tg).cuda()
            parts[name] = (ctx.eval_at_points(d, flags=fl) if wl.points is not None else ctx.eval_at_charges(flags=fl)
                           ).cpu().numpy()
        ctx.destroy()
        nt = tg.shape[0]
        if nt <= 70000:
            idx = np.arange(nt)
        else:
            g = parts["both" if "both" in parts else "panels"]
            mag = np.linalg.norm(g[:, :3], axis=1)
            rng = np.random.default_rng([41, cfg])
            idx = np.unique(np.concatenate([rng.choice(nt, args.sample, replace=False), np.argsort(mag)[-64:],
                                            np.argsort(mag)[:64], np.argsort(np.abs(g[:, 3]))[-64:],
                                            np.argsort(np.abs(g[:, 3]))[:256]]))
        on, op = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=tg[idx],
                                self_index=idx.astype(np.int64) if wl.points is None else None, eps_pp=wl.eps_pp,
                                eps_panel=wl.eps_panel)
        refs = {"nbody": on, "panels": op, "both": on + op}
        report["config_%d" % cfg] = {"targets_compared": int(idx.size),
                                     **{name: errors(parts[name][idx], refs[name]) for name in parts}}
        print("config %d done" % cfg, file=sys.stderr, flush=True)
    print(json.dumps(report, indent=1))


if __name__ == "__main__":
    main()
