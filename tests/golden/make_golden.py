"""Writes tests/golden/oracle_regression.txt: values of the fp64 ORACLE (nothing else is called) on fixed seeded
inputs, so that a later change of the oracle's arithmetic shows up as a diff of a committed file and has to be
justified in its commit message (the paper itself prints no field value for this path -- only timings, PAPER.md:177-187,
:289-296 -- so there is no fixture from the paper).

    python tests/golden/make_golden.py        # rewrites the fixture; run from the repo root
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import nn, ref  # noqa: E402
from paper_2110_09214_b200 import workloads as W  # noqa: E402  (seeded inputs only: no arithmetic of the method)

IDX = [0, 1, 777, 2047, 2048, 3000, 4095]


def rows():
    wl = W.make_workload(1)
    t = wl.xyzq[IDX]
    on, op = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=t,
                            self_index=np.array(IDX, dtype=np.int64), eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
    ex = ref.eval_panels_analytic(wl.verts, wl.sigma, t)
    nnv, _ = nn.nn_field(wl.xyzq, wl.eps_pp, 2.0, leaf=64, group=512, ref=ref)
    out = []
    for k, i in enumerate(IDX):
        for name, v in (("nbody_eq3.8", on[k]), ("panels_7pt_eq2.13-14", op[k]), ("panels_exact_eq2.13-14", ex[k]),
                        ("nbody_nn_theta2_leaf64_group512", nnv[i])):
            out.append("cfg1 target %4d %-34s %s" % (i, name, " ".join("%.15e" % x for x in v)))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; columns: Ex Ey Ez [V/m] phi [V]\n")
        f.write("\n".join(rows()) + "\n")
    print("wrote", path)
