#!/usr/bin/env python
"""Instruction mix of the innermost loops of libobem.so's evaluation kernels, read from `cuobjdump -sass`.

    python tests/sass_counts.py [path/to/libobem.so] [--min 150]

For every kernel whose name contains `obem_eval_kernel`, `obem_panels_kernel` or `panels_multi_kernel`: registers,
and for each innermost loop of at least --min instructions its length and mnemonic counts (FFMA2 / FADD2 / FMUL2 =
packed FP32-pipe instructions, MUFU = rsqrt, LDS = the broadcast source loads, UBLKCP / SYNCS elsewhere in the kernel
= the TMA bulk copies and mbarrier waits).  This is what profiles/*_sass.md tabulates; no GPU needed."""
import collections
import os
import re
import subprocess
import sys


def kernels(lib):
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    cur, body = None, {}
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            body[cur] = []
        elif cur is not None:
            body[cur].append(line)
    return body


def loops(lines, min_len):
    ins = []
    for ln in lines:
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", ln)
        if m:
            ins.append((int(m.group(1), 16), m.group(2).strip()))
    at = {a: i for i, (a, _) in enumerate(ins)}
    found = []
    for i, (a, t) in enumerate(ins):
        if "BRA" in t:
            m = re.search(r"0x([0-9a-f]+)", t)
            if m and int(m.group(1), 16) <= a and int(m.group(1), 16) in at:
                found.append((at[int(m.group(1), 16)], i))
    inner = [l for l in found if not any(o != l and o[0] >= l[0] and o[1] <= l[1] for o in found)]
    whole = collections.Counter(re.sub(r"^@!?U?P\d+\s+", "", t).split()[0].split(".")[0] for _, t in ins)
    res = []
    for s, e in inner:
        if e - s + 1 < min_len:
            continue
        c = collections.Counter(re.sub(r"^@!?U?P\d+\s+", "", t).split()[0].split(".")[0] for _, t in ins[s:e + 1])
        res.append((ins[s][0], e - s + 1, dict(c.most_common())))
    return res, whole


def main():
    args = [a for a in sys.argv[1:] if not a.startswith("--")]
    min_len = int(sys.argv[sys.argv.index("--min") + 1]) if "--min" in sys.argv else 150
    if "--min" in sys.argv:
        args = [a for a in args if a != sys.argv[sys.argv.index("--min") + 1]]
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    lib = args[0] if args else os.path.join(root, "paper_2110_09214_b200", "libobem.so")
    regs = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True).stdout
    for name, lines in kernels(lib).items():
        if not any(k in name for k in ("obem_eval_kernel", "obem_panels_kernel", "panels_multi_kernel")):
            continue
        demangled = subprocess.run(["cu++filt", name], capture_output=True, text=True).stdout.strip() or name
        m = re.search(re.escape(name) + r".*?REG:(\d+)", regs, flags=re.S)
        ls, whole = loops(lines, min_len)
        print("%s\n  registers %s; whole kernel: UBLKCP %d, SYNCS %d, BAR %d" % (
            demangled, m.group(1) if m else "?", whole.get("UBLKCP", 0), whole.get("SYNCS", 0), whole.get("BAR", 0)))
        for addr, n, c in ls:
            packed = c.get("FFMA2", 0) + c.get("FADD2", 0) + c.get("FMUL2", 0)
            print("  loop @%#x: %d instructions, %d packed FP32, %d MUFU, %d LDS, other %d: %s" % (
                addr, n, packed, c.get("MUFU", 0), c.get("LDS", 0), n - packed - c.get("MUFU", 0) - c.get("LDS", 0), c))


if __name__ == "__main__":
    main()
