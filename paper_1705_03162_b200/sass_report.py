"""Static evidence about the built kernels, read from libswept_b200.so with cuobjdump (no GPU needed):

    python -m paper_1705_03162_b200.sass_report [--md out.md]

For every hot kernel: registers / static shared memory / stack (`cuobjdump -res-usage`, the ptxas -v figures),
the opcode histogram of its SASS by class, the TMA bulk-copy instructions (UBLKCP), and — for the kernels whose
inner loop is a fixed instruction sequence — the instruction mix of that loop (the innermost backward-branch body
with the most FP64 instructions).  For the Euler kernels it also prints the instructions per cell and stage, the
count SURVEY.md §8(d) asks to be taken from SASS.  A measurement tool like sweep.py, not library code.
"""
from __future__ import annotations

import argparse
import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libswept_b200.so")

CLASSES = [
    ("fp64", re.compile(r"^(DADD|DMUL|DFMA|DSETP|DMNMX)$")),
    ("fp64 div/sqrt helpers (MUFU.RCP64H/RSQ64H)", re.compile(r"^MUFU$")),
    ("fp32", re.compile(r"^(FADD|FMUL|FFMA|FSETP|FMNMX|FSEL|FCHK)$")),
    ("shuffle", re.compile(r"^SHFL$")),
    ("shared ld/st", re.compile(r"^(LDS|STS|LDSM|ATOMS)$")),
    ("global ld/st/atomic", re.compile(r"^(LDG|STG|ATOMG|ATOM|RED|LD|ST|CCTL|MEMBAR|ERRBAR)$")),
    ("TMA bulk copy (UBLKCP) / mbarrier (SYNCS)", re.compile(r"^(UBLKCP|UBLKPF|SYNCS|UTMA.*)$")),
    ("barrier / warp sync", re.compile(r"^(BAR|WARPSYNC|BSSY|BSYNC|NANOSLEEP|DEPBAR|FENCE)$")),
    ("control", re.compile(r"^(BRA|EXIT|CALL|RET|BRX|JMP|NOP|BREAK|YIELD)$")),
]

#: (label, substring of the mangled name) of the kernels DESIGN.md talks about
KERNELS = [
    ("FLOW heat f64 n=512 (headline), 16-byte copies", "swept_flow_kernelINS_4HeatIdEELi16ELb0ELb0E"),
    ("FLOW heat f64 n=512, TMA staging", "swept_flow_kernelINS_4HeatIdEELi16ELb1ELb0E"),
    ("FLOW KS f64 n=1024", "swept_flow_kernelINS_2KSIdLi0EEELi32ELb0ELb0E"),
    ("CHAR heat f64 B=16 L=32 WholeDiamond", "swept_char_kernelINS_4HeatIdEELi16ELi32ELi2E"),
    ("CHAR KS f64 B=32 L=32 WholeDiamond", "swept_char_kernelINS_2KSIdLi0EEELi32ELi32ELi2E"),
    ("CLUSTER heat f64 n=64 (P=2), periodic", "swept_cluster_kernelINS_4HeatIdEELi2ELb0E"),
    ("CLUSTER heat f64 n=64 (P=2), walls", "swept_cluster_kernelINS_4HeatIdEELi2ELb1E"),
    ("CLUSTER KS f64 n=128 (P=4)", "swept_cluster_kernelINS_2KSIdLi0EEELi4ELb0E"),
    ("TIER heat f64 P=1 WholeDiamond", "swept_tier_kernelINS_4HeatIdEELi1ELi2E"),
    ("TIER Euler f64 Heun P=2 WholeDiamond", "swept_tier_kernelINS_5EulerIdLi1EEELi2ELi2E"),
    ("TIER KS3 f64 P=1 WholeDiamond", "swept_tier_kernelINS_3KS3IdEELi1ELi2E"),
    ("per-step heat f64 P=4", "per_step_kernelINS_4HeatIdEELi4E"),
    ("per-step KS f64 fused P=4 (shuffle halo)", "per_step_fused_kernelINS_2KSIdLi0EEELi4ELb1E"),
    ("per-step Euler f64 Heun (one interface per lane)", "per_step_lane_kernelINS_5EulerIdLi1EEE"),
    ("per-step resident heat f64 P=16", "per_step_resident_kernelINS_4HeatIdEELi16E"),
]


def opcode(text: str) -> str:
    text = re.sub(r"^@!?U?P\w+\s+", "", text.strip())
    return text.split()[0].split(".")[0].rstrip(";")


def classify(hist):
    out = collections.OrderedDict((name, 0) for name, _ in CLASSES)
    out["integer / move / other"] = 0
    for op, cnt in hist.items():
        for name, rx in CLASSES:
            if rx.match(op):
                out[name] += cnt
                break
        else:
            out["integer / move / other"] += cnt
    return out


def parse(lib: str):
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    res = subprocess.run(["cuobjdump", "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    usage = {}
    for m in re.finditer(r"Function (\S+):\n\s+(REG:.*)", res):
        usage[m.group(1)] = m.group(2).strip()
    funcs = {}
    for blk in sass.split("Function : ")[1:]:
        name = blk.split("\n", 1)[0].strip()
        ins = [(int(m.group(1), 16), m.group(2)) for m in re.finditer(r"/\*([0-9a-f]{4,6})\*/\s+(.*?);", blk)]
        funcs[name] = ins
    return funcs, usage


def hottest_loop(ins):
    """Innermost loop body (backward branch) with the largest share of FP64 instructions."""
    addr = {a: i for i, (a, _) in enumerate(ins)}
    best = None
    for i, (a, t) in enumerate(ins):
        m = re.search(r"\bBRA\b.*?0x([0-9a-f]+)", t)
        if not m:
            continue
        tgt = int(m.group(1), 16)
        if tgt >= a or tgt not in addr:
            continue
        body = ins[addr[tgt]:i + 1]
        h = collections.Counter(opcode(x[1]) for x in body)
        f = sum(h[k] for k in ("DADD", "DMUL", "DFMA"))
        if f and (best is None or f / len(body) > best[0] or (f / len(body) == best[0] and len(body) > best[1])):
            best = (f / len(body), len(body), h, f)
    return best


def main(argv=None) -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--md", default="")
    args = ap.parse_args(argv)
    if not os.path.exists(LIB):
        raise SystemExit("build the library first: python -m paper_1705_03162_b200.build")
    funcs, usage = parse(LIB)
    lines = ["# SASS / resource summary of the hot kernels (sm_100a)", "",
             "Produced by `python -m paper_1705_03162_b200.sass_report --md <this file>` from the built "
             "`libswept_b200.so` (`cuobjdump -sass`, `cuobjdump -res-usage`); static instruction counts, not executed ones.",
             ""]
    for label, key in KERNELS:
        names = [n for n in funcs if key in n]
        if not names:
            lines += [f"## {label}", "", f"(no kernel matching `{key}` in the library)", ""]
            continue
        name = names[0]
        ins = funcs[name]
        hist = collections.Counter(opcode(t) for _, t in ins)
        cls = classify(hist)
        lines += [f"## {label}", "", f"`{name}`", "", f"- resources: `{usage.get(name, '?')}`",
                  f"- {len(ins)} SASS instructions: " + ", ".join(f"{k} {v}" for k, v in cls.items() if v),
                  f"- UBLKCP (cp.async.bulk) instructions: {hist.get('UBLKCP', 0)}"]
        loop = hottest_loop(ins)
        if loop:
            share, n, h, f = loop
            other = ", ".join(f"{k} {v}" for k, v in h.most_common() if k not in ("DADD", "DMUL", "DFMA"))
            lines.append(f"- FP64-densest loop body: {n} instructions, {f} FP64 (DADD {h['DADD']}, DMUL {h['DMUL']}, "
                         f"DFMA {h['DFMA']}) = {share:.0%}; others: {other}; issue-slot ceiling of the FP64 pipe "
                         f"2F/(2F+O) = {2 * f / (2 * f + n - f):.0%}")
        if "per_step_lane_kernel" in name:
            # straight-line kernel: every lane executes every instruction once; 28 of 32 lanes update a cell
            f64 = cls["fp64"] + cls["fp64 div/sqrt helpers (MUFU.RCP64H/RSQ64H)"]
            lines.append(f"- per cell and stage (28 useful lanes of 32): {len(ins) * 32 / 28:.0f} thread-instructions "
                         f"on the fast path, of which {f64 * 32 / 28:.0f} FP64-pipe (incl. {hist.get('MUFU', 0)} MUFU seeds), "
                         f"{hist.get('SHFL', 0) * 32 / 28:.0f} SHFL; the IEEE division / square-root slow paths (CALL "
                         f"targets inside the kernel, {hist.get('CALL', 0)} call sites) are included statically but only "
                         "run for denormal / huge operands")
        lines.append("")
    text = "\n".join(lines)
    print(text)
    if args.md:
        with open(args.md, "w") as f:
            f.write(text + "\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
