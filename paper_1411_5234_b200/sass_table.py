"""Count the FP64-pipe instructions of the force kernels' inner loops in the shipped SASS and apply the pipe model of
DESIGN.md section 6 to them (a DFMA/DMUL/DADD holds the pipe 2 cycles, 3 if it reads three different register pairs none of
which the operand-reuse cache supplies, i.e. the previous FP64 instruction flagged that register `.reuse` in the same slot).

    python -m paper_1411_5234_b200.sass_table [--list] [kernel-substring ...]

Text in, text out: runs `cuobjdump -sass paper_1411_5234_b200/libnb.so`, finds the innermost loops that hold at least 20 FP64
instructions, and prints for each a markdown row (instruction mix, `.reuse` flags per operand slot, three-source DFMAs that are
not covered, modelled pipe cycles) and, with --list, the loop body itself.  No GPU needed.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

LIB = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libnb.so")
DEFAULT = ["force_li_kernelILb0ELi6", "force_wu_kernelILb0ELi6", "force_lim_kernelILb0", "force_li_kernelILb0ELi4", "force_li_kernelILb0ELi8"]
FP64 = re.compile(r"(DFMA|DMUL|DADD)\S*\s+(.*)")


def functions(lib=LIB):
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    for f in re.split(r"\n\s*Function : ", out)[1:]:
        name = f.split("\n", 1)[0].strip()
        ins = []
        for line in f.split("\n"):
            m = re.match(r"\s*/\*([0-9a-f]{4})\*/\s+(.*?);", line)
            if m:
                ins.append((int(m.group(1), 16), m.group(2).strip()))
        yield name, ins


def inner_loops(ins):
    addr = {a: k for k, (a, _) in enumerate(ins)}
    loops = []
    for k, (a, t) in enumerate(ins):
        m = re.search(r"BRA(?:\.U)?(?:\.ANY)?\s+(?:!?U?P\d,\s*)?(0x[0-9a-f]+)", t)
        if m:
            tgt = int(m.group(1), 16)
            if tgt < a and tgt in addr:
                loops.append((addr[tgt], k))
    return [l for l in loops if not any(o != l and o[0] >= l[0] and o[1] <= l[1] for o in loops)]


def analyse(body):
    """Two passes over the loop body (the second starts with the reuse cache as the first left it)."""
    mix = collections.Counter()
    for t in body:
        t = re.sub(r"^@!?U?P\d\s+", "", t)
        mix[t.split()[0].split(".")[0]] += 1
    cache, res = {}, None
    for _ in range(2):
        cyc = n3 = three_src = 0
        reuse_flags = collections.Counter()
        uncovered = []
        for t in body:
            t = re.sub(r"^@!?U?P\d\s+", "", t)
            m = FP64.match(t)
            if not m:
                continue
            ops = [o.strip() for o in m.group(2).split(",")][1:]
            regs, reads, new = set(), set(), {}
            for slot, o in enumerate(ops):
                r = re.match(r"[-|]*\s*(R\d+)(\.reuse)?", o)
                if not r or r.group(1) == "RZ":
                    continue
                regs.add(r.group(1))
                if cache.get(slot) != r.group(1):
                    reads.add(r.group(1))
                if r.group(2):
                    new[slot] = r.group(1)
                    reuse_flags["ABC"[slot]] += 1
            cache = new
            three_src += len(regs) == 3
            c = max(2, len(reads))
            cyc += c
            if c == 3:
                n3 += 1
                uncovered.append(t)
        res = dict(cycles=cyc, n3=n3, three_src=three_src, reuse=dict(reuse_flags), uncovered=uncovered)
    res["mix"] = mix
    return res


def main():
    args = [a for a in sys.argv[1:] if not a.startswith("--")]
    listing = "--list" in sys.argv
    keys = args or DEFAULT
    print("| kernel | loop | instr | DFMA | DMUL | DADD | MUFU | LDS | FP32 (FFMA/FMUL/FADD) | F2F | 3-register DFMAs | `.reuse` flags (slot A/B/C) | not covered (3 cycles) | modelled pipe cycles | 2 x FP64 / cycles |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    bodies = []
    for name, ins in functions():
        if not any(k in name for k in keys):
            continue
        short = re.sub(r"^_ZN\d+_GLOBAL__N__[0-9a-f_]+nb_force_cu_[0-9a-f]+\d\d", "", name)
        for s, e in inner_loops(ins):
            body = [t for _, t in ins[s:e + 1]]
            nfp = sum(1 for t in body if FP64.match(re.sub(r"^@!?U?P\d\s+", "", t)))
            nf32 = sum(1 for t in body if re.match(r"(@!?U?P\d\s+)?(FFMA|FMUL|FADD)", t))
            if nfp < 20 and nf32 < 20:
                continue
            r = analyse(body)
            mx = r["mix"]
            ru = r["reuse"]
            print(f"| `{short}` | {ins[s][0]:#x}-{ins[e][0]:#x} | {len(body)} | {mx['DFMA']} | {mx['DMUL']} | {mx['DADD']} | {mx['MUFU']} | {mx['LDS']} | "
                  f"{mx['FFMA'] + mx['FMUL'] + mx['FADD']} | {mx['F2F']} | {r['three_src']} | {ru.get('A', 0)}/{ru.get('B', 0)}/{ru.get('C', 0)} | {r['n3']} | "
                  f"{r['cycles']} | {2 * nfp / max(r['cycles'], 1):.3f} |")
            bodies.append((short, ins[s][0], body, r))
    if listing:
        for short, a, body, r in bodies:
            print(f"\n### {short}, loop at {a:#x}: body ({len(body)} instructions; `*` = FP64 instruction the model charges 3 cycles)\n\n```")
            unc = collections.Counter(r["uncovered"])
            for t in body:
                tt = re.sub(r"^@!?U?P\d\s+", "", t)
                star = "*" if unc.get(tt, 0) > 0 else " "
                print(f"{star} {t}")
            print("```")


if __name__ == "__main__":
    main()
