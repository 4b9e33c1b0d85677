"""Operand census of the FP64 loops in a SASS listing (cuobjdump -sass), for profiles/r02_mode_loop.md.

    cuobjdump -sass <binary or library> | python sass_census.py - <substring of the kernel name>

For every loop (backward branch) with at least 60 DFMAs it prints the number of FP64 instructions by how many of their
register source operands are "fresh" -- not served by the operand-reuse cache, i.e. not the same register in the same operand
slot as in the preceding FP64 instruction with .reuse set there -- and the cost by the measured rule of DESIGN.md section 6:
an FP64 instruction occupies the pipe for max(2, fresh operands) cycles."""
import collections
import re
import sys


def load(f):
    funcs, cur = collections.OrderedDict(), None
    for line in f:
        m = re.search(r"Function : (\S+)", line)
        if m:
            cur = m.group(1)
            funcs[cur] = []
            continue
        m = re.search(r"/\*([0-9a-f]{4,})\*/\s+(.*?)\s*;", line)
        if m and cur is not None and not line.strip().startswith("/* 0x"):
            funcs[cur].append((int(m.group(1), 16), m.group(2)))
    return funcs


def opname(t):
    p = t.split()
    return p[1] if p[0].startswith("@") else p[0]


def loops(ins):
    for a, t in ins:
        m = re.search(r"BRA\S*\s+(?:\S+,\s*)?(0x[0-9a-f]+)", t)
        if m and int(m.group(1), 16) < a:
            tgt = int(m.group(1), 16)
            yield tgt, a, [x for x in ins if tgt <= x[0] <= a]


def census(body):
    prev, total, hist = {}, 0, collections.Counter()
    for _, t in body:
        if not opname(t).startswith(("DFMA", "DMUL", "DADD")):
            continue
        args = t.split(None, 2)[2] if t.startswith("@") else t.split(None, 1)[1]
        fresh, cur = 0, {}
        for slot, s in enumerate(x.strip() for x in args.split(",")[1:]):
            m = re.match(r"[-|]*(R\d+)(\.reuse)?", s)
            if not m:
                continue
            if prev.get(slot) != m.group(1):
                fresh += 1
            if m.group(2):
                cur[slot] = m.group(1)
        prev = cur
        total += max(2, fresh)
        hist[fresh] += 1
    return total, hist


if __name__ == "__main__":
    funcs = load(sys.stdin if sys.argv[1] == "-" else open(sys.argv[1]))
    for name, ins in funcs.items():
        if sys.argv[2] not in name:
            continue
        print(name[:110])
        for tgt, a, body in loops(ins):
            nd = sum(opname(t).startswith("DFMA") for _, t in body)
            nl = sum(opname(t).startswith(("LDS", "LDG", "LD.")) for _, t in body)
            if nd >= 60:
                total, hist = census(body)
                n = sum(hist.values())
                print("  loop %x-%x: %d instructions, %d DFMA, %d loads; FP64 by fresh operands %s; %d cycles = %.2f per FP64 instruction"
                      % (tgt, a, len(body), nd, nl, dict(sorted(hist.items())), total, total / n))
