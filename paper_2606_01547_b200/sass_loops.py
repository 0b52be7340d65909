"""Opcode histogram of the loops of one kernel of libjt.so (static SASS; no GPU needed).

    python -m paper_2606_01547_b200.sass_loops <substring of the demangled kernel name> [--min-instr N] [--lib PATH]

Finds every backward branch in the kernel's SASS (cuobjdump -sass), takes [target, branch] as a loop body, and
prints, innermost loops first, the instruction count per opcode class.  bench.py's TIER_COST (algorithmic instructions
per evaluation on the binding pipe) is recounted from this output: loop body count of the pipe's opcodes / (records per
iteration x rays per thread).  The summaries under profiles/ name the exact command.
"""
import argparse
import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
FP64 = ("DFMA", "DMUL", "DADD", "DSETP", "DMNMX")
FP32 = ("FFMA", "FMUL", "FADD", "FFMA2", "FMUL2", "FADD2", "FSETP", "FMNMX", "FMNMX3", "FSEL", "FSET")


def kernels(lib):
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    name, body, res = None, [], {}
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            if name:
                res[name] = body
            name, body = m.group(1), []
            continue
        m = re.match(r"\s*/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m and name:
            body.append((int(m.group(1), 16), m.group(2).strip()))
    if name:
        res[name] = body
    return res


def demangle(names):
    out = subprocess.run(["cu++filt"] + list(names), capture_output=True, text=True).stdout.splitlines()
    return dict(zip(names, out)) if len(out) == len(names) else {n: n for n in names}


def opcode(text):
    t = re.sub(r"^@!?U?P\d+\s+", "", text)
    return t.split()[0].split(".")[0]


_DUMP = {}


def loop_table(kernel, lib=None):
    """[(n_instructions, n_inner_loops, opcode Counter), ...] for every loop of the ONE kernel whose demangled name contains
    `kernel`, innermost first.  The SASS dump of a library is cached per path (cuobjdump takes half a minute on libjt.so).
    tests/test_roofline_numerator.py checks bench.py's TIER_COST against this."""
    lib = lib or os.path.join(HERE, "libjt.so")
    if lib not in _DUMP:
        ks = kernels(lib)
        _DUMP[lib] = (ks, demangle(list(ks)))
    ks, dm = _DUMP[lib]
    hits = [n for n in ks if kernel in dm[n]]
    if len(hits) != 1:
        raise LookupError("kernel substring %r matches %d functions" % (kernel, len(hits)))
    body = ks[hits[0]]
    index = {a: i for i, (a, _) in enumerate(body)}
    loops = []
    for i, (a, t) in enumerate(body):
        m = re.search(r"\bBRA(?:\.U)?\b.*\b0x([0-9a-f]+)", t)
        if m:
            tgt = int(m.group(1), 16)
            if tgt <= a and tgt in index:
                loops.append((index[tgt], i))
    loops.sort(key=lambda l: l[1] - l[0])
    out = []
    for lo, hi in loops:
        inner = [l for l in loops if l != (lo, hi) and lo <= l[0] and l[1] <= hi]
        out.append((hi - lo + 1, len(inner), collections.Counter(opcode(t) for _, t in body[lo:hi + 1])))
    return out


def fp64_ops(hist):
    return sum(hist[o] for o in FP64)


def fp32_lane_ops(hist):
    return sum(hist[o] * (2 if o.endswith("2") else 1) for o in FP32)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("kernel")
    ap.add_argument("--min-instr", type=int, default=24)
    ap.add_argument("--lib", default=os.path.join(HERE, "libjt.so"))
    args = ap.parse_args()
    ks = kernels(args.lib)
    dm = demangle(list(ks))
    hits = [n for n in ks if args.kernel in dm[n]]
    if len(hits) != 1:
        sys.exit("kernel substring matches %d functions:\n%s" % (len(hits), "\n".join(dm[n] for n in hits[:40])))
    body = ks[hits[0]]
    print("kernel:", dm[hits[0]], "(%d instructions)" % len(body))
    index = {a: i for i, (a, _) in enumerate(body)}
    loops = []
    for i, (a, t) in enumerate(body):
        m = re.search(r"\bBRA(?:\.U)?\b.*\b0x([0-9a-f]+)", t)
        if m:
            tgt = int(m.group(1), 16)
            if tgt <= a and tgt in index:
                loops.append((index[tgt], i))
    loops.sort(key=lambda l: l[1] - l[0])
    for lo, hi in loops:
        n = hi - lo + 1
        if n < args.min_instr:
            continue
        inner = [l for l in loops if l != (lo, hi) and lo <= l[0] and l[1] <= hi]
        hist = collections.Counter(opcode(t) for _, t in body[lo:hi + 1])
        fp64 = sum(hist[o] for o in FP64)
        fp32_lane = sum(hist[o] * (2 if o.endswith("2") else 1) for o in FP32)
        fp32_slots = sum(hist[o] for o in FP32)
        print("\nloop 0x%04x .. 0x%04x: %d instructions%s" % (body[lo][0], body[hi][0], n,
              " (contains %d inner loops)" % len(inner) if inner else ""))
        print("  FP64-pipe %d | FP32-pipe %d issue slots = %d lane-ops (packed x2) | MUFU %d | LDS %d | other %d" % (
            fp64, fp32_slots, fp32_lane, hist["MUFU"], hist["LDS"],
            n - fp64 - fp32_slots - hist["MUFU"] - hist["LDS"]))
        print("  " + ", ".join("%s %d" % kv for kv in hist.most_common()))


if __name__ == "__main__":
    main()
