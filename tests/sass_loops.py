"""SASS opcode histogram of the inner (pixel) loops of the interaction kernels.

    python tests/sass_loops.py [kernel-name-substring ...] > profiles/<name>.txt

Disassembles libdbie_b200.so with cuobjdump, finds in every matching kernel the innermost loops
(backward branches) that contain a reciprocal square root (MUFU.RSQ64H in fp64, MUFU.RSQ in fp32:
one per point-pixel distance), and prints for each its instruction mix by pipe.  This is where the
"FP64 instructions per interaction" figures of DESIGN.md section 6 and bench.py come from: FP64
instructions of the loop / (MUFU.RSQ per trip x lambda triples per geometry).  Runs on the CPU.
"""
from __future__ import annotations

import collections
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(os.path.dirname(HERE), "paper_1306_1122_b200", "libdbie_b200.so")
INSTR = re.compile(r"^\s+/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)(.*?);")
FP64 = ("DFMA", "DMUL", "DADD", "DSETP", "DMNMX")


def kernels(lib: str):
    """Yield (mangled name, [(addr, opcode, operands)])."""
    out = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    name, body = None, []
    for line in out.splitlines():
        m = re.match(r"\s+Function : (\S+)", line)
        if m:
            if name:
                yield name, body
            name, body = m.group(1), []
            continue
        m = INSTR.match(line)
        if m and name:
            body.append((int(m.group(1), 16), m.group(2), m.group(3)))
    if name:
        yield name, body


def demangle(n: str) -> str:
    try:
        return subprocess.run(["cu++filt", n], capture_output=True, text=True).stdout.strip() or n
    except OSError:
        return n


def pipe_of(op: str) -> str:
    base = op.split(".")[0]
    if base in FP64:
        return "fp64"
    if base == "MUFU":
        return "sfu"
    if base in ("FFMA", "FMUL", "FADD", "FMNMX", "FSET", "FSETP", "FCHK"):
        return "fp32"
    if base in ("LDS", "LDG", "STG", "STS", "LDC", "LDCU", "LD", "ST", "ATOM", "ATOMG", "RED", "LDSM", "UBLKCP", "SYNCS"):
        return "mem"
    if base in ("BRA", "BSSY", "BSYNC", "EXIT", "CALL", "RET", "BAR", "WARPSYNC", "NOP", "BREAK", "JMP"):
        return "ctrl"
    return "int/other"


def loops(body):
    addr_index = {a: i for i, (a, _, _) in enumerate(body)}
    found = []
    for i, (a, op, rest) in enumerate(body):
        if op.split(".")[0] != "BRA":
            continue
        m = re.search(r"0x([0-9a-f]+)", rest)
        if not m:
            continue
        t = int(m.group(1), 16)
        if t < a and t in addr_index:
            found.append((addr_index[t], i))
    # innermost = contains no other loop
    inner = [l for l in found if not any(o != l and l[0] <= o[0] and o[1] <= l[1] for o in found)]
    return [l for l in inner if any(op.startswith("MUFU.RSQ") for _, op, _ in body[l[0]:l[1] + 1])]


def loop_table(lib: str = LIB, pats=("interact",)):
    """[(demangled kernel name, [loop dict])] for every matching kernel; a loop dict has the instruction counts
    by pipe and by opcode and `rsqrt`, the point-pixel distances per trip."""
    out = []
    for name, body in kernels(lib):
        d = demangle(name)
        if not any(p in d for p in pats):
            continue
        rows = []
        for (i0, i1) in loops(body):
            seg = body[i0:i1 + 1]
            ops = collections.Counter(op for _, op, _ in seg)
            pipes = collections.Counter(pipe_of(op) for _, op, _ in seg)
            base = collections.Counter()
            for k, v in ops.items():
                base[k.split(".")[0]] += v
            rows.append({"start": seg[0][0], "end": seg[-1][0], "n": len(seg), "pipes": pipes, "opcodes": base,
                         "rsqrt": sum(v for k, v in ops.items() if k.startswith("MUFU.RSQ"))})
        if rows:
            out.append((d, rows))
    return out


def main():
    pats = sys.argv[1:] or ["interact"]
    for d, rows in loop_table(LIB, pats):
        print(f"== {d}")
        for r in rows:
            pipes, rsq = r["pipes"], r["rsqrt"]
            print(f"  loop 0x{r['start']:04x}-0x{r['end']:04x}: {r['n']} instructions, {rsq} rsqrt (point-pixel distances) per trip")
            print("    by pipe: " + ", ".join(f"{k} {v}" for k, v in sorted(pipes.items(), key=lambda kv: -kv[1])))
            print(f"    per distance: fp64 {pipes['fp64'] / rsq:.2f}, fp32 {pipes['fp32'] / rsq:.2f}, sfu {pipes['sfu'] / rsq:.2f}, "
                  f"all {r['n'] / rsq:.2f}")
            print("    opcodes: " + ", ".join(f"{k} {v}" for k, v in sorted(r["opcodes"].items(), key=lambda kv: -kv[1])))


if __name__ == "__main__":
    main()
