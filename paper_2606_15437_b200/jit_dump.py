"""Shows what the compiled engine generates for a batch: kernel list, CUDA C source, SASS, innermost loop.

    python -m paper_2606_15437_b200.jit_dump [--formulas N] [--n 5] [--class K] [--group 2]
                                             [--kernel I|largest] [--list | --source | --sass | --inner-loop]

The batch is the seeded census corpus (workloads.corpus_c2, the bench's C3 workload) cut to --formulas.  Pure
host: the source comes from kripke_debug_jit_source (the text NVRTC would be given), is compiled here with nvcc
for sm_100a and disassembled with cuobjdump; no GPU is needed.  --inner-loop prints the innermost loop of the
valuation nest (the backward branch with the shortest body) with an opcode histogram: the place where the
LOP3 / POPC / IMAD mix of the scan is decided.
"""
from __future__ import annotations

import argparse
import collections
import os
import re
import subprocess
import sys
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

from . import binding as kb  # noqa: E402

CLASSES = {"K": 0, "T": 1, "S4": 2, "S5": 3}
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CUOBJDUMP = os.path.join(os.path.dirname(NVCC), "cuobjdump")


def sass_of(source: str):
    """(SASS text of the kernel, ptxas resource line) for one generated source."""
    with tempfile.TemporaryDirectory() as tmp:
        cu, cubin = os.path.join(tmp, "kripke_jit.cu"), os.path.join(tmp, "kripke_jit.cubin")
        with open(cu, "w") as fh:
            fh.write(source)
        res = subprocess.run([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-lineinfo", "-Xptxas", "-v",
                              "-cubin", "-o", cubin, cu], capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError(res.stderr)
        used = [line for line in res.stderr.splitlines() if "Used" in line]
        sass = subprocess.run([CUOBJDUMP, "-sass", cubin], capture_output=True, text=True, check=True).stdout
    return sass, (used[0].strip() if used else "")


INSTR = re.compile(r"^\s*/\*([0-9a-f]{4,})\*/\s+(.*?);")


def instructions(sass: str):
    """[(address, text)] of the kernel's instructions."""
    out = []
    for line in sass.splitlines():
        m = INSTR.match(line)
        if m:
            out.append((int(m.group(1), 16), m.group(2).strip()))
    return out


def opcode(text: str) -> str:
    parts = text.split()
    if parts and parts[0].startswith("@"):
        parts = parts[1:]
    return parts[0].split(".")[0] if parts else ""


def loops(ins):
    """Loop-closing branches as (body length in instructions, target address, branch address), shortest first:
    predicated backward BRA (the unconditional ones after the kernel's end are ptxas's out-of-line return
    thunks for divergent warp-collectives and the final self-branch, not loops)."""
    index = {a: i for i, (a, _) in enumerate(ins)}
    found = []
    for i, (a, text) in enumerate(ins):
        m = re.match(r"@!?U?P\d+\s+BRA(?:\.\w+)*\s+0x([0-9a-f]+)", text)
        if m:
            target = int(m.group(1), 16)
            if target < a and target in index:
                found.append((i - index[target] + 1, target, a))
    return sorted(found)


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--formulas", type=int, default=5624)
    ap.add_argument("--n", type=int, default=5)
    ap.add_argument("--class", dest="cls", default="K", choices=sorted(CLASSES))
    ap.add_argument("--group", type=int, default=2, help="programs that mention this many variables")
    ap.add_argument("--kernel", default="largest", help="kernel index within the group, or 'largest' (most logic ops per word)")
    mode = ap.add_mutually_exclusive_group()
    mode.add_argument("--list", action="store_true")
    mode.add_argument("--source", action="store_true")
    mode.add_argument("--sass", action="store_true")
    mode.add_argument("--inner-loop", action="store_true")
    args = ap.parse_args()

    code, offs = W.pack_programs(W.corpus_c2(args.formulas))
    first = kb.debug_jit_source(code, offs, 2, args.n, CLASSES[args.cls], args.group, 0)
    if first is None:
        raise SystemExit("the emitter has no compiled layout for this shape")
    n_kernels = first[1]
    table = [kb.debug_jit_source(code, offs, 2, args.n, CLASSES[args.cls], args.group, i) for i in range(n_kernels)]
    pick = max(range(n_kernels), key=lambda i: table[i][2]) if args.kernel == "largest" else int(args.kernel)
    head = (f"corpus_c2({args.formulas}), n={args.n}, class {args.cls}, programs over {args.group} variable(s): "
            f"{n_kernels} kernel(s) before any spill-driven split")
    if args.list or not (args.source or args.sass or args.inner_loop):
        print(head)
        for i, (src, _, ops, _) in enumerate(table):
            print(f"  kernel {i}: {ops} lop3.b32 per 32-model word (all loop levels), {len(src)} bytes of source"
                  + ("   <- largest" if i == pick else ""))
        return
    source, _, ops, _ = table[pick]
    if args.source:
        print(source)
        return
    sass, used = sass_of(source)
    if args.sass:
        print(sass)
        return
    ins = instructions(sass)
    nest = loops(ins)
    if not nest:
        raise SystemExit("no backward branch found")
    length, target, branch = nest[0]
    body = [(a, t) for a, t in ins if target <= a <= branch]
    hist = collections.Counter(opcode(t) for _, t in body)
    print(head)
    print(f"kernel {pick}: {ops} lop3.b32 per 32-model word over all loop levels; {used}")
    print(f"kernel: {len(ins)} SASS instructions; backward branches (loop nest, innermost first): "
          + ", ".join(f"0x{b:04x}->0x{t:04x} ({n} instr)" for n, t, b in nest))
    print(f"innermost loop 0x{target:04x}..0x{branch:04x}: {length} instructions; opcodes: "
          + ", ".join(f"{op} {c}" for op, c in hist.most_common()))
    print()
    for a, t in body:
        print(f"/*{a:04x}*/  {t} ;")


if __name__ == "__main__":
    main()
