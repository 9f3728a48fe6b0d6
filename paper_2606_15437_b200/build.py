"""Builds libkripke_b200.so in-tree with nvcc for sm_100a (no GPU needed to build).

    python -m paper_2606_15437_b200.build [--force] [--verbose]

Objects go to paper_2606_15437_b200/_build/, the library to paper_2606_15437_b200/libkripke_b200.so
(git-ignored, but shipped to the GPU box by gpurun).  ptxas resource reports (-Xptxas -v) are kept
next to each object as <name>.ptxas.txt.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "_build")
LIB = os.path.join(HERE, "libkripke_b200.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]

# (object name, source, extra flags)
UNITS = [
    ("api", "api.cpp", []),
    ("lower", "lower.cpp", []),
    ("sliced_dispatch", "sliced_dispatch.cpp", []),
    ("scan_scalar", "scan_scalar.cu", []),
    ("scan_static", "scan_static.cu", []),
    ("calibrate", "calibrate.cu", []),
    ("scan_frames", "scan_frames.cu", []),
    ("bitmaps", "bitmaps.cu", []),
    ("frame_gen", "frame_gen.cu", []),
    ("jit_dag", "jit_dag.cpp", []),
    ("jit_emit", "jit_emit.cpp", []),
    ("jit_opt", "jit_opt.cpp", []),
    ("jit_runtime", "jit_runtime.cpp", []),
] + [(f"scan_sliced_inst{g}", "scan_sliced_inst.cu", [f"-DKRIPKE_INST_GROUP={g}"]) for g in range(4)] \
  + [(f"scan_frames_inst{g}", "scan_frames_inst.cu", [f"-DKRIPKE_FR_GROUP={g}"]) for g in range(4)]


def _headers_mtime() -> float:
    inc = os.path.join(os.path.dirname(HERE), "include", "kripke.h")
    files = [inc] + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh", ".inc"))]
    return max(os.path.getmtime(f) for f in files)


def _compile(unit, force, verbose):
    name, src, extra = unit
    src_path = os.path.join(CSRC, src)
    obj = os.path.join(OUT, name + ".o")
    stamp = max(os.path.getmtime(src_path), _headers_mtime(), os.path.getmtime(__file__))
    if not force and os.path.exists(obj) and os.path.getmtime(obj) >= stamp:
        return obj, False
    cmd = [NVCC] + ARCH + COMMON + extra + ["-c", src_path, "-o", obj]
    res = subprocess.run(cmd, capture_output=True, text=True)
    with open(os.path.join(OUT, name + ".ptxas.txt"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed for {src}:\n{res.stderr}\n{res.stdout}")
    if verbose:
        print(res.stderr)
    return obj, True


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OUT, exist_ok=True)
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        results = list(ex.map(lambda u: _compile(u, force, verbose), UNITS))
    objs = [o for o, _ in results]
    if force or any(changed for _, changed in results) or not os.path.exists(LIB):
        tmp = LIB + f".{os.getpid()}.tmp"
        cmd = [NVCC] + ARCH + ["-shared", "-o", tmp] + objs + ["-lnvrtc"]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("link failed:\n" + res.stderr)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
