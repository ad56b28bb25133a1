"""Build libsaltband.so (and the FP32-peak probe) in-tree with nvcc for sm_100a.

Usage: python -m paper_2504_08081_b200.build [--force] [-v] [--checked]
nvcc cross-compiles without a GPU.  The .so files are git-ignored but travel with gpurun.
--checked also builds libsaltband_checked.so (-DSB_CHECKED: index bounds of the node-weight kernel's shared
arrays are asserted on the device); SALTBAND_LIB=checked makes the binding load it (profiles/r2_sanitizer.md).
"""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
INCLUDE = os.path.join(ROOT, "include")

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "-I", INCLUDE, "-I", CSRC,
]

TARGETS = {
    "libsaltband.so": ["saltband.cu"],
    "libsbprobe.so": ["sb_probe.cu"],
}


def _stale(out: str, deps) -> bool:
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> None:
    nvcc = os.environ.get("NVCC", "nvcc")
    headers = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    headers.append(os.path.join(INCLUDE, "saltband.h"))
    targets = dict(TARGETS)
    if checked:
        targets["libsaltband_checked.so"] = ["saltband.cu"]
    for lib, srcs in targets.items():
        out = os.path.join(PKG, lib)
        src_paths = [os.path.join(CSRC, s) for s in srcs]
        if not all(os.path.exists(s) for s in src_paths):
            continue
        if not (force or _stale(out, src_paths + headers)):
            continue
        extra = ["-DSB_CHECKED"] if lib.endswith("_checked.so") else []
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", out] + src_paths
        print("[build]", " ".join(cmd), file=sys.stderr)
        subprocess.run(cmd, check=True)


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv)
