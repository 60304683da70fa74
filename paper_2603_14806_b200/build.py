"""Builds libfoldcp_trimul.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2603_14806_b200.build [--force] [-v] [--debug-knobs]

--debug-knobs builds a SEPARATE library, libfoldcp_trimul_dbg.so, with -DFOLDCP_DEBUG_KNOBS: the A/B
environment knobs of DESIGN.md section 10 exist only there.  The product library reads no
environment variable.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG_DIR, "csrc")
INCLUDE = os.path.join(os.path.dirname(PKG_DIR), "include")
LIB_PATH = os.path.join(PKG_DIR, "libfoldcp_trimul.so")

SOURCES = ["api.cu", "simt_kernels.cu", "simt_backward.cu", "k1_project.cu", "k2_contract.cu",
           "k3_finalize.cu", "k_backward.cu", "triattn.cu", "static_ws.cu"]
HEADERS = ["common.h", "ptx.cuh", "ln_rows.cuh", "tile_sched.cuh", "rank1.cuh"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "static",
    "--expt-relaxed-constexpr",
]


def _nvcc() -> str:
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        raise RuntimeError("nvcc not found; cannot build libfoldcp_trimul.so")
    return nvcc


def needs_build() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    deps.append(os.path.join(INCLUDE, "foldcp_trimul.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, debug_knobs: bool = False) -> str:
    if debug_knobs:
        out = LIB_PATH.replace(".so", "_dbg.so")
        cmd = [_nvcc()] + NVCC_FLAGS + ["-DFOLDCP_DEBUG_KNOBS", "-I", INCLUDE, "-o", out]
        cmd += [os.path.join(CSRC, s) for s in SOURCES]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("nvcc failed building libfoldcp_trimul_dbg.so")
        return out
    if not force and not needs_build():
        return LIB_PATH
    cmd = [_nvcc()] + NVCC_FLAGS + ["-I", INCLUDE, "-o", LIB_PATH]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libfoldcp_trimul.so")
    if verbose:
        sys.stderr.write(res.stdout + res.stderr)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv,
                debug_knobs="--debug-knobs" in sys.argv))
