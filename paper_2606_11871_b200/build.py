"""Builds libwarpguard.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo).

    python -m paper_2606_11871_b200.build [--force]
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIB = PKG / "libwarpguard.so"
SOURCES = ["wg_api.cu", "wg_kernels_v1.cu", "wg_kernels_v2.cu", "wg_shadow.cu", "wg_probe.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC,-O2,-Wall",
    "-Xptxas", "-v",
    "--use_fast_math",  # no floating point on the path; harmless, keeps integer division helpers lean
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not Path(exe).exists():
        raise RuntimeError("nvcc not found: libwarpguard.so cannot be built (there is no CPU fallback)")
    return exe


def _newest_source() -> float:
    files = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.h")) + list((ROOT / "include").glob("*"))
    return max(f.stat().st_mtime for f in files)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and LIB.exists() and LIB.stat().st_mtime >= _newest_source():
        return LIB
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc(), *NVCC_FLAGS, "-shared", "-I", str(ROOT / "include"), "-o", str(tmp)]
    cmd += [str(CSRC / s) for s in SOURCES]
    cmd += ["-lcudart_static", "-lpthread", "-ldl", "-lrt"]
    r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed building libwarpguard.so")
    if verbose:
        sys.stderr.write(r.stderr)
    (PKG / "build_ptxas.log").write_text(r.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    p = build(force="--force" in sys.argv, verbose=True)
    print(p)
