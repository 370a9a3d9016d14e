"""Builds libwarpguard.so (the product) and libwg_probe.so (bench.py's integer-pipe micro-benchmark, not part of the
product) in-tree with nvcc for sm_100a (no JIT cache: the .so files travel with the repo).

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
PROBE_LIB = PKG / "libwg_probe.so"
SOURCES = ["wg_api.cu", "wg_check.cu", "wg_shadow.cu"]
PROBE_SOURCES = ["wg_probe.cu"]
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


def _link(lib: Path, sources: list[str], log: str | None, verbose: bool, extra: list[str] | None = None) -> None:
    tmp = lib.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc(), *NVCC_FLAGS, *(extra or []), "-shared", "-I", str(ROOT / "include"), "-o", str(tmp)]
    cmd += [str(CSRC / s) for s in sources]
    cmd += ["-lcudart_static", "-lpthread", "-ldl", "-lrt"]
    r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError(f"nvcc failed building {lib.name}")
    if verbose:
        sys.stderr.write(r.stderr)
    if log:
        (PKG / log).write_text(r.stderr)
    os.replace(tmp, lib)


def build(force: bool = False, verbose: bool = False, extra: list[str] | None = None) -> Path:
    newest = _newest_source()
    if force or not LIB.exists() or LIB.stat().st_mtime < newest:
        _link(LIB, SOURCES, "build_ptxas.log", verbose, extra)
    if force or not PROBE_LIB.exists() or PROBE_LIB.stat().st_mtime < newest:
        _link(PROBE_LIB, PROBE_SOURCES, None, False)
    return LIB


if __name__ == "__main__":
    p = build(force="--force" in sys.argv, verbose=True, extra=[a for a in sys.argv[1:] if a.startswith("-D")])
    print(p)
