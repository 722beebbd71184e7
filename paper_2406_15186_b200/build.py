"""Build libpulscan.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libpulscan.so"
SOURCES = [CSRC / "pulscan_api.cu"]
DEPS = sorted(CSRC.glob("*.cu*")) + [HERE.parent / "include" / "pulscan.h"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "--expt-relaxed-constexpr"]


def build(force: bool = False, verbose: bool = False) -> Path:
    newest = max(p.stat().st_mtime for p in DEPS)
    if not force and LIB.exists() and LIB.stat().st_mtime >= newest:
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = LIB.with_suffix(f".{os.getpid()}.tmp")
    extra = os.environ.get("PULSCAN_NVCC_EXTRA", "").split()
    cmd = [nvcc, *NVCC_FLAGS, *extra] + (["-Xptxas", "-v"] if verbose else []) + ["-o", str(tmp)] + [str(s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libpulscan.so")
    if verbose:
        sys.stderr.write(res.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
