"""Build libscmd.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libscmd.so"
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC", "--fmad=true", "-Xptxas", "-v",
]


def sources():
    return sorted(CSRC.glob("*.cu")), sorted(CSRC.glob("*.cuh")) + [PKG.parent / "include" / "scmd.h"]


def needs_build() -> bool:
    if not LIB.exists():
        return True
    cu, deps = sources()
    newest = max(p.stat().st_mtime for p in cu + deps + [Path(__file__)])
    return LIB.stat().st_mtime < newest


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    cu, _ = sources()
    cmd = ["nvcc", *NVCC_FLAGS, *[str(p) for p in cu], "-o", str(LIB), "-lcudart"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = PKG / "csrc" / "build.log"
    log.write_text(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed ({res.returncode}); see {log}")
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
    print(LIB)
