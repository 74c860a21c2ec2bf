"""Build libscmd.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libscmd.so"
PROBE_SRC = PKG / "csrc_probe" / "scmd_probe.cu"       # diagnostics, a library of their own (include/scmd_probe.h)
PROBE_LIB = PKG / "libscmd_probe.so"
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "--fmad=true", "-Xptxas", "-v",
]
OBJ = PKG / "csrc" / "obj"


def sources():
    return sorted(CSRC.glob("*.cu")), sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.h")) + [PKG.parent / "include" / "scmd.h"]


def needs_build() -> bool:
    if not LIB.exists() or not PROBE_LIB.exists():
        return True
    cu, deps = sources()
    probe_deps = [PROBE_SRC, PROBE_SRC.parent / "sc_probe.cuh", PKG.parent / "include" / "scmd_probe.h"]
    newest = max(p.stat().st_mtime for p in cu + deps + [Path(__file__)])
    return LIB.stat().st_mtime < newest or PROBE_LIB.stat().st_mtime < max(newest, *(p.stat().st_mtime for p in probe_deps))


def build_probe(log_text: list) -> int:
    """libscmd_probe.so: one translation unit, linked on its own (it shares only csrc/sc_device.cuh with libscmd)."""
    cmd = ["nvcc", *NVCC_FLAGS, "-shared", str(PROBE_SRC), "-o", str(PROBE_LIB), "-lcudart"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log_text.append(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    return res.returncode


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    cu, deps = sources()
    OBJ.mkdir(exist_ok=True)
    newest_dep = max(p.stat().st_mtime for p in deps + [Path(__file__)])
    log = PKG / "csrc" / "build.log"

    def compile_one(src: Path):
        obj = OBJ / (src.stem + ".o")
        if not force and obj.exists() and obj.stat().st_mtime >= max(newest_dep, src.stat().st_mtime):
            return obj, 0, ""
        cmd = ["nvcc", *NVCC_FLAGS, "-c", str(src), "-o", str(obj)]
        res = subprocess.run(cmd, capture_output=True, text=True)
        return obj, res.returncode, " ".join(cmd) + "\n" + res.stdout + res.stderr

    # one translation unit per instantiation family (csrc/inst_*.cu), compiled in parallel
    with ThreadPoolExecutor(max_workers=min(len(cu), os.cpu_count() or 4)) as pool:
        results = list(pool.map(compile_one, cu))
    text = [t for _, _, t in results]
    rc = max(r for _, r, _ in results)
    if rc == 0:
        cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", *[str(o) for o, _, _ in results],
               "-o", str(LIB), "-lcudart"]
        res = subprocess.run(cmd, capture_output=True, text=True)
        text.append(" ".join(cmd) + "\n" + res.stdout + res.stderr)
        rc = res.returncode
    if rc == 0:
        rc = build_probe(text)
    log.write_text("\n".join(text))
    if verbose or rc != 0:
        sys.stderr.write("\n".join(text))
    if rc != 0:
        raise RuntimeError(f"nvcc failed ({rc}); see {log}")
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
    print(LIB)
