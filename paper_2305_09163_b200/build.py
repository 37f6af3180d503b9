"""Builds libmfc_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2305_09163_b200.build [--force] [--verbose]

One translation unit per dimension count plus the C-ABI file, compiled in parallel, linked into
paper_2305_09163_b200/libmfc_b200.so (git-ignored; it travels to the GPU box with the tree).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
OBJ = HERE / "build"
LIB = HERE / "libmfc_b200.so"
SOURCES = ["mfc_api.cu", "mfc_static.cu", "mfc_inst_d1.cu", "mfc_inst_d2.cu", "mfc_inst_d3.cu"]
HEADERS = [CSRC / "mfc_math.cuh", CSRC / "mfc_kernels.cuh", CSRC / "mfc_fused.cuh", CSRC / "mfc_fused_tma.cuh", CSRC / "mfc_fused_roles.cuh", CSRC / "mfc_launch.h", CSRC / "mfc_inst.cuh", HERE.parent / "include" / "mfc.h"]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "--fmad=true"]
# extra flags for experiments (e.g. MFC_NVCC_EXTRA="-DMFC_XPRE=2"); the committed numbers are measured without any
NVCC_FLAGS += os.environ.get("MFC_NVCC_EXTRA", "").split()


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libmfc_b200 cannot be built (there is no CPU fallback)")
    return exe


def _stale(target: Path, deps) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(Path(d).stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    OBJ.mkdir(exist_ok=True)
    exe = nvcc()
    jobs = []
    for src in SOURCES:
        s = CSRC / src
        o = OBJ / (s.stem + ".o")
        if force or _stale(o, [s, Path(__file__)] + HEADERS):
            cmd = [exe] + ARCH + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", str(s), "-o", str(o)]
            jobs.append(cmd)
    if jobs:
        def run(cmd):
            r = subprocess.run(cmd, capture_output=True, text=True)
            return cmd, r
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            for cmd, r in ex.map(run, jobs):
                if verbose or r.returncode != 0:
                    sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
                if r.returncode != 0:
                    raise RuntimeError("nvcc failed: " + " ".join(cmd))
    objs = [str(OBJ / (Path(s).stem + ".o")) for s in SOURCES]
    if force or jobs or _stale(LIB, objs):
        tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = [exe] + ARCH + ["-shared", "-o", str(tmp)] + objs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed: " + " ".join(cmd))
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    p = build(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
    print(p)
