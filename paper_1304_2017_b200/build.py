"""In-tree nvcc build of liboat.so for sm_100a (B200).

    python -m paper_1304_2017_b200.build [--force]

The library is built next to its sources (paper_1304_2017_b200/csrc/liboat.so) so
that it travels to the GPU box with the repo snapshot; nothing is installed into
site-packages and no JIT cache is used.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

CSRC = Path(__file__).resolve().parent / "csrc"
LIB = CSRC / "liboat.so"
SOURCES = ["oat_api.cu", "oat_march.cu", "oat_tile.cu", "oat_kernels.cu", "oat_next.cu", "oat_probe.cu", "oat_noalloc.cu"]
HEADERS = ["oat_internal.h", "../../include/oat.h", "../../include/oat_probe.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",
    "-Xcompiler", "-fPIC",
]


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found; liboat.so cannot be built (there is no CPU fallback)")
    return p


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = [CSRC / s for s in SOURCES] + [(CSRC / h).resolve() for h in HEADERS] + [Path(__file__)]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    nvcc = nvcc_path()
    with tempfile.TemporaryDirectory(prefix="oat_build_") as tmp:
        def compile_one(src):
            obj = os.path.join(tmp, src.replace(".cu", ".o"))
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, str(CSRC / src)]
            return obj, subprocess.run(cmd, capture_output=True, text=True)
        with ThreadPoolExecutor(max_workers=len(SOURCES)) as pool:       # one nvcc per translation unit, in parallel
            done = list(pool.map(compile_one, SOURCES))
        for _, res in done:
            if verbose or res.returncode != 0:
                sys.stderr.write(res.stdout + res.stderr)
        if any(res.returncode != 0 for _, res in done):
            raise RuntimeError("nvcc failed building liboat.so")
        res = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", str(LIB)] + [o for o, _ in done],
                             capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("nvcc failed linking liboat.so")
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
    print(LIB)
