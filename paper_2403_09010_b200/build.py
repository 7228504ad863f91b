"""Builds libsymdel.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension)."""
from __future__ import annotations

import shutil
import subprocess
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
SO = HERE / "libsymdel.so"
SOURCES = ["symdel_api.cu", "generate.cu", "radix_sort.cu", "join.cu", "verify.cu", "static_sort.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC",
              "-Xcompiler", "-fvisibility=hidden", "--expt-relaxed-constexpr"]


def needs_build() -> bool:
    if not SO.exists():
        return True
    t = SO.stat().st_mtime
    deps = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.h")) + [HERE.parent / "include" / "symdel.h"]
    return any(p.stat().st_mtime > t for p in deps)


def build_native(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return SO
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    cmd = [nvcc, *NVCC_FLAGS, "-shared", *[str(CSRC / s) for s in SOURCES], "-o", str(SO)]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True)
    return SO


if __name__ == "__main__":
    import sys

    print(build_native(force=True, verbose="-v" in sys.argv))
