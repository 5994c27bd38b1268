"""In-tree builds of the native pieces of the package (no JIT cache: the .so files travel with the
repository snapshot to the GPU box).

  csrc/libmwf.so        the C-ABI CUDA library (include/mwf.h), sm_100a only
  workload/libbhtree.so the host-side tree / group / list builder (harness input generation)
"""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
]


def _stale(target: str, sources: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _run(cmd: list[str]) -> None:
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("build failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))


def build_workload(force: bool = False) -> str:
    src = os.path.join(_HERE, "workload", "bhtree.cpp")
    out = os.path.join(_HERE, "workload", "libbhtree.so")
    if force or _stale(out, [src]):
        _run(["g++", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-o", out, src])
    return out


def mwf_sources() -> list[str]:
    d = os.path.join(_HERE, "csrc")
    return sorted(os.path.join(d, f) for f in os.listdir(d) if f.endswith(".cu"))


def build_mwf(force: bool = False) -> str:
    out = os.path.join(_HERE, "csrc", "libmwf.so")
    srcs = mwf_sources()
    deps = srcs + [os.path.join(_HERE, "csrc", f) for f in os.listdir(os.path.join(_HERE, "csrc")) if f.endswith((".cuh", ".h"))]
    deps.append(os.path.join(_ROOT, "include", "mwf.h"))
    if force or _stale(out, deps):
        nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
        if not os.path.exists(nvcc):
            raise RuntimeError("nvcc not found; cannot build libmwf.so")
        _run([nvcc] + NVCC_FLAGS + ["-I", os.path.join(_ROOT, "include"), "-o", out] + srcs)
    return out


def build_all(force: bool = False) -> None:
    build_workload(force)
    build_mwf(force)


if __name__ == "__main__":
    build_all(force=True)
    print("built")
