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

NVCC_COMPILE = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
NVCC_LINK = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static"]


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
    """Every csrc/*.cu is compiled to its own object (in parallel, only when stale) and linked into libmwf.so."""
    from concurrent.futures import ThreadPoolExecutor
    csrc = os.path.join(_HERE, "csrc")
    out = os.path.join(csrc, "libmwf.so")
    srcs = mwf_sources()
    headers = [os.path.join(csrc, f) for f in os.listdir(csrc) if f.endswith((".cuh", ".h"))]
    headers.append(os.path.join(_ROOT, "include", "mwf.h"))
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        if os.path.exists(out) and not force:
            return out
        raise RuntimeError("nvcc not found; cannot build libmwf.so")
    objdir = os.path.join(csrc, "build")
    os.makedirs(objdir, exist_ok=True)
    objs = [os.path.join(objdir, os.path.basename(f)[:-3] + ".o") for f in srcs]
    todo = [(f, o) for f, o in zip(srcs, objs) if force or _stale(o, [f] + headers)]
    extra = os.environ.get("MWF_NVCC_EXTRA", "").split()
    with ThreadPoolExecutor(max_workers=min(8, max(1, len(todo)))) as ex:
        list(ex.map(lambda fo: _run([nvcc] + NVCC_COMPILE + extra + ["-I", os.path.join(_ROOT, "include"), "-c", "-o", fo[1], fo[0]]), todo))
    if todo or force or _stale(out, objs):
        _run([nvcc] + NVCC_LINK + ["-o", out] + objs)
    return out


def build_all(force: bool = False) -> None:
    build_workload(force)
    build_mwf(force)


if __name__ == "__main__":
    build_all(force=True)
    print("built")
