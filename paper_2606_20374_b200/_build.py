"""In-tree native builds (no JIT cache: the .so files sit beside their sources so that they travel
to the GPU box with the repo snapshot).  nvcc cross-compiles sm_100a without a GPU."""
from __future__ import annotations

import os
import shutil
import subprocess
from typing import List

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
NVCC = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _stale(target: str, sources: List[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _run(cmd: List[str]) -> None:
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        raise RuntimeError("build failed: " + " ".join(cmd) + "\n" + r.stdout)


def build_argus(force: bool = False, extra: List[str] | None = None) -> str:
    """libargus.so: the CUDA kernels + the C ABI of include/argus.h."""
    src_dir = os.path.join(PKG, "csrc")
    srcs = sorted(os.path.join(src_dir, f) for f in os.listdir(src_dir) if f.endswith(".cu"))
    deps = srcs + [os.path.join(src_dir, f) for f in os.listdir(src_dir) if f.endswith((".cuh", ".h"))]
    deps.append(os.path.join(ROOT, "include", "argus.h"))
    out = os.path.join(PKG, "libargus.so")
    if force or _stale(out, deps):
        _run([NVCC, *ARCH, "-O3", "-std=c++17", "-lineinfo", "--shared", "-Xcompiler", "-fPIC",
              "-I", os.path.join(ROOT, "include"), *(extra or []), "-o", out, *srcs])
    return out


def build_workload_host(force: bool = False) -> str:
    d = os.path.join(PKG, "workload")
    out = os.path.join(d, "libwl_host.so")
    srcs = [os.path.join(d, "expand_host.c"), os.path.join(d, "expand_core.h")]
    if force or _stale(out, srcs):
        _run(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-pthread", "-o", out, srcs[0]])
    return out


def build_workload_device(force: bool = False) -> str:
    d = os.path.join(PKG, "workload")
    out = os.path.join(d, "libwl_device.so")
    srcs = [os.path.join(d, "expand_device.cu"), os.path.join(d, "expand_core.h")]
    if force or _stale(out, srcs):
        _run([NVCC, *ARCH, "-O3", "-lineinfo", "--shared", "-Xcompiler", "-fPIC", "-o", out, srcs[0]])
    return out


def build_all(force: bool = False) -> List[str]:
    return [build_argus(force), build_workload_host(force), build_workload_device(force)]
