"""In-tree build of libhelios_b200.so (nvcc, sm_100a only)."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
# HELIOS_B200_LIB: path of an already built libhelios_b200.so to load instead of the in-tree one
LIB_PATH = os.environ.get("HELIOS_B200_LIB") or os.path.join(HERE, "libhelios_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "--use_fast_math=false",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libhelios_b200.so cannot be built (there is no CPU fallback)")


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh")))


def is_stale() -> bool:
    if os.environ.get("HELIOS_B200_LIB"):
        return False
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    deps = sources() + [os.path.join(INCLUDE, "helios.h")]
    return any(os.path.getmtime(s) > t for s in deps)


def build_library(force: bool = False, verbose: bool = False, defines=(), out: str = None) -> str:
    """nvcc -> LIB_PATH (or `out`); `defines` are extra -D macros (kernel experiments)."""
    out = out or LIB_PATH
    if not force and out == LIB_PATH and not is_stale():
        return LIB_PATH
    tmp = out + f".tmp{os.getpid()}"
    cmd = [_nvcc()] + [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [f"-D{d}" for d in defines]
    cmd += ["-I", INCLUDE, "-o", tmp, os.path.join(CSRC, "helios_api.cu")]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stderr)
    os.replace(tmp, out)
    return out
