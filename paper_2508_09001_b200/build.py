"""Builds libretro.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2508_09001_b200.build [--force]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot."""
from __future__ import annotations

import contextlib
import fcntl
import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
LIB_DIR = os.path.join(PKG, "lib")
LIB_PATH = os.path.join(LIB_DIR, "libretro.so")
DBG_LIB_PATH = os.path.join(LIB_DIR, "libretro_dbg.so")
NVTX_LIB_PATH = os.path.join(LIB_DIR, "libretro_nvtx.so")
INCLUDE = os.path.join(os.path.dirname(PKG), "include")



def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cu"))


def _stale(lib_path: str = None) -> bool:
    lib_path = lib_path or LIB_PATH
    if not os.path.exists(lib_path):
        return True
    t = os.path.getmtime(lib_path)
    deps = sources() + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")]
    deps.append(os.path.join(INCLUDE, "retro.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build_debug(force: bool = False) -> str:
    """The same library with -DRETRO_DEBUG_CHECKS (device-side index validation) -> lib/libretro_dbg.so."""
    return build(force=force, lib_path=DBG_LIB_PATH, extra_flags=["-DRETRO_DEBUG_CHECKS"], obj_suffix=".dbg.o")


def build_nvtx(force: bool = False) -> str:
    """The same library with -DRETRO_NVTX (every entry point is an NVTX range) -> lib/libretro_nvtx.so."""
    return build(force=force, lib_path=NVTX_LIB_PATH, extra_flags=["-DRETRO_NVTX"], obj_suffix=".nvtx.o")


@contextlib.contextmanager
def _build_lock():
    """One builder at a time per checkout: the ranks of a torchrun launch (or parallel test workers) that all find
    the library stale take turns; every rank after the first then finds it up to date."""
    os.makedirs(LIB_DIR, exist_ok=True)
    with open(os.path.join(LIB_DIR, ".build.lock"), "w") as f:
        fcntl.flock(f, fcntl.LOCK_EX)
        try:
            yield
        finally:
            fcntl.flock(f, fcntl.LOCK_UN)


def build(force: bool = False, verbose: bool = False, lib_path: str = LIB_PATH, extra_flags=(),
          obj_suffix: str = ".o") -> str:
    if not force and not _stale(lib_path):
        return lib_path
    with _build_lock():
        if not force and not _stale(lib_path):      # another process built it while this one waited
            return lib_path
        return _build_locked(verbose, lib_path, extra_flags, obj_suffix)


def _build_locked(verbose: bool, lib_path: str, extra_flags, obj_suffix: str) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    for src in sources():
        obj = os.path.join(LIB_DIR, os.path.basename(src)[:-3] + obj_suffix)
        cmd = [nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
               "-Xcompiler", "-fPIC", "-I", INCLUDE, "-c", src, "-o", obj]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += list(extra_flags)
        cmd += os.environ.get("RETRO_NVCC_FLAGS", "").split()     # extra nvcc flags for experiments
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = False
    for src, pr in procs:
        out, _ = pr.communicate()
        if pr.returncode != 0 or verbose:
            sys.stderr.write(f"--- nvcc {os.path.basename(src)}\n{out}\n")
        failed |= pr.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building libretro.so")
    # link to a temporary name and rename: a process that has the old library mapped keeps a consistent file
    tmp_path = lib_path + f".tmp{os.getpid()}"
    link = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp_path] + objs
    r = subprocess.run(link, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout)
        raise RuntimeError("nvcc link failed for libretro.so")
    os.replace(tmp_path, lib_path)
    return lib_path


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--debug" in sys.argv:
        print(build_debug(force="--force" in sys.argv))
    if "--nvtx" in sys.argv:
        print(build_nvtx(force="--force" in sys.argv))
