"""Builds libgk.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2604_06085_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libgk.so")
OBJDIR = os.path.join(HERE, "build")
# (source, extra defines, object name): the stage kernel is instantiated once per storage type in
# its own translation unit so that the units compile in parallel
UNITS = [
    ("gk_lib.cu", [], "gk_lib.o"),
    ("gk_noalloc.cu", [], "gk_noalloc.o"),   # gk_spectra_static: context-free, fixed scratch in the library image
    ("gk_stage_inst.cu", ["-DGK_ST_ID=0"], "gk_stage_c64.o"),
    ("gk_stage_inst.cu", ["-DGK_ST_ID=1"], "gk_stage_f16.o"),
    ("gk_stage_inst.cu", ["-DGK_ST_ID=2"], "gk_stage_bf16.o"),
]


def _csrc_files():
    """Every translation unit includes (directly or not) every header of csrc/: one dependency list."""
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".h")))


NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def src_hash() -> str:
    """sha256 (16 hex digits) over the names and contents of every file of csrc/: compiled into gk_version() so that
    counters captured from one build (profiles/stage_traffic.json) are never quoted for another."""
    import hashlib
    h = hashlib.sha256()
    for path in _csrc_files():
        h.update(os.path.basename(path).encode() + b"\0")
        with open(path, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def _flags_now() -> str:
    fast = bool(os.environ.get("GK_FAST_BUILD"))           # developer builds only: complex64 storage
    return " ".join([*NVCC_FLAGS, *(["-DGK_ONLY_C64"] if fast else [])])


def _include_files():
    return sorted(os.path.join(INCLUDE, f) for f in os.listdir(INCLUDE) if f.endswith(".h"))


def is_stale() -> bool:
    """The library is rebuilt if it is missing, older than any file of csrc/ or include/, or was built with
    other flags (GK_FAST_BUILD)."""
    flagfile = os.path.join(OBJDIR, "flags.txt")
    if not os.path.exists(LIB) or not os.path.exists(flagfile) or open(flagfile).read() != _flags_now():
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in _csrc_files() + _include_files())


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than its sources; returns the library path."""
    if not force and not is_stale():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(OBJDIR, exist_ok=True)
    fast = bool(os.environ.get("GK_FAST_BUILD"))           # developer builds only: complex64 storage
    units = UNITS[:3] if fast else UNITS
    extra = ["-DGK_ONLY_C64"] if fast else []

    flagfile = os.path.join(OBJDIR, "flags.txt")
    flags_now = _flags_now()
    same_flags = os.path.exists(flagfile) and open(flagfile).read() == flags_now

    def compile_unit(u):
        src, defs, obj = u
        objp = os.path.join(OBJDIR, obj)
        if src == "gk_lib.cu":
            defs = [*defs, f'-DGK_SRC_HASH="{src_hash()}"']
        cmd = [_nvcc(), *NVCC_FLAGS, *extra, *defs, "-c", os.path.join(CSRC, src), "-o", objp]
        deps = _csrc_files() + _include_files()
        if not force and same_flags and os.path.exists(objp) and all(os.path.getmtime(d) <= os.path.getmtime(objp) for d in deps):
            return cmd, subprocess.CompletedProcess(cmd, 0, "(up to date)\n", "")
        res = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, res

    with ThreadPoolExecutor(len(units)) as ex:
        results = list(ex.map(compile_unit, units))
    log = ""
    for cmd, res in results:
        log += " ".join(cmd) + "\n" + res.stdout + res.stderr
    tmp = LIB + f".{os.getpid()}.tmp"
    ok = all(res.returncode == 0 for _, res in results)
    if ok:
        cmd = [_nvcc(), "--shared", "-gencode", "arch=compute_100a,code=sm_100a",
               *[os.path.join(OBJDIR, u[2]) for u in units], "-o", tmp]
        res = subprocess.run(cmd, capture_output=True, text=True)
        log += " ".join(cmd) + "\n" + res.stdout + res.stderr
        ok = res.returncode == 0
    with open(os.path.join(HERE, "build.log"), "w") as fh:
        fh.write(log)
    if not ok:
        sys.stderr.write(log)
        raise RuntimeError("nvcc failed building libgk.so")
    os.replace(tmp, LIB)
    with open(flagfile, "w") as fh:
        fh.write(flags_now)
    if verbose:
        print(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
