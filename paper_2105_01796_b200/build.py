"""Build libkf_fit.so (the C-ABI library of include/kf_fit.h) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU, so this runs on the CPU box too (`__graft_entry__.build()`).
The built library is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(_ROOT, "include")
LIB_PATH = os.path.join(_HERE, "libkf_fit.so")
OBJ_DIR = os.path.join(_HERE, "build")  # git-ignored


def sources() -> list:
    """The translation units of the library: csrc/*.cu (kf_fit.cu = C ABI + host logic; the others one kernel family each)."""
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def headers() -> list:
    """Every header a translation unit can include: csrc/*.cuh, csrc/*.h and include/*.h (globbed, so a new file is watched)."""
    return sorted(glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")) +
                  glob.glob(os.path.join(INCLUDE, "*.h")))


NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC",
    # IEEE double throughout: no fast-math; FMA contraction stays on
    "--fmad=true",
]


def nvcc_path() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libkf_fit.so cannot be built (there is no CPU fallback)")


STAMP = os.path.join(OBJ_DIR, "flags.txt")


def flag_stamp(extra_flags=()) -> str:
    """What the stamp file of a build holds: the path-independent nvcc flags, tuning -D macros included (the -I paths
    are left out: the repository sits at another path on the GPU box)."""
    return " ".join([*NVCC_FLAGS, *extra_flags])


def built_flags():
    """The flag stamp of the library that is there now (None: no stamp)."""
    try:
        with open(STAMP) as f:
            return f.read()
    except OSError:
        return None


def built_defines() -> list:
    """The -D macros the library that is there now was built with ([] for the default build)."""
    return [w for w in (built_flags() or "").split() if w.startswith("-D")]


def is_stale(extra_flags=()) -> bool:
    """True when the library is missing, older than a source or header, or was built with other flags than
    `extra_flags` asks for: a tuning build (`python build.py -DKF_FWD_MIN_BLOCKS=2`) is stale for every later default
    call (lib(), tests, bench, __graft_entry__.build), which therefore rebuilds instead of silently using it."""
    if not os.path.exists(LIB_PATH):
        return True
    if built_flags() != flag_stamp(extra_flags):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(p) > t for p in sources() + headers())


def _run(cmd):
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    return res.stderr


def build_library(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    """Compile every csrc/*.cu to an object (side by side, one nvcc each) and link them into libkf_fit.so.
    An object is rebuilt when its source or any header is newer (or `force`, or other flags than last time)."""
    if not force and not is_stale(extra_flags):
        return LIB_PATH
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(OBJ_DIR, exist_ok=True)
    nvcc = nvcc_path()
    flags = [*NVCC_FLAGS, *extra_flags, "-I", INCLUDE, "-I", CSRC]
    if verbose:
        flags = ["-Xptxas", "-v", *flags]
    same_flags = built_flags() == flag_stamp(extra_flags)
    newest_header = max(os.path.getmtime(p) for p in headers())
    jobs, objs = [], []
    for src in sources():
        obj = os.path.join(OBJ_DIR, os.path.splitext(os.path.basename(src))[0] + ".o")
        objs.append(obj)
        fresh = (not force and same_flags and os.path.exists(obj) and
                 os.path.getmtime(obj) > max(os.path.getmtime(src), newest_header))
        if not fresh:
            jobs.append([nvcc, *flags, "-c", "-o", obj, src])
    if verbose:
        for j in jobs:
            print(" ".join(j), file=sys.stderr)
    with ThreadPoolExecutor(max_workers=max(1, min(len(jobs), os.cpu_count() or 1))) as pool:
        for log in pool.map(_run, jobs):
            if verbose:
                print(log, file=sys.stderr)
    if os.path.exists(STAMP):
        os.remove(STAMP)  # a build that fails half-way leaves no stamp: the next call starts over
    _run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB_PATH, *objs])
    with open(STAMP, "w") as f:
        f.write(flag_stamp(extra_flags))
    return LIB_PATH


if __name__ == "__main__":
    # python build.py [--force] [-v] [-DNAME=VALUE ...]   (-D flags go to nvcc: the tuning macros KF_FWD_BLOCK,
    # KF_FWD_BLOCK_SMALL, KF_FWD_MIN_BLOCKS, KF_RTS_MIN_BLOCKS, KF_TILE, ... of csrc/kf_common.cuh)
    defines = [a for a in sys.argv[1:] if a.startswith("-D")]
    print(build_library(force="--force" in sys.argv or bool(defines), verbose="-v" in sys.argv, extra_flags=defines))
