"""In-tree build of libmadspace_b200.so with nvcc for sm_100a (no torch types, no JIT cache).

The per-multiplicity kernels (csrc/ms_inst.cu, -DMS_N=2..9 -DMS_PART=0..2) compile as 24 translation units in parallel;
csrc/ms_api.cu holds the C ABI.  Objects live in csrc/build/ (git-ignored); the shared library lands beside
this file so that it travels to the GPU box with the repository snapshot.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
BUILD = os.path.join(CSRC, "build")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libmadspace_b200.so")

NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-diag-suppress", "177"]
HEADERS = ["ms_math.cuh", "ms_kernels.cuh", "ms_params.h", "ms_launch.h", "ms_vegas_inv.cuh"]
N_RANGE = range(9, 1, -1)


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")
    return exe


def _newest_source() -> float:
    files = [os.path.join(CSRC, f) for f in HEADERS + ["ms_inst.cu", "ms_api.cu"]]
    files.append(os.path.join(INCLUDE, "madspace_b200.h"))
    return max(os.path.getmtime(f) for f in files)


def _compile(args):
    src, obj, extra = args
    cmd = [_nvcc()] + NVCC_FLAGS + extra + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source():
        return LIB
    os.makedirs(BUILD, exist_ok=True)
    # one builder at a time: under torchrun every rank calls lib() -> build(), and all of them would compile into the
    # same csrc/build/*.o paths; the others wait here and then find the library up to date
    import fcntl
    with open(os.path.join(BUILD, ".lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source():
                return LIB
            return _build_locked(verbose)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(verbose: bool) -> str:
    jobs = [(os.path.join(CSRC, "ms_api.cu"), os.path.join(BUILD, "ms_api.o"), ["-I", INCLUDE])]
    for n in N_RANGE:                                  # largest multiplicities first: they take longest
        for part in (0, 1, 2):
            jobs.append((os.path.join(CSRC, "ms_inst.cu"), os.path.join(BUILD, "ms_inst_n%d_p%d.o" % (n, part)),
                         ["-DMS_N=%d" % n, "-DMS_PART=%d" % part]))
    import time
    t0 = time.time()
    with cf.ThreadPoolExecutor(max_workers=min(len(jobs), max(os.cpu_count() or 4, 4))) as ex:
        objs = list(ex.map(_compile, jobs))
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc(), "-shared", "-o", tmp] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed: %s\n%s" % (r.stdout, r.stderr))
    os.replace(tmp, LIB)
    if verbose:
        print("compiled %d translation units from source with %s %s in %.0f s" % (len(jobs), _nvcc(), " ".join(NVCC_FLAGS[:5]),
                                                                                 time.time() - t0))
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force=True, verbose=True)
