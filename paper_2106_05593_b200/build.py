"""Builds libmmc_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmmc_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CU = ["api.cu", "kernels_sweep.cu", "kernels_layout.cu", "demag.cu", "static_scratch.cu"]
CPP = ["mmc_host.cpp"]
NVFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + os.environ.get("MMC_NVCC_FLAGS", "").split()   # e.g. -DMMC_COLS_MINB=2 (tuning knobs of csrc/)


def _newer(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _flags_changed() -> bool:
    """The full compile command lines are part of the build's identity: a change of MMC_NVCC_FLAGS (the -D tuning knobs of
    csrc/) or of the compiler must rebuild everything, or an A/B run would time the same binary twice."""
    stamp = os.path.join(OBJ, "flags.stamp")
    ident = " ".join([NVCC] + NVFLAGS) + "\n"
    try:
        with open(stamp) as fh:
            same = fh.read() == ident
    except OSError:
        same = False
    if not same:
        with open(stamp, "w") as fh:
            fh.write(ident)
    return not same


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    force = _flags_changed() or force
    hdrs = [os.path.join(CSRC, h) for h in ("mmc_internal.h", "fft_reg.cuh", "fft_reg8.cuh", "fft_smem.cuh")] + [os.path.join(HERE, "..", "include", "mmc.h")]
    objs = []
    jobs = []
    for f in CU + CPP:
        src = os.path.join(CSRC, f)
        obj = os.path.join(OBJ, f.rsplit(".", 1)[0] + ".o")
        objs.append(obj)
        if force or _newer(obj, [src] + hdrs):
            if f.endswith(".cu"):
                cmd = [NVCC] + NVFLAGS + ["-c", src, "-o", obj]
            else:
                cmd = ["g++", "-O2", "-std=gnu++17", "-fPIC", "-I/usr/local/cuda/include", "-c", src, "-o", obj]
            jobs.append((f, cmd))

    def compile_one(job):
        f, cmd = job
        r = subprocess.run(cmd, capture_output=True, text=True)
        with open(os.path.join(OBJ, f + ".log"), "w") as fh:
            fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        return f, cmd, r

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=max(1, min(len(jobs), os.cpu_count() or 1))) as ex:     # the translation units compile side by side
        for f, cmd, r in ex.map(compile_one, jobs):
            if verbose or r.returncode:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode:
                raise RuntimeError("compile failed: " + " ".join(cmd))
    if force or _newer(LIB, objs):
        cmd = [NVCC, "-shared", "-o", LIB] + objs + ["-L/usr/local/cuda/lib64", "-lcufft", "-lquadmath",
                                                      "-Xlinker", "-rpath,/usr/local/cuda/lib64"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
