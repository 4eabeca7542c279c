"""Compile the CUDA path into paper_2305_16652_b200/libhcc_b200.so (sm_100a only).

nvcc cross-compiles without a GPU.  -fmad=false: every source-level floating-point
operation is one IEEE operation; fused multiply-adds appear only where fmaf() is written
(the arithmetic include/hcc.h states must hold bit for bit)."""
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(_HERE, "libhcc_b200.so")
HEADER = os.path.join(os.path.dirname(_HERE), "include", "hcc.h")
SOURCES = ["bvh.cu", "cut.cu", "cutflat.cu", "encode.cu", "sort.cu", "trace.cu", "pipeline.cu"]

NVCC = os.environ.get("NVCC", "nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-fmad=false", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _deps():
    return [HEADER, os.path.join(CSRC, "common.cuh")]


def _stale(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    objs, jobs = [], []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src[:-3] + ".o")
        objs.append(o)
        if force or _stale(o, [s] + _deps()):
            cmd = [NVCC, *FLAGS, "-c", s, "-o", o]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            jobs.append(cmd)
    if jobs:
        with ThreadPoolExecutor(max_workers=min(6, len(jobs))) as ex:
            for r in ex.map(lambda c: subprocess.run(c, capture_output=True, text=True), jobs):
                if verbose and r.stderr:
                    print(r.stderr)
                if r.returncode != 0:
                    raise RuntimeError("nvcc failed:\n" + " ".join(r.args) + "\n" + r.stdout + r.stderr)
    if jobs or force or _stale(LIB, objs):
        cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp", *objs]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
        os.replace(LIB + ".tmp", LIB)
    return LIB


def build_pipe_rates():
    """The instruction-rate microbenchmark (csrc/pipe_rates.cu): a standalone debug program, not part of the library."""
    out = os.path.join(_HERE, "pipe_rates")
    cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           os.path.join(CSRC, "pipe_rates.cu"), "-o", out]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    return out


if __name__ == "__main__":
    import sys
    if "--pipe-rates" in sys.argv:
        print(build_pipe_rates())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
