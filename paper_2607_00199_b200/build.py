"""In-tree build of libalegb.so (the C-ABI library of include/alegb.h) for sm_100a.

    python -m paper_2607_00199_b200.build [--force] [--verbose]

Host setup code (csrc/host_ref.cpp) is compiled with g++ (it uses __float128); the kernels and the ABI with
nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo.  The shared object lands next to this file so that it
travels with the repository snapshot; nothing is installed anywhere else.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libalegb.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CXX = os.environ.get("CXX", "g++")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
CXX_FLAGS = ["-O2", "-std=c++17", "-fPIC"]

CU_SOURCES = ["kernels.cu", "stage_pipe.cu", "pml_mma.cu", "cubature.cu", "fp64_peak.cu", "alegb_api.cu"]
CXX_SOURCES = ["host_ref.cpp"]
HEADERS = ["alegb_internal.h", "device_common.cuh", "host_ref.h", os.path.join("..", "..", "include", "alegb.h")]


def _newer(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps if os.path.exists(d))


def _run(cmd, verbose, log):
    r = subprocess.run(cmd, capture_output=True, text=True)
    log.append("$ " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose:
        sys.stdout.write(log[-1])
    if r.returncode != 0:
        raise RuntimeError("build failed:\n" + log[-1])


def build(force=False, verbose=False):
    """Compile (if stale) and return the path of libalegb.so."""
    os.makedirs(OBJ, exist_ok=True)
    headers = [os.path.join(CSRC, h) for h in HEADERS]
    log, objs = [], []
    for src in CXX_SOURCES:
        s, o = os.path.join(CSRC, src), os.path.join(OBJ, src + ".o")
        if force or _newer(o, [s] + headers):
            _run([CXX] + CXX_FLAGS + ["-c", s, "-o", o], verbose, log)
        objs.append(o)
    jobs = []
    for src in CU_SOURCES:
        s, o = os.path.join(CSRC, src), os.path.join(OBJ, src + ".o")
        if not os.path.exists(s):
            continue
        if force or _newer(o, [s] + headers):
            jobs.append([NVCC] + NVCC_FLAGS + ["-c", s, "-o", o])
        objs.append(o)
    if jobs:   # the translation units are independent: compile them side by side
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as pool:
            logs = [[] for _ in jobs]
            list(pool.map(lambda jl: _run(jl[0], verbose, jl[1]), zip(jobs, logs)))
        for l in logs:
            log.extend(l)
    if force or _newer(LIB, objs):
        _run([NVCC, "-shared", "-o", LIB] + objs + ["-lquadmath"], verbose, log)
    with open(os.path.join(OBJ, "build.log"), "a") as f:
        f.write("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
