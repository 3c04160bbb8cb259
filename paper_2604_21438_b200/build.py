"""Build libsfh.so (CUDA, sm_100a only) in-tree with nvcc.

    python -m paper_2604_21438_b200.build [--force] [--nofma] [--verbose]

nvcc cross-compiles without a GPU.  --nofma builds libsfh_nofma.so with -fmad=false (a debugging
aid: without FMA contraction the kernels round like the -ffp-contract=off CPU oracle).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["sfh_mesh.cpp", "sfh_kernels.cu", "sfh_kernels_mf.cu", "sfh_kernels_aux.cu", "sfh_kernels_scalar.cu", "sfh_api.cu", "sfh_noalloc.cu"]
HEADERS = ["sfh_internal.h", "sfh_device.cuh", "sfh_kernels.cuh", "sfh_stage.cuh", os.path.join("..", "..", "include", "sfh.h")]


def lib_path(nofma=False):
    return os.path.join(HERE, "libsfh_nofma.so" if nofma else "libsfh.so")


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def build(force=False, nofma=False, verbose=False):
    out = lib_path(nofma)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(d) for d in deps):
        return out
    cmd = [_nvcc(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--threads", "0", "-o", out]
    if nofma:
        cmd += ["-fmad=false"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, f) for f in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building %s" % out)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, nofma="--nofma" in sys.argv, verbose="--verbose" in sys.argv))
