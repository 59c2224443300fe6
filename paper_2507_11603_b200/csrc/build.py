"""Builds libthor_b200.so in-tree with nvcc for sm_100a only (no other arch, no fallback)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(os.path.dirname(HERE), "libthor_b200.so")
SOURCES = ["api.cu", "walk.cu", "unit_kernels.cu"]
DEPS = SOURCES + ["walk.cuh", "params.cuh", "philox.cuh", "dda.cuh", "voigt.cuh", "voigt_table.inc", "sampler.cuh",
                  os.path.join("..", "..", "include", "thor.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--shared",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-cudart", "shared",
              # approximate (2 ulp) division and square root for the samplers; the DDA and Voigt use explicit
              # __fdiv_rn / __fmul_rn / __fadd_rn / __frcp_rn intrinsics, which these flags do not touch
              "-prec-div=false", "-prec-sqrt=false"]


def build(force=False, verbose=False):
    deps = [os.path.join(HERE, d) for d in DEPS]
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + [os.path.join(HERE, s) for s in SOURCES] + ["-o", LIB]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        print(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libthor_b200.so")
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
