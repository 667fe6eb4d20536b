"""Build the C-ABI CUDA libraries in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1812_07977_b200.build [--force]

Produces, next to this file:
  libhydro_b200.so         production build  (-fmad=true)
  libhydro_b200_verify.so  verification build (-fmad=false -DHYDRO_VERIFY): reproduces the
                           oracle's rounding order, used by the 1e-14 one-step parity tests.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["hydro_api.cu"]
HEADERS = ["hydro_math.cuh", "hydro_math_fast.cuh", "hydro_faces.cuh", "hydro_kernels.cuh", "hydro_stage_fused.cuh",
           "hydro_stage_fused_kernel.cuh", "hydro_stage_fused_plan.cuh", "hydro_stage_fused2d.cuh",
           "hydro_stage_fused1d.cuh", "hydro_stage_warp2d.cuh",
           "hydro_tma.cuh"]
LIB = os.path.join(HERE, "libhydro_b200.so")
LIB_VERIFY = os.path.join(HERE, "libhydro_b200_verify.so")

COMMON = os.environ.get("HYD_EXTRA_NVCC", "").split() + ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
          "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale(target):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    deps.append(os.path.join(os.path.dirname(HERE), "include", "hydro.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(target, extra, log):
    cmd = [_nvcc()] + COMMON + extra + ["-o", target] + [os.path.join(CSRC, s) for s in SOURCES]
    env = dict(os.environ)
    env.pop("CC", None); env.pop("CXX", None)      # the image's CC wrapper is not nvcc's host compiler
    out = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, env=env)
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + out.stdout)
    if out.returncode != 0:
        sys.stderr.write(out.stdout)
        raise RuntimeError(f"nvcc failed for {target}")


def build(force=False, verbose=False):
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    for target, extra in ((LIB, ["-fmad=true"]),
                          (LIB_VERIFY, ["-fmad=false", "-DHYDRO_VERIFY=1"])):
        if force or _stale(target):
            log = os.path.join(HERE, "build", os.path.basename(target) + ".log")
            _compile(target, extra, log)
            if verbose:
                print(open(log).read())
    return LIB, LIB_VERIFY


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
