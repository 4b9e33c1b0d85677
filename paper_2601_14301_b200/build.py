"""Compile csrc/ into paper_2601_14301_b200/libtrimeg.so for sm_100a with nvcc (in-tree)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtrimeg.so")
SOURCES = ["trimeg_lib.cu", "trimeg_push.cu", "trimeg_push_wcache.cu", "trimeg_push_lane.cu", "trimeg_push_wcache_core.cu",
           "trimeg_push_lane_core.cu", "trimeg_push_lane_spline.cu", "trimeg_scatter.cu", "trimeg_em.cu", "trimeg_em_core.cu"]
DEPS = SOURCES + ["trimeg_device.cuh", "trimeg_lane.cuh", "trimeg_rk4.cuh", "trimeg_internal.h", "trimeg_mesh.cuh", "bell_tables.inc", os.path.join("..", "..", "include", "trimeg.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-ffp-contract=off", "-shared"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def build(force: bool = False, verbose: bool = False, profile: bool = False) -> str:
    """profile: compile the in-kernel clock64 phase timers of the warp kernels in (-DTRIMEG_PROFILE)."""
    deps = [os.path.join(CSRC, d) for d in DEPS]
    profile = profile or os.environ.get("TRIMEG_PROFILE", "") not in ("", "0")
    if not force and not profile and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    extra = os.environ.get("TRIMEG_NVCC_EXTRA", "").split()          # experiments only (e.g. "-Xptxas -O1")
    cmd = [nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + (["-DTRIMEG_PROFILE"] if profile else []) + \
          ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, profile="--profile" in sys.argv))
