"""Build libpd.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

Usage: python -m paper_2606_26089_b200.build [--force]   (also called by __graft_entry__.build()).
nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the gpurun snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpd.so")
SOURCES = ["pd_card.cpp", "pd_api.cu", "pd_particles.cu", "pd_towers.cu", "pd_features.cu", "pd_filter.cu", "pd_pileup.cu", "pd_impact.cu", "pd_truth.cu"]
HEADERS = [os.path.join(CSRC, "pd_internal.h"), os.path.join(CSRC, "pd_math.cuh"), os.path.join(CSRC, "pd_scan.cuh"), os.path.join(CSRC, "pd_impact_math.cuh"), os.path.join(ROOT, "include", "pd.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-Wall,-Wextra", "--expt-relaxed-constexpr",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    newest = max(os.path.getmtime(p) for p in srcs + HEADERS + [os.path.abspath(__file__)])
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    objs = []
    for src in srcs:
        obj = os.path.join(CSRC, os.path.basename(src) + ".o")
        cmd = [_nvcc(), *NVCC_FLAGS, "-x", "cu", "-c", src, "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.check_call(cmd)
        objs.append(obj)
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *objs])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
