"""Build paper_1204_1121_b200/libblipgpu.so (the C-ABI library of include/blipgpu.h) with nvcc
for sm_100a, in-tree.  nvcc cross-compiles without a GPU."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libblipgpu.so")
SOURCES = [os.path.join(CSRC, "blipgpu.cu"), os.path.join(CSRC, "blipgpu_dev.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cuh", ".h"))] + [
    os.path.join(ROOT, "include", "blipgpu.h"), os.path.join(ROOT, "include", "blipgpu_dev.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC,-ffp-contract=off", "-shared",
]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force=False, verbose=False):
    # BLIPGPU_LIBRARY (read here, by the Python binding, not by the library): load this build of the
    # same ABI instead, e.g. tests/harness/libblipgpu_checked.so to run the GPU suite with the
    # kernels' bounds asserts on (profiles/r2_checks.md)
    override = os.environ.get("BLIPGPU_LIBRARY")
    if override:
        if not os.path.exists(override):
            raise FileNotFoundError(f"BLIPGPU_LIBRARY={override} does not exist")
        return override
    if not force and not stale():
        return LIB
    cmd = [nvcc(), *NVCC_FLAGS, "-I", os.path.join(ROOT, "include"), "-o", LIB, *SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
