"""Build tests/harness/blip_harness (plain C, gcc) against paper_1204_1121_b200/libblipgpu.so and
the CUDA runtime.  Used by tests/test_gpu_harness.py, by bench.py's per-call latency rows and
by the compute-sanitizer runs recorded under profiles/."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
SRC = os.path.join(HERE, "blip_harness.c")
EXE = os.path.join(HERE, "blip_harness")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def build(force=False, checked=False):
    """checked=True: the library is compiled with -DBLIP_CHECKED (every index the kernels compute is
    compared with its bound and a violation traps; csrc/blip_types.h) into
    tests/harness/libblipgpu_checked.so and the harness is linked against that."""
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    from paper_1204_1121_b200 import _build
    if checked:
        lib = os.path.join(HERE, "libblipgpu_checked.so")
        if force or not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in _build.DEPS):
            subprocess.run([_build.nvcc(), *_build.NVCC_FLAGS, "-DBLIP_CHECKED", "-I", os.path.join(ROOT, "include"),
                            "-o", lib, *_build.SOURCES], check=True)
        exe, name = EXE + "_checked", "blipgpu_checked"
    else:
        lib = _build.build()
        exe, name = EXE, "blipgpu"
    libdir = os.path.dirname(lib)
    deps = [SRC, lib, os.path.join(ROOT, "include", "blipgpu.h"), os.path.join(ROOT, "include", "blipgpu_dev.h")]
    if not force and os.path.exists(exe) and all(os.path.getmtime(exe) >= os.path.getmtime(d) for d in deps):
        return exe
    cmd = ["gcc", "-O2", "-std=c11", "-D_POSIX_C_SOURCE=200809L", "-Wall", "-Wextra", "-I", os.path.join(ROOT, "include"),
           "-I", os.path.join(CUDA, "include"), "-o", exe, SRC, "-L", libdir, "-l" + name,
           "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-lm", "-ldl",
           "-Wl,-rpath," + libdir, "-Wl,-rpath," + os.path.join(CUDA, "lib64")]
    subprocess.run(cmd, check=True)
    return exe


def build_tcgen05_check(force=False):
    """tests/harness/tcgen05_check.cu -> tests/harness/tcgen05_check (nvcc, sm_100a): the tensor-memory /
    tcgen05.mma facts the tensor-core kernel relies on, checked against a host loop."""
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    from paper_1204_1121_b200 import _build
    src, exe = os.path.join(HERE, "tcgen05_check.cu"), os.path.join(HERE, "tcgen05_check")
    if force or not os.path.exists(exe) or os.path.getmtime(src) > os.path.getmtime(exe):
        subprocess.run([_build.nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-o", exe, src], check=True)
    return exe


def build_mma_sync_probe(force=False):
    """tests/harness/mma_sync_probe.cu (+ .cuh) -> tests/harness/mma_sync_probe (nvcc, sm_100a): the settled
    mma.sync tf32 recast experiment of SURVEY.md §8f NEXT-2, kept out of the shipped library."""
    if ROOT not in sys.path:
        sys.path.insert(0, ROOT)
    from paper_1204_1121_b200 import _build
    srcs = [os.path.join(HERE, "mma_sync_probe.cu"), os.path.join(HERE, "mma_sync_probe.cuh")]
    exe = os.path.join(HERE, "mma_sync_probe")
    if force or not os.path.exists(exe) or any(os.path.getmtime(x) > os.path.getmtime(exe) for x in srcs):
        subprocess.run([_build.nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe, srcs[0]], check=True)
    return exe


if __name__ == "__main__":
    print(build(force=True, checked="--checked" in sys.argv))
