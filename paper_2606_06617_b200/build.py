"""Build libpswf_lr.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_06617_b200.build [--force]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["pswf_lr.cu", "kernels_generic.cu", "kernels_stencil.cu", "kernels_gather.cu", "kernels_fft.cu", "kernels_real.cu"]
HEADERS = ["plan.hpp", "launch.hpp", "host_tables.hpp", "real_tables.hpp", "kernels_common.cuh", "kernels_scale.cuh",
           os.path.join("..", "..", "include", "pswf_lr.h")]
LIB = os.path.join(HERE, "libpswf_lr.so")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    nvcc = os.path.join(CUDA_HOME, "bin", "nvcc")
    objs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, s), "-o", o]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed on %s" % s)
        objs.append(o)
    libdir = os.path.join(CUDA_HOME, "lib64")
    cmd = [nvcc, "-shared", "-o", LIB] + objs + ["-L" + libdir, "-lcufft", "-Xlinker", "-rpath=" + libdir]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
