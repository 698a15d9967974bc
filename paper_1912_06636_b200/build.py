"""Build libaims_gpu.so in-tree with nvcc for sm_100a (B200).  `python -m paper_1912_06636_b200.build`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "csrc", "aims_gpu.cu"), os.path.join(HERE, "csrc", "batching.cu")]
LIB = os.path.join(HERE, "libaims_gpu.so")
DEPS = [os.path.join(HERE, "csrc", f) for f in ("aims_gpu.cu", "batching.cu", "common.cuh", "basis.cuh", "hamiltonian.cuh", "density.cuh", "forces.cuh", "hessian.cuh", "bloch.cuh", "partition.cuh")]
DEPS.append(os.path.join(os.path.dirname(HERE), "include", "aims_gpu.h"))


def nvcc_path():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    return "nvcc"


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + ".%d.tmp" % os.getpid()
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
           "-Xcompiler", "-fPIC", "--threads", "2", "-o", tmp] + SRC
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
