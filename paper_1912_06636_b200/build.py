"""Build libaims_gpu.so in-tree with nvcc for sm_100a (B200).  `python -m paper_1912_06636_b200.build`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "csrc", f) for f in ("aims_gpu.cu", "batching.cu", "periodic.cu")]
LIB = os.path.join(HERE, "libaims_gpu.so")
DEPS = [os.path.join(HERE, "csrc", f) for f in sorted(os.listdir(os.path.join(HERE, "csrc"))) if f.endswith((".cu", ".cuh"))]
DEPS.append(os.path.join(os.path.dirname(HERE), "include", "aims_gpu.h"))


def nvcc_path():
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    return "nvcc"


def build(force=False, verbose=False, defines=(), tag=None):
    """defines / tag: a PROBE build for the profiles (e.g. `--define AIMS_PROBE_H_EPILOGUE=0 --tag noepi` writes
    libaims_gpu_noepi.so, which reports its switches through aims_gpu_build_flags(); run it with `bench.py --lib <path>` or
    binding.load_library(path, allow_probe=True)).  The product library is the untagged one and is built without switches."""
    lib = LIB if not tag else os.path.join(HERE, "libaims_gpu_%s.so" % tag)
    if not force and not defines and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in DEPS):
        return lib
    tmp = lib + ".%d.tmp" % os.getpid()
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
           "-Xcompiler", "-fPIC", "--threads", "2", "-o", tmp] + ["-D" + d for d in defines] + SRC
    if defines:
        cmd.insert(-len(SRC), '-DAIMS_BUILD_FLAGS="%s"' % " ".join(defines))
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    subprocess.check_call(cmd)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    argv = sys.argv[1:]
    defs = [argv[i + 1] for i, a in enumerate(argv) if a == "--define"]
    tag = next((argv[i + 1] for i, a in enumerate(argv) if a == "--tag"), None)
    if defs and not tag:
        raise SystemExit("--define needs --tag (the product library is never built with probe switches)")
    print(build(force="--force" in argv, verbose="-v" in argv, defines=defs, tag=tag))
