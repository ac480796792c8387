"""Build step: compile csrc/*.cu into libpic_b200.so for sm_100a with nvcc (in-tree, so the
built library travels to the GPU box with the snapshot).  No torch dependency: the library is
plain CUDA runtime + C-ABI (include/pic.h)."""
import glob
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpic_b200.so")
LIB_CHECK = os.path.join(_HERE, "libpic_b200_check.so")   # bounds-checked debug build
CHECK_FLAGS = ["-DPIC_BOUNDS_CHECK=1", "-rdc=true"]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale(lib=LIB):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = glob.glob(os.path.join(CSRC, "*")) + [os.path.join(_HERE, "..", "include", "pic.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, check=False):
    """nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo ... -> libpic_b200.so
    (check=True: the bounds-checked debug build libpic_b200_check.so, csrc/pic_check.cuh)"""
    lib = LIB_CHECK if check else LIB
    if not force and not _stale(lib):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (CHECK_FLAGS if check else []) + \
        (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + sources()
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
