"""Build paper_1601_02063_b200/libodyssey.so (the C-ABI library of include/odyssey.h) in-tree with nvcc
for sm_100a.  nvcc cross-compiles without a GPU; the built .so travels to the GPU box with the snapshot."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libodyssey.so")
SOURCES = ["odyssey_api.cu"]
DEPS = ["odyssey_api.cu", "odyssey_kernels.cuh", "geodesic.cuh", "emission.cuh", "params.h", "bessel_k2_coeffs.h",
        "dmath.cuh", "dmath_coeffs.h",
        os.path.join("..", "..", "include", "odyssey.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force=False, verbose=False):
    """Compile if any source is newer than the library.  Returns the library path; the ptxas
    resource report (registers, spills) is written next to it as libodyssey.ptxas.txt."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", LIB] + SOURCES
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    with open(os.path.join(HERE, "libodyssey.ptxas.txt"), "w") as f:
        f.write("$ " + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libodyssey.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
