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


def build_variant(out_path, extra_flags):
    """Compile a variant of the library (e.g. ["-DODY_DEVICE_CHECKS"]) to out_path; returns out_path."""
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + [f for f in NVCC_FLAGS if f not in ("-Xptxas", "-v")] + list(extra_flags) + ["-o", out_path] + SOURCES
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building " + out_path + "\n" + res.stderr[-2000:])
    return out_path


def build(force=False, verbose=False):
    """Compile if any source is newer than the library.  Returns the library path; the ptxas
    resource report (registers, spills) is written next to it as libodyssey.ptxas.txt.
    ODYSSEY_LIB in the environment names an already built library to load instead (a variant from build_variant)."""
    if os.environ.get("ODYSSEY_LIB"):
        return os.environ["ODYSSEY_LIB"]
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
