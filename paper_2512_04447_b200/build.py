"""Build step for librsdft.so (the CUDA path): one nvcc call, sm_100a only, in-tree.

    python -m paper_2512_04447_b200.build [--force]

nvcc cross-compiles without a GPU, so this runs on the CPU box; the built .so travels to the
GPU box with the repo snapshot (it is git-ignored, not gpurun-ignored)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librsdft.so")
PROBE_LIB = os.path.join(HERE, "libpeakprobe.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def sources():
    deps = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh"))]
    deps.append(os.path.join(ROOT, "include", "rsdft.h"))
    return deps


def _stale(lib, deps, force):
    return force or not os.path.exists(lib) or any(os.path.getmtime(lib) < os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    """Compile csrc/rsdft.cu -> librsdft.so (the product) and csrc/peak_probe.cu -> libpeakprobe.so
    (bench.py's roofline-denominator probe) if any source is newer than the library."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = ["-Xptxas", "-v"] if verbose else []
    if _stale(LIB, [d for d in sources() if not d.endswith("peak_probe.cu")], force):
        subprocess.check_call([nvcc] + NVCC_FLAGS + extra + ["-o", LIB, os.path.join(CSRC, "rsdft.cu")])
    if _stale(PROBE_LIB, [os.path.join(CSRC, "peak_probe.cu")], force):
        subprocess.check_call([nvcc] + NVCC_FLAGS + extra + ["-o", PROBE_LIB, os.path.join(CSRC, "peak_probe.cu")])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
