"""Build the C-ABI CUDA library in-tree: csrc/*.cu -> paper_1008_0135_b200/libvr_b200.so (sm_100a only).

nvcc cross-compiles without a GPU; the .so is git-ignored but travels to the GPU box with gpurun.

Experiment variants (VR_DEFINES="-DVR_EXP_..." in the environment, the switches recorded under profiles/) are written
to a file of their own, libvr_b200.exp-<hash of the defines>.so, and vr.py loads that file only while VR_DEFINES is set
to the same string: an experiment build can never stand in for the product library.
"""
import glob
import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libvr_b200.so")
SOURCES = [os.path.join(CSRC, "vr_api.cu")]


def deps():
    """Everything the library is compiled from: every file under csrc/ and the public headers."""
    return sorted(glob.glob(os.path.join(CSRC, "*")) + glob.glob(os.path.join(ROOT, "include", "*.h")))


def defines():
    return os.environ.get("VR_DEFINES", "").split()


def lib_path() -> str:
    """Path of the library for the current VR_DEFINES: the product file when there are none."""
    d = defines()
    if not d:
        return LIB
    return os.path.join(HERE, "libvr_b200.exp-" + hashlib.sha1(" ".join(d).encode()).hexdigest()[:10] + ".so")


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def build(force: bool = False, verbose: bool = False) -> str:
    out = lib_path()
    newest = max(os.path.getmtime(p) for p in deps())
    if not force and os.path.exists(out) and os.path.getmtime(out) >= newest:
        return out
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + defines() + (["-Xptxas", "-v"] if verbose else []) + ["-o", out] + SOURCES
    subprocess.run(cmd, check=True, cwd=HERE)
    return out


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
