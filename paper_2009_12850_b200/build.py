"""Build the C-ABI CUDA library in-tree for sm_100a.

    python -m paper_2009_12850_b200.build [--force] [--verbose]

Output: paper_2009_12850_b200/libmonc_adv.so (git-ignored; travels to the GPU
box with the gpurun snapshot) and, with --checked, libmonc_adv_checked.so: the
same sources with -DMONC_ADV_CHECKED=1 (ring slots poisoned with NaN before every
refill, pseudo-random delays around every slot access; csrc/monc_adv_tma.cuh),
used by tests/test_gpu_checked.py.  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmonc_adv.so")
LIB_CHECKED = os.path.join(HERE, "libmonc_adv_checked.so")
SOURCES = [os.path.join(CSRC, "monc_adv.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "monc_adv_kernels.cuh"),
                  os.path.join(CSRC, "monc_adv_tma.cuh"),
                  os.path.join(ROOT, "include", "monc_adv.h"),
                  os.path.join(ROOT, "include", "monc_adv_tuning.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-split-compile", "0",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
         "-I", os.path.join(ROOT, "include"), "-I", CSRC]


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    lib = LIB_CHECKED if checked else LIB
    if (not force and os.path.exists(lib)
            and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in DEPS)):
        return lib
    cmd = ([NVCC] + FLAGS + (["-DMONC_ADV_CHECKED=1"] if checked else [])
           + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + SOURCES)
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, checked="--checked" in sys.argv))
