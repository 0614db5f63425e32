"""Build the CUDA path into paper_2503_22139_b200/libgsvox.so (in-tree, sm_100a only).

nvcc cross-compiles without a GPU; the .so travels to the GPU box with the gpurun snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgsvox.so")
PROBE_LIB = os.path.join(HERE, "libgsvox_probe.so")      # bench-only ALU microbenchmarks (include/gsvox_probe.h)
SOURCES = ["gsvox_api.cu", "gsvox_host.cu", "gsvox_preprocess.cu", "gsvox_forward.cu", "gsvox_backward.cu",
           "gsvox_epilogue.cu", "gsvox_dvf.cu", "gsvox_warp.cu", "gsvox_project.cu", "gsvox_splat.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-O2,-Wall", "-shared", "-cudart", "static"]


def _deps():
    out = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    out.append(os.path.join(os.path.dirname(HERE), "include", "gsvox.h"))
    out.append(os.path.join(os.path.dirname(HERE), "include", "gsvox_probe.h"))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    fresh = lambda lib: os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in _deps())
    if not force and fresh(LIB) and fresh(PROBE_LIB):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    for lib, sources in ((LIB, SOURCES), (PROBE_LIB, ["gsvox_probe.cu"])):
        tmp = lib + ".tmp.%d" % os.getpid()
        cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp,
               *[os.path.join(CSRC, s) for s in sources]]
        subprocess.run(cmd, check=True)
        os.replace(tmp, lib)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
