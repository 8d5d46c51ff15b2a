"""Build libtf_b200.so (the C-ABI of include/tf.h) in-tree with nvcc for sm_100a.

    python -m paper_1806_10550_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtf_b200.so")
SOURCES = [os.path.join(CSRC, "tf_b200.cu")]
HEADERS = [os.path.join(CSRC, f) for f in ("tf_device.cuh", "tf_reduce.cuh", "tf_penta.cuh", "tf_async.cuh", "tf_bwd.cuh", "tf_tma.cuh", "tf_fwd.cuh", "tf_partition.cuh", "tf_topo.cuh", "tf_spectrum.cuh", "tf_blocks.cuh", "tf_control.cuh", "tf_pcr.cuh")] + \
          [os.path.join(os.path.dirname(HERE), "include", "tf.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v", "-ldl"]


def stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force=False, verbose=False):
    if not force and not stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, *NVCC_FLAGS, "-o", LIB, *SOURCES]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or r.returncode != 0:
        print(" ".join(cmd))
        print(r.stdout)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libtf_b200.so")
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="--verbose" in sys.argv or "-v" in sys.argv)
    print(LIB)
