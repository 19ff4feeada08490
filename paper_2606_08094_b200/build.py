"""Builds paper_2606_08094_b200/libvlaternary.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_08094_b200.build [--force] [--verbose]
"""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libvlaternary.so")
SOURCES = ["api.cu", "pack.cu", "act_quant.cu", "gemm_small.cu", "gemm_large.cu", "gemm_program.cu", "gemm_lprog.cu", "api_program.cu", "attention.cu", "no_alloc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "--threads", "0"]


STAMP = SO + ".srchash"


def source_hash():
    """sha256 over csrc/ and the public header: what the .so was built from (mtimes do not survive a copy)."""
    paths = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC))
    paths.append(os.path.join(os.path.dirname(HERE), "include", "vla_ternary.h"))
    h = hashlib.sha256()
    for p in paths:
        h.update(os.path.basename(p).encode())
        h.update(open(p, "rb").read())
    return h.hexdigest()


def is_current():
    return os.path.exists(SO) and os.path.exists(STAMP) and open(STAMP).read().strip() == source_hash()


def build(force=False, verbose=False):
    if not force and is_current():
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = SO + ".tmp%d" % os.getpid()
    cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []),
           *[os.path.join(CSRC, s) for s in SOURCES], "-o", tmp]
    subprocess.run(cmd, check=True)
    os.replace(tmp, SO)
    with open(STAMP, "w") as f:
        f.write(source_hash() + "\n")
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
