"""Build libnm.so (the C-ABI library of include/nm.h) in-tree with nvcc for sm_100a.

    python -m paper_2411_11725_b200.build [--force]

Cross-compiles without a GPU.  The shared object lands next to this file so that it travels
with the repository snapshot to the GPU box.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnm.so")
CU = ["nm_api.cu", "nm_local.cu", "nm_node_col.cu", "nm_demag.cu", "nm_demag_fast.cu", "nm_demag_pipe.cu", "nm_tensor.cu",
      "nm_noalloc.cu"]
CPP = ["nm_newell_host.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _newer(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def build(force=False, verbose=False):
    """Compile every translation unit and link libnm.so; returns its path."""
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps.append(os.path.join(HERE, "..", "include", "nm.h"))
    deps.append(os.path.abspath(__file__))
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    if not force and not _newer(LIB, deps):
        return LIB
    objs = []
    procs = []
    for f in CU:
        o = os.path.join(objdir, f + ".o")
        objs.append(o)
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-c", os.path.join(CSRC, f), "-o", o]
        procs.append((cmd, subprocess.Popen(cmd)))
    for f in CPP:
        o = os.path.join(objdir, f + ".o")
        objs.append(o)
        cmd = ["g++", "-O2", "-std=gnu++17", "-fPIC", "-c", os.path.join(CSRC, f), "-o", o]
        procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("build failed: " + " ".join(cmd))
    tmp = LIB + ".%d.tmp" % os.getpid()
    cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs + ["-lquadmath", "-lpthread", "-lcudart"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
