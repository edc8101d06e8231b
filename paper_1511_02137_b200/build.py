"""Build libhydro.so (the C-ABI CUDA library of include/hydro.h) in-tree for sm_100a.

    python -m paper_1511_02137_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhydro.so")
SOURCES = [os.path.join(CSRC, "hydro.cu"), os.path.join(CSRC, "hydro_noalloc.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "hydro_kernels.cuh"), os.path.join(CSRC, "hydro_sweep_ring.cuh"), os.path.join(CSRC, "hydro_lowup.cuh"),
                  os.path.join(os.path.dirname(HERE), "include", "hydro.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--fmad=true",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v", "-lcudart"]


def source_sha():
    """sha256 (first 16 hex digits) of the CUDA sources + the C header: the identity of the kernels a profile was taken at."""
    import hashlib
    h = hashlib.sha256()
    for d in sorted(DEPS):
        with open(d, "rb") as f:
            h.update(os.path.basename(d).encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = [nvcc()] + NVCC_FLAGS + os.environ.get("HYDRO_NVCC_EXTRA", "").split() + SOURCES + ["-o", tmp]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)               # git-ignored: ptxas -v register / spill report
    with open(os.path.join(HERE, "build", "libhydro.ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
