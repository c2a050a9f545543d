"""In-tree build of libnd_moc.so (nvcc for sm_100a + g++ for the host ray tracer).

    python -m paper_2607_01591_b200._build [--force]

The host tracer is compiled by g++ with -ffp-contract=off (rule R-T/R-W: bit-exact FP64 geometry); the CUDA
translation unit by nvcc with -gencode arch=compute_100a,code=sm_100a -lineinfo.  nvcc cross-compiles without a GPU.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libnd_moc.so")
BUILD = os.path.join(HERE, "build")

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC", "-Xcompiler", "-fopenmp",
              "-Xptxas", "-v", "--expt-relaxed-constexpr"]
GXX_FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-fPIC", "-Wall"]

CU_SOURCES = ["nd_api.cu", "nd_trace_device.cu", "nd_microbench.cu", "nd_swath_device.cu", "nd_noalloc.cu"]
CXX_SOURCES = ["nd_tracks.cpp", "nd_swath.cpp", "nd_cmfd_host.cpp"]


def _nvcc():
    return shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"


def source_id() -> str:
    """Short hash of every source the library is built from (csrc/ and include/): nd_build_id() returns it, bench.py
    prints it, and ncu captures under profiles/ are named after it, so a profile of another build is never quoted."""
    import hashlib
    h = hashlib.sha256()
    for d in (CSRC, INCLUDE):
        for f in sorted(os.listdir(d)):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:12]


def _newest_source_mtime():
    m = 0.0
    for d in (CSRC, INCLUDE):
        for f in os.listdir(d):
            m = max(m, os.path.getmtime(os.path.join(d, f)))
    return m


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source_mtime():
        return LIB
    os.makedirs(BUILD, exist_ok=True)
    objs = []
    build_id = '-DND_BUILD_ID="%s"' % source_id()
    for src in CU_SOURCES:
        obj = os.path.join(BUILD, src + ".o")
        cmd = [_nvcc(), *NVCC_FLAGS, build_id, "-I", INCLUDE, "-I", CSRC, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        with open(os.path.join(BUILD, src + ".ptxas.log"), "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
        if verbose:
            print(r.stderr)
        objs.append(obj)
    for src in CXX_SOURCES:
        obj = os.path.join(BUILD, src + ".o")
        cmd = ["g++", *GXX_FLAGS, "-I", INCLUDE, "-I", CSRC, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("g++ failed:\n" + r.stdout + r.stderr)
        objs.append(obj)
    cmd = [_nvcc(), "-shared", "-o", LIB, *objs, "-Xcompiler", "-fopenmp", "-lgomp"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
