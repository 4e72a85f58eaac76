"""Build libpm.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2211_09815_b200.build [--force] [-v] [--debug]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the tree to the GPU box.
--debug builds libpm_debug.so with -DPM_DEBUG: the probe build (work-skipping knobs of the CIC kernels, per-stage
high-precision variants of F(x) for the precision A/B of DESIGN.md section 7).  Nothing in the package, the tests or
bench.py loads it unless PM_LIB names it explicitly.
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpm.so")
LIB_DEBUG = os.path.join(HERE, "libpm_debug.so")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.inc")) + \
        glob.glob(os.path.join(ROOT, "include", "*.h"))


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _deps())


def build(force=False, verbose=False, debug=False):
    lib = LIB_DEBUG if debug else LIB
    if not force and not debug and not needs_build():
        return lib
    nvcc = os.path.join(CUDA_HOME, "bin", "nvcc")
    # one nvcc process per source file, in parallel (the CIC and FFT files take a minute each), then the link
    objdir = os.path.join(HERE, "build", "dbg" if debug else "rel")
    os.makedirs(objdir, exist_ok=True)
    flags = ["-Xcompiler", "-fPIC", "-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
             "-I", os.path.join(ROOT, "include"), "-I", CSRC]
    if debug:
        flags.append("-DPM_DEBUG")
    if verbose:
        flags.insert(0, "-Xptxas=-v")
    newest_hdr = max(os.path.getmtime(f) for f in _deps() if not f.endswith(".cu"))
    procs, objs = [], []
    for src in sources():
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        objs.append(obj)
        if not force and os.path.exists(obj) and os.path.getmtime(obj) > max(os.path.getmtime(src), newest_hdr):
            continue
        procs.append((src, subprocess.Popen([nvcc, "-c"] + flags + ["-o", obj, src])))
    for src, pr in procs:
        if pr.wait() != 0:
            raise subprocess.CalledProcessError(pr.returncode, f"nvcc -c {src}")
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib] + objs + ["-lcufft", "-Xlinker", "-rpath," + os.path.join(CUDA_HOME, "lib64")],
                   check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, debug="--debug" in sys.argv))
