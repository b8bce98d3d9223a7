"""Build libdftb200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdftb200.so")
SOURCES = ["plan.cu", "sphere.cu", "projtab.cu", "fft.cu", "fft2.cu", "nonlocal.cu"]
HEADERS = [os.path.join(CSRC, "internal.h"), os.path.join(CSRC, "fft_codelets.cuh"), os.path.join(CSRC, "ptx.cuh"), os.path.join(HERE, "..", "include", "dft.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC,-ffp-contract=off", "-Xptxas", "-v"]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile every CUDA source and link the shared library; returns its path."""
    objs, jobs = [], []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(CSRC, s[:-3] + ".o")
        objs.append(obj)
        if force or _stale(obj, [src] + HEADERS):
            jobs.append([NVCC] + FLAGS + ["-c", src, "-o", obj])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        return r.stderr

    logs = []
    if jobs:
        with ThreadPoolExecutor(len(jobs)) as ex:
            logs = list(ex.map(run, jobs))
    if jobs or force or _stale(LIB, objs):
        tmp = LIB + ".tmp%d" % os.getpid()
        run([NVCC, "-shared", "-o", tmp] + objs)
        os.replace(tmp, LIB)
    return LIB, "".join(logs)


if __name__ == "__main__":
    lib, log = build(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(lib)
