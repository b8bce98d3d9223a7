"""Build libdftb200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdftb200.so")
# (source, object, extra flags): fft2.cu is compiled in four parts, each instantiating a part of the radix pairs
SOURCES = [("plan.cu", "plan.o", []), ("sphere.cu", "sphere.o", []), ("projtab.cu", "projtab.o", []), ("fft.cu", "fft.o", []),
           ("fft_small.cu", "fft_small.o", []), ("fft_small2.cu", "fft_small2.o", []),
           ("fft2.cu", "fft2_p0.o", ["-DFFT2_PART=0"]), ("fft2.cu", "fft2_p1.o", ["-DFFT2_PART=1"]),
           ("fft2.cu", "fft2_p2.o", ["-DFFT2_PART=2"]), ("fft2.cu", "fft2_p3.o", ["-DFFT2_PART=3"]), ("nonlocal.cu", "nonlocal.o", []),
           ("gamma.cu", "gamma.o", []), ("spinor.cu", "spinor.o", []), ("noalloc.cu", "noalloc.o", [])]
HEADERS = [os.path.join(CSRC, "internal.h"), os.path.join(CSRC, "fft_codelets.cuh"), os.path.join(CSRC, "ptx.cuh"), os.path.join(CSRC, "fft_tw_literals.cuh"), os.path.join(CSRC, "fft_small.cuh"), os.path.join(CSRC, "nonlocal_strassen.inc"), os.path.join(HERE, "..", "include", "dft.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC,-ffp-contract=off", "-Xptxas", "-v"]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile every CUDA source and link the shared library; returns its path.  The whole build holds an exclusive
    file lock, so the ranks of a multi-GPU launch on a fresh box do not compile the same objects at the same time
    (the first one builds, the others find everything up to date)."""
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            return _build_locked(force, verbose)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(force, verbose):
    objs, jobs = [], []
    for s, o, extra in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(CSRC, o)
        objs.append(obj)
        if force or _stale(obj, [src] + HEADERS):
            jobs.append([NVCC] + FLAGS + extra + ["-c", src, "-o", obj])

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
