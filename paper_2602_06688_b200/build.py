"""Build libpyr.so in-tree with nvcc for sm_100a (no torch headers involved).

csrc/pyr.cu holds the plan and the C ABI of the pyramid path, csrc/sh.cu the Shack-Hartmann path,
csrc/chain.cu the steps either side of the sensor (include/chain.h);
csrc/pyr_inst.cu is compiled once per FFT size
(-DPYR_INST_N=<N>), in parallel, so that the template instantiations do not serialise."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libpyr.so")
SIZES = (16, 32, 64, 128, 256, 512, 1024, 2048)
DEPS = [os.path.join(CSRC, f) for f in ("pyr.cu", "pyr_inst.cu", "pyr_kernels.cuh", "pyr_fft.cuh", "sh.cu", "chain.cu")] + [
    os.path.join(HERE, "..", "include", "pyr.h"), os.path.join(HERE, "..", "include", "sh.h"),
    os.path.join(HERE, "..", "include", "chain.h")]

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
CFLAGS = ARCH + ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in DEPS)


def _compile(job):
    src, obj, extra, verbose = job
    cmd = [nvcc()] + CFLAGS + (["-Xptxas", "-v"] if verbose else []) + extra + ["-c", "-o", obj, src]
    r = subprocess.run(cmd, capture_output=True, text=True)
    return r.returncode, r.stdout + r.stderr, " ".join(cmd)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu -> libpyr.so (cross-compiles without a GPU)."""
    if not (force or needs_build()):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    tag = ".%d" % os.getpid()
    jobs = [(os.path.join(CSRC, "pyr.cu"), os.path.join(OBJ, "pyr%s.o" % tag), [], verbose),
            (os.path.join(CSRC, "sh.cu"), os.path.join(OBJ, "sh%s.o" % tag), [], verbose),
            (os.path.join(CSRC, "chain.cu"), os.path.join(OBJ, "chain%s.o" % tag), [], verbose)]
    for n in sorted(SIZES, reverse=True):     # longest first
        jobs.append((os.path.join(CSRC, "pyr_inst.cu"), os.path.join(OBJ, "inst_%d%s.o" % (n, tag)),
                     ["-DPYR_INST_N=%d" % n], verbose))
    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        results = list(ex.map(_compile, jobs))
    for rc, out, cmd in results:
        if verbose or rc:
            sys.stderr.write(out)
        if rc:
            raise RuntimeError("nvcc failed: " + cmd)
    tmp = LIB + ".tmp" + tag
    objs = [j[1] for j in jobs]
    subprocess.check_call([nvcc()] + ARCH + ["-shared", "-cudart", "static", "-o", tmp] + objs)
    os.replace(tmp, LIB)
    for o in objs:
        os.remove(o)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
