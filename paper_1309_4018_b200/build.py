"""Build libpygbe.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1309_4018_b200.build [--force]

One object per translation unit, compiled in parallel: pygbe.cu (ABI + all kernels except M2P) and
m2p_inst.cu once per expansion order P = 1..12 (the fully unrolled Taylor recurrences).
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libpygbe.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fopenmp", "-Xptxas", "-v"]      # OpenMP: host loops of create only
FLAGS += os.environ.get("PYGBE_CFLAGS", "").split()      # e.g. -DPYGBE_TG=64 for tuning experiments
PMAX = 12


def _newest_source():
    t = 0.0
    for f in os.listdir(CSRC):
        t = max(t, os.path.getmtime(os.path.join(CSRC, f)))
    t = max(t, os.path.getmtime(os.path.join(HERE, "..", "include", "pygbe.h")))
    return t


def _compile(job):
    src, obj, extra = job
    if src.endswith("m2p_inst.cu"):
        deps = [src, os.path.join(CSRC, "m2p.cuh"), os.path.join(CSRC, "mathx.cuh")]
    else:
        deps = [src] + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".inc"))]
        deps.append(os.path.join(HERE, "..", "include", "pygbe.h"))
    if os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(d) for d in deps):
        return obj, ""
    cmd = [NVCC] + FLAGS + extra + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s" % (" ".join(cmd), r.stderr[-4000:]))
    with open(obj + ".log", "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stderr)
    return obj, r.stderr


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    if force:
        for f in os.listdir(OBJ):
            os.remove(os.path.join(OBJ, f))
    jobs = [(os.path.join(CSRC, "pygbe.cu"), os.path.join(OBJ, "pygbe.o"), []),
            (os.path.join(CSRC, "noalloc.cu"), os.path.join(OBJ, "noalloc.o"), [])]
    # the largest orders first: they take longest
    # PYGBE_FAST_BUILD=<n>: development shortcut, orders above n are compiled as stubs that refuse to run
    fast = int(os.environ.get("PYGBE_FAST_BUILD", "0"))
    for p in range(PMAX, 0, -1):
        extra = ["-DM2P_P=%d" % p]
        name = "m2p_%d.o" % p
        if fast and p > fast:
            extra.append("-DM2P_STUB")
            name = "m2p_%d_stub.o" % p
        jobs.append((os.path.join(CSRC, "m2p_inst.cu"), os.path.join(OBJ, name), extra))
    with ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        objs = [o for o, _ in ex.map(_compile, jobs)]
    if (not os.path.exists(LIB)) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fopenmp", "-o", LIB] + objs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed: %s\n%s" % (" ".join(cmd), r.stderr[-4000:]))
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
