"""Builds paper_2606_28372_b200/libcao.so (hand-written CUDA for sm_100a + the C ABI of include/cao.h) in-tree.

Objects are compiled in parallel (one nvcc process each) and linked into one shared library:
  cao_space.cu, cao_runs.cu, and cao_gen_algo.cu four times (-DCAO_GEN_ALGO=0..3: the fused generation kernel of
  DE / PSO / Firefly / GA)."""
from __future__ import annotations
import glob
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libcao.so")
# --fmad=false: no FMA contraction anywhere (the fp32 PSO / Firefly updates must match the oracle bit for bit);
# IEEE division / sqrt, no flush-to-zero.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
              "-Xcompiler", "-fPIC"]


def units():
    """(source, object name, extra flags)"""
    u = []
    for src in sorted(glob.glob(os.path.join(CSRC, "*.cu"))):
        base = os.path.splitext(os.path.basename(src))[0]
        if base == "cao_gen_algo":
            u += [(src, f"cao_gen_algo{a}.o", [f"-DCAO_GEN_ALGO={a}"]) for a in range(4)]
        else:
            u.append((src, base + ".o", []))
    return u


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = glob.glob(os.path.join(CSRC, "*")) + [os.path.join(HERE, "..", "include", "cao.h"), __file__]
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        os.makedirs(OBJ, exist_ok=True)
        extra = (["-Xptxas", "-v"] if verbose else []) + os.environ.get("CAO_NVCC_EXTRA", "").split()

        def compile_one(u):
            src, obj, flags = u
            out = os.path.join(OBJ, obj)
            subprocess.check_call([nvcc, *NVCC_FLAGS, *extra, *flags, "-c", src, "-o", out])
            return out

        with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
            objs = list(ex.map(compile_one, units()))
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static",
                               *objs, "-o", tmp])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
