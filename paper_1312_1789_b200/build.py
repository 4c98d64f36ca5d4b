"""nvcc build of csrc/ into csrc/libnbody.so for sm_100a (in-tree, so the .so travels to the GPU box).

Two flag sets (R12): the bit-exact fp64 kernels are compiled with -fmad=false; the force kernel keeps
FMA contraction and flushes fp32 denormals (-ftz=true).  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libnbody.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
COMMON = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
          "-I", os.path.join(ROOT, "include"), "-I", CSRC]
UNITS = {
    "nbody_exact.cu": ["-fmad=false", "-prec-div=true", "-prec-sqrt=true"],
    "nbody_force.cu": ["-ftz=true"],
    "nbody_probe.cu": [],
}
HEADERS = [os.path.join(CSRC, "nbody_internal.h"), os.path.join(CSRC, "nbody_exact.cuh"), os.path.join(ROOT, "include", "nbody.h"),
           os.path.join(ROOT, "include", "nbody_bench.h")]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    objs = []
    relink = force
    for src, flags in UNITS.items():
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", ".o"))
        if force or _stale(o, [s, *HEADERS, os.path.abspath(__file__)]):
            cmd = [NVCC, *COMMON, *flags, "-c", s, "-o", o]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
                print(" ".join(cmd), file=sys.stderr)
            subprocess.check_call(cmd)
            relink = True
        objs.append(o)
    if relink or _stale(LIB, objs):
        tmp = LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call([NVCC, "-shared", "-o", tmp, *objs, "-lcudart_static", "-lpthread", "-ldl", "-lrt"])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
