"""Build libhmc.so (the C-ABI CUDA library, include/hmc.h) in-tree with nvcc for sm_100a.

    python -m paper_1206_5878_b200.build [--force]

nvcc cross-compiles without a GPU.  Flags that matter:
  -gencode arch=compute_100a,code=sm_100a   B200 only, no other target
  -fmad=false                               no FMA contraction: fp64 results are bit-comparable (R2)
  -lineinfo                                 so ncu's source page maps to these files
  -cudart static                            the .so loads on a box without libcudart on the path
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhmc.so")
SOURCES = ["hmc_api.cu", "hmc_sort.cu", "hmc_sort_fast.cu", "hmc_potential.cu", "hmc_orbit.cu", "hmc_diag.cu", "hmc_relax.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-cudart", "static",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


# "product" is the library; "tmax3" is a TEST-ONLY build of the same sources with the cap on rejection trials
# lowered to 3, so that the GPU tests reach S4's exhaustion path (draw_exhaustive, MAXTRIES) and compare it
# with the oracle built the same way (oracle/: -DT_MAX=3u).  Nothing but tests loads it.
# "pairs" is a TEST-ONLY build in which S3's exact search runs by lane pairs at every N (the product takes that
# path from N = 2^25 on, where the node table is far beyond the TLB's reach), so that small parity cases reach it.
VARIANTS = {
    "product": ("libhmc.so", []),
    "tmax3": ("libhmc_tmax3.so", ["-DHMC_T_MAX=3u"]),
    "pairs": ("libhmc_pairs.so", ["-DHMC_S3_PAIRS_MIN_N=1"]),
}


def lib_path(variant: str = "product") -> str:
    return os.path.join(HERE, VARIANTS[variant][0])


def _stale(lib: str) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh"))]
    deps += [os.path.join(ROOT, "include", "hmc.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, variant: str = "product") -> str:
    LIB = lib_path(variant)
    defines = VARIANTS[variant][1]
    if not (force or _stale(LIB)):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    suffix = ".o" if variant == "product" else ".%s.o" % variant
    for src in SOURCES:
        obj = os.path.join(CSRC, src[:-3] + suffix)
        cmd = [nvcc, *NVCC_FLAGS, *defines, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode:
            sys.stderr.write(out)
        if p.returncode:
            raise RuntimeError("nvcc failed on %s" % src)
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.run([nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a",
                    "-Xcompiler", "-fPIC", *objs, "-o", tmp], check=True)
    os.replace(tmp, LIB)
    return LIB


def build_all(force: bool = False, verbose: bool = False):
    return [build(force, verbose, v) for v in VARIANTS]


if __name__ == "__main__":
    for path in build_all(force="--force" in sys.argv, verbose="-v" in sys.argv):
        print(path)
