"""Build paper_1908_01949_b200/libcdc_seedscan.so (the C-ABI library of include/cdc_seedscan.h) with nvcc
for sm_100a, in-tree.  best.cu, refine.cu and peel.cu are compiled with -fmad=false (IEEE fp64 without contraction, C11)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcdc_seedscan.so")
OBJ = os.path.join(HERE, "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", *ARCH]
SOURCES = {                      # file -> extra flags
    "abi.cu": [], "abi_events.cu": [], "abi_scan.cu": [], "abi_e2e.cu": [],
    "events.cu": [], "hough.cu": [], "hough_noalloc.cu": [], "scan.cu": ["-Xptxas", "-v"], "scan_pair.cu": ["-Xptxas", "-v"], "scan_refill.cu": ["-Xptxas", "-v"], "scan_adaptive.cu": [], "peak.cu": [],
    "best.cu": ["-fmad=false"], "refine.cu": ["-fmad=false"], "abi_refine.cu": [], "quality.cu": [], "paper_v1.cu": [], "paper_v2.cu": [],
    "peel.cu": ["-fmad=false"], "abi_peel.cu": [],
}
HEADERS = [os.path.join(CSRC, "paper_common.cuh"), os.path.join(CSRC, "peel.cuh"), os.path.join(CSRC, "refine.cuh"), os.path.join(CSRC, "cdc_internal.cuh"), os.path.join(CSRC, "eval64.cuh"), os.path.join(CSRC, "scan_common.cuh"), os.path.join(CSRC, "scan_args.cuh"), os.path.join(CSRC, "pair_math.cuh"), os.path.join(CSRC, "scan_one.cuh"), os.path.join(HERE, "..", "include", "cdc_seedscan.h")]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    objs = []
    for src, extra in SOURCES.items():
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s, *HEADERS, __file__]):
            cmd = [NVCC, *COMMON, *extra, "-c", s, "-o", o]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if verbose or r.returncode != 0:
                sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            if r.returncode != 0:
                raise RuntimeError("nvcc failed on " + src)
    if force or _stale(LIB, objs):
        cmd = [NVCC, "-shared", *ARCH, "-o", LIB, *objs]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
