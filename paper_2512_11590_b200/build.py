"""Build paper_2512_11590_b200/libhprmat.so from csrc/*.cu (the product) and libhprmat_bench.so from bench_csrc/*.cu (bench.py's
peak probe, never loaded by the product) with nvcc for sm_100a (in-tree, no JIT cache).

    python -m paper_2512_11590_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library links the static CUDA runtime and nothing else (no cuBLAS/cuSOLVER).
"""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libhprmat.so")
BENCH_LIB = os.path.join(HERE, "libhprmat_bench.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
         "--expt-relaxed-constexpr"]


def _deps_mtime():
    hdrs = glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(HERE, "..", "include", "*.h"))
    return max(os.path.getmtime(h) for h in hdrs)


def build(force: bool = False, verbose: bool = False) -> str:
    _build_one(os.path.join(HERE, "bench_csrc"), "bench_", BENCH_LIB, force, verbose)
    return _build_one(CSRC, "", LIB, force, verbose)


def _build_one(src_dir: str, prefix: str, LIB: str, force: bool, verbose: bool) -> str:
    srcs = sorted(glob.glob(os.path.join(src_dir, "*.cu")))
    os.makedirs(OBJ, exist_ok=True)
    hdr_m = _deps_mtime()
    jobs = []
    obj_of = lambda s: os.path.join(OBJ, prefix + os.path.basename(s)[:-3] + ".o")
    for s in srcs:
        o = obj_of(s)
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr_m):
            jobs.append((s, o))

    def cc(job):
        s, o = job
        cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {s}:\n{r.stdout}\n{r.stderr}")
        return r.stderr

    with ThreadPoolExecutor(max_workers=min(8, max(1, len(jobs)))) as ex:
        for log in ex.map(cc, jobs):
            if verbose and log:
                print(log, file=sys.stderr)
    objs = [obj_of(s) for s in srcs]
    if jobs or force or not os.path.exists(LIB):
        cmd = [NVCC, "-shared", "-o", LIB + ".tmp"] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
