"""Build libdsk.so (hand-written CUDA for sm_100a) in-tree:  python -m paper_1407_2600_b200.build

nvcc cross-compiles without a GPU.  The .so stays next to this file (git-ignored, travels with gpurun).
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["dsk_api.cu", "keysort.cu", "tree.cu", "upward.cu", "walk.cu", "force.cu", "m2p.cu", "farfield.cu", "background.cu", "kdk.cu", "peak.cu"]
HEADERS = [os.path.join(CSRC, "dsk_internal.cuh"), os.path.join(CSRC, "force_task.cuh"), os.path.join(CSRC, "cube_series.inc"), os.path.join(HERE, "..", "include", "dsk.h")]
LIB = os.path.join(HERE, "libdsk.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr", "-ftz=true", "-prec-div=true", "-prec-sqrt=true"]
FLAGS += os.environ.get("DSK_EXTRA_NVCC_FLAGS", "").split()      # tuning sweeps only (e.g. -DDSK_NLEAF=32)


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    objs, jobs = [], []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(HERE, "build", s.replace(".cu", ".o"))
        objs.append(obj)
        if force or _stale(obj, [src] + HEADERS):
            cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, r

    with ThreadPoolExecutor(max_workers=8) as ex:
        for cmd, r in ex.map(run, jobs):
            if verbose or r.returncode:
                sys.stderr.write(" ".join(cmd[-3:]) + "\n" + r.stdout + r.stderr)
            if r.returncode:
                raise RuntimeError("nvcc failed: " + cmd[-3])
    if jobs or not os.path.exists(LIB):
        subprocess.run([NVCC, "-shared", "-o", LIB] + objs + ["-lcudart"], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
