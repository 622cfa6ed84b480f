"""Build libtaiga.so (hand-written sm_100a CUDA behind the C ABI of include/taiga.h), in-tree.

Every csrc/*.cu is compiled to its own object (in parallel, only when it or a header changed) and the
objects are linked into paper_2506_15812_b200/libtaiga.so."""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libtaiga.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def build(force: bool = False, verbose: bool = False) -> str:
    headers = glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + [
        os.path.join(os.path.dirname(HERE), "include", "taiga.h"), os.path.abspath(__file__)]
    hdr_time = max(os.path.getmtime(h) for h in headers)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max([hdr_time] + [os.path.getmtime(s) for s in sources()]):
        return LIB                             # up to date (e.g. the library shipped to the GPU box without its objects)
    os.makedirs(OBJ, exist_ok=True)
    jobs, objs = [], []
    for src in sources():
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_time):
            jobs.append([NVCC] + FLAGS + (["-Xptxas=-v"] if verbose else []) + ["-c", src, "-o", obj])
    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            for r in ex.map(lambda c: subprocess.run(c, capture_output=not verbose, text=True), jobs):
                if r.returncode != 0:
                    sys.stderr.write((r.stdout or "") + (r.stderr or ""))
                    raise subprocess.CalledProcessError(r.returncode, r.args)
    if jobs or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        subprocess.run([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
