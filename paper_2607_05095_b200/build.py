"""Builds libfasttg.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2607_05095_b200.build [--force]

One nvcc process per translation unit, run in parallel, then one link step.  Objects live in
``csrc/build/`` (git-ignored); the shared library is ``paper_2607_05095_b200/libfasttg.so``.
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libfasttg.so")
SOURCES = ["api.cu", "block.cu", "fused_fwd.cu", "fused_bwd.cu", "fused_edge.cu", "unfused.cu", "softmax.cu", "cache.cu", "sampler.cu", "probe_bulk.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-fvisibility=hidden", "-I", os.path.join(ROOT, "include"), "-I", CSRC]
# No --use_fast_math: measured in round 2, it changed neither the errors nor the times; the only approximate
# instruction on the path is the explicit ex2.approx of the softmax.  TG_FAST_MATH=1 re-enables it for comparison.
if os.environ.get("TG_FAST_MATH", "0") == "1":
    NVCC_FLAGS.insert(5, "--use_fast_math")
# extra nvcc flags for experiments (e.g. TG_NVCC_EXTRA="-DTG_CHUNK_MAX_EDGES=512"); part of the build stamp
NVCC_FLAGS += os.environ.get("TG_NVCC_EXTRA", "").split()


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found; libfasttg cannot be built")


def _stamp() -> str:
    h = hashlib.sha256()
    h.update(" ".join(NVCC_FLAGS).replace(ROOT, "<root>").encode())   # independent of where the checkout lives
    names = sorted(os.listdir(CSRC))
    for n in names:
        p = os.path.join(CSRC, n)
        if os.path.isfile(p) and n.endswith((".cu", ".cuh", ".h")):
            h.update(n.encode())
            h.update(open(p, "rb").read())
    for n in sorted(os.listdir(os.path.join(ROOT, "include"))):
        h.update(open(os.path.join(ROOT, "include", n), "rb").read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    stamp_file = os.path.join(OBJ, "stamp.txt")
    stamp = _stamp()
    if not force and os.path.exists(LIB) and os.path.exists(stamp_file) and open(stamp_file).read() == stamp:
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()

    def compile_one(src):
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    r = subprocess.run([nvcc, "-shared", "-o", LIB, *objs, "-lcudart"], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    with open(stamp_file, "w") as f:
        f.write(stamp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
