"""Build libbq.so (the C-ABI library of include/bq.h) with nvcc for sm_100a, in-tree.

    python -m paper_2111_04457_b200.build [--force]

One nvcc invocation per translation unit (run in parallel), then one link step.  The built .so is
git-ignored but travels to the GPU box with the gpurun snapshot.  A stamp file holding the hash of all
sources makes rebuilds a no-op.
"""
from __future__ import annotations

import concurrent.futures
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
LIB = os.path.join(HERE, "libbq.so")
STAMP = LIB + ".stamp"
OBJDIR = os.path.join(HERE, "build")

UNITS = ["lattice.cu", "hop.cu", "hop_inst_fp64_18.cu", "hop_inst_fp64_12.cu", "hop_inst_fp32_18.cu", "hop_inst_fp32_12.cu",
         "hop_inst_half_18.cu", "hop_inst_half_12.cu", "clover.cu", "blas.cu", "solve.cu", "bench_hooks.cu", "dd.cu", "noalloc.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "--extended-lambda", "-Xcompiler", "-fPIC", "-I", INCLUDE, "-I", CSRC,
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _source_hash() -> str:
    h = hashlib.sha256()
    names = sorted(os.listdir(CSRC)) + ["../../include/bq.h", "../../include/bq_test.h"]
    for n in names:
        p = os.path.join(CSRC, n)
        if os.path.isfile(p):
            h.update(n.encode())
            with open(p, "rb") as f:
                h.update(f.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib_path: str | None = None) -> str:
    """Default: the in-tree libbq.so.  extra_flags / lib_path build a tuning variant (e.g. -DHOP_BLOCK=64) elsewhere."""
    variant = lib_path is not None
    LIB = lib_path or globals()["LIB"]
    STAMP = LIB + ".stamp"
    OBJDIR = os.path.join(os.path.dirname(LIB), "build_" + os.path.basename(LIB)) if variant else globals()["OBJDIR"]
    h = _source_hash() + " ".join(extra_flags)
    if not force and os.path.exists(LIB) and os.path.exists(STAMP):
        with open(STAMP) as f:
            if f.read().strip() == h:
                return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    nvcc = _nvcc()

    def compile_one(unit: str) -> str:
        obj = os.path.join(OBJDIR, unit.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + list(extra_flags) + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, unit), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {unit}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    with concurrent.futures.ThreadPoolExecutor(max_workers=len(UNITS)) as ex:
        objs = list(ex.map(compile_one, UNITS))
    cmd = [nvcc, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    with open(STAMP, "w") as f:
        f.write(h)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
