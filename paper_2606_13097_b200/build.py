"""Builds libfcg.so (the C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_2606_13097_b200.build [--force]

Objects are cached under paper_2606_13097_b200/build/ and rebuilt when a source or header is
newer.  nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libfcg.so")

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cu"))


def _headers():
    hs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))]
    hs.append(os.path.join(ROOT, "include", "fcg.h"))
    return hs


# (nvcc splits -Xcompiler arguments at commas, so one flag per sanitizer)
SANITIZE_FLAGS = ["-Xcompiler", "-fsanitize=address", "-Xcompiler", "-fsanitize=undefined", "-Xcompiler", "-fno-omit-frame-pointer"]


def build(force: bool = False, verbose: bool = False, sanitize: bool = False) -> str:
    """sanitize=True: the HOST code of the library (planner, arena bookkeeping, blob packing) built with ASan + UBSan into
    libfcg_asan.so (objects under build_asan/).  Load it with FCG_LIBRARY=<path> and LD_PRELOAD=$(gcc -print-file-name=libasan.so),
    ASAN_OPTIONS=protect_shadow_gap=0 (CUDA maps memory where ASan keeps its shadow gap); see profiles/r03_sanitizer.md."""
    global BUILD, LIB
    if sanitize:
        saved = (BUILD, LIB)
        BUILD, LIB = os.path.join(HERE, "build_asan"), os.path.join(HERE, "libfcg_asan.so")
        NVCC_FLAGS.extend(SANITIZE_FLAGS)
        try:
            return _build(force, verbose, SANITIZE_FLAGS)
        finally:
            BUILD, LIB = saved
            del NVCC_FLAGS[-len(SANITIZE_FLAGS):]
    return _build(force, verbose, [])


def _build(force: bool, verbose: bool, link_flags) -> str:
    os.makedirs(BUILD, exist_ok=True)
    nvcc = _nvcc()
    newest_header = max(os.path.getmtime(h) for h in _headers())
    jobs = []
    objs = []
    for src in _sources():
        obj = os.path.join(BUILD, os.path.basename(src)[:-3] + ".o")
        objs.append(obj)
        stale = force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), newest_header)
        if stale:
            jobs.append((src, obj))

    def compile_one(job):
        src, obj = job
        cmd = [nvcc, *NVCC_FLAGS, "-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log = obj[:-2] + ".log"
        with open(log, "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            print(r.stderr, file=sys.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=max(1, min(8, len(jobs)))) as ex:
        list(ex.map(compile_one, jobs))
    if jobs or force or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        cmd = [nvcc, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static", *link_flags]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    path = build(force="--force" in sys.argv, verbose="-v" in sys.argv, sanitize="--sanitize" in sys.argv)
    print(path)
