"""Build libdmuon.so in-tree with nvcc for sm_100a (no GPU needed: nvcc cross-compiles).

    python -m paper_2606_27153_b200.build [--force]
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libdmuon.so")
SOURCES = ["api.cu", "planner.cu", "assign.cu", "elementwise.cu", "gemm_sm100.cu", "ns_small_sm100.cu", "gemm_check.cu"]
HEADERS = ["common.h", "planner.h", "umma.cuh", "epilogue.cuh", os.path.join("..", "..", "include", "dmuon.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-fvisibility=hidden", "-diag-suppress", "177"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build_id() -> str:
    """Hash of every source and header of the library: the key under which tuned tile configurations are cached, so
    that a new build never trusts an older build's timings (PAPER.md:184 persistent kernel cache)."""
    h = hashlib.sha1()
    for name in sorted(SOURCES) + sorted(HEADERS):
        with open(os.path.normpath(os.path.join(CSRC, name)), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:12]


def build_library(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    os.makedirs(OBJ, exist_ok=True)
    headers = [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS]
    nvcc = _nvcc()
    jobs = []
    bid = build_id()
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        carries_id = src == "planner.cu"
        id_file = o + ".id"       # the id compiled into planner.o: ANY source change makes that object stale
        if carries_id and os.path.exists(o) and (not os.path.exists(id_file) or open(id_file).read().strip() != bid):
            os.remove(o)
        if force or _stale(o, [s] + headers):
            defs = [f'-DDMUON_BUILD_ID="{bid}"'] if carries_id else []
            if carries_id:
                with open(id_file, "w") as f:
                    f.write(bid)
            jobs.append([nvcc] + NVCC_FLAGS + list(extra_flags) + defs + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr

    with ThreadPoolExecutor(max_workers=max(1, min(len(jobs), os.cpu_count() or 1))) as ex:
        for out in ex.map(run, jobs):
            if verbose and out:
                print(out)
    objs = [os.path.join(OBJ, s.replace(".cu", ".o")) for s in SOURCES]
    if force or jobs or _stale(LIB, objs):
        run([nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
