"""In-tree build of the C-ABI library: nvcc -> paper_2606_02218_b200/libsagc.so (sm_100a only).

`python -m paper_2606_02218_b200.build` or `build()`; nvcc cross-compiles without a GPU.
Also writes the SASS listing used as evidence (profiles/) when asked.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsagc.so")
SOURCES = ["linear.cu", "tc_linear.cu", "attention.cu", "attention_noalloc.cu", "attention_tc.cu", "decode_step.cu", "elementwise.cu", "sampler.cu", "paging.cu", "groupstats.cu", "runtime.cu"]
HEADERS = ["common.cuh", "kernels.cuh", "tc_ptx.cuh", "attention_body.cuh", os.path.join("..", "..", "include", "sagc.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]
if os.environ.get("SAGC_PDL_EARLY"):
    NVCC_FLAGS += ["-DSAGC_PDL_EARLY"]
if os.environ.get("SAGC_ATT_TIMELINE"):     # clock64 timeline of the tcgen05 attention kernel (debug builds only)
    NVCC_FLAGS += ["-DSAGC_ATT_TIMELINE"]
if os.environ.get("SAGC_TRACE_BUILD"):       # in-kernel timeline (debug builds only)
    NVCC_FLAGS += ["-DSAGC_TRACE", "-rdc=true"]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = _nvcc()
    os.makedirs(OBJ, exist_ok=True)
    hdrs = [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS]
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        if force or _stale(o, [s] + hdrs):
            jobs.append((s, o))

    def run(job):
        s, o = job
        cmd = [nvcc] + NVCC_FLAGS + ["-c", s, "-o", o]
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        p = subprocess.run(cmd, capture_output=True, text=True)
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed for {s}:\n{p.stdout}\n{p.stderr}")
        return o

    if jobs:
        with ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
            list(ex.map(run, jobs))
    objs = [os.path.join(OBJ, s.replace(".cu", ".o")) for s in SOURCES]
    if force or jobs or _stale(LIB, objs):
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs
        p = subprocess.run(cmd, capture_output=True, text=True)
        if p.returncode != 0:
            raise RuntimeError(f"link failed:\n{p.stdout}\n{p.stderr}")
    return LIB


def sass_listing(out_path: str, pattern: str = "") -> None:
    """cuobjdump -sass of the built library (optionally only functions matching `pattern`)."""
    cmd = ["cuobjdump", "-sass", LIB]
    if pattern:
        cmd += ["-fun", pattern]
    p = subprocess.run(cmd, capture_output=True, text=True, check=True)
    with open(out_path, "w") as f:
        f.write(p.stdout)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
