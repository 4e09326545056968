"""Build libtdde.so in-tree with nvcc for sm_100a (no torch extension machinery: the library is a plain C ABI).

    python -m paper_2512_21697_b200.build [--force] [--verbose]

Each .cu is compiled to an object under csrc/build/ (git-ignored) and linked into
paper_2512_21697_b200/libtdde.so.  Objects are rebuilt only when a source or header is newer.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
INCLUDE = os.path.join(ROOT, "include")
OUT = os.environ.get("TDDE_LIB_OUT", os.path.join(HERE, "libtdde.so"))      # overrides: build-variant experiments
EXTRA = os.environ.get("TDDE_NVCC_FLAGS", "").split()
SOURCES = ["tdde_apply.cu", "tdde_apply_mma.cu", "tdde_apply_block2.cu", "tdde_apply_sparse.cu", "tdde_vec.cu", "tdde_precond.cu", "tdde_partition.cu", "tdde_create.cu", "tdde_driver.cu", "tdde_shard.cu", "tdde_misc.cu", "tdde_noalloc.cu", "tdde_eigen.cu", "tdde_paper_variant.cu"]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-DTDDE_WITH_BENCH"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found; libtdde.so cannot be built (there is no CPU fallback)")


def _newest_header() -> float:
    t = 0.0
    for d in (CSRC, INCLUDE):
        for f in os.listdir(d):
            if f.endswith((".h", ".cuh")):
                t = max(t, os.path.getmtime(os.path.join(d, f)))
    return max(t, os.path.getmtime(os.path.abspath(__file__)))


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = _nvcc()
    bdir = os.path.join(CSRC, "build" + ("_" + "".join(c for c in "".join(EXTRA) if c.isalnum()) if EXTRA else ""))
    os.makedirs(bdir, exist_ok=True)
    hdr_t = _newest_header()
    flags = list(FLAGS)
    jobs = []
    objs = []
    for src in SOURCES:
        sp = os.path.join(CSRC, src)
        op = os.path.join(bdir, src.replace(".cu", ".o"))
        objs.append(op)
        if force or not os.path.exists(op) or os.path.getmtime(op) < max(os.path.getmtime(sp), hdr_t):
            jobs.append((src, [nvcc, *ARCH, *flags, *EXTRA, "-I", INCLUDE, "-I", CSRC, "-c", sp, "-o", op]))

    def run(job):
        name, cmd = job
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {name}:\n{r.stdout}\n{r.stderr}")
        with open(os.path.join(bdir, name.replace(".cu", ".ptxas.txt")), "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stderr)
        if verbose:
            print(r.stderr)
        return name

    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            list(ex.map(run, jobs))
    if jobs or force or not os.path.exists(OUT):
        cmd = [nvcc, *ARCH, "-shared", "-o", OUT, *objs, "-cudart", "static", "-ldl"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
