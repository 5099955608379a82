"""Build libcans_poisson.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Usage: ``python -m paper_2001_05234_b200.build [--force]`` or ``build()`` from Python.
The translation units compile in parallel; objects go to ``csrc/build/``.
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libcans_poisson.so")
SOURCES = ["xw_kernels.cu", "yt_kernels.cu", "cans_poisson.cu", "z_solve.cu", "probes.cu", "chkdt_static.cu",
           "xy_group_a.cu", "xy_group_b.cu", "xy_group_c.cu", "xy_group_d.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-I", os.path.join(ROOT, "include"),
]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA toolkit is required to build libcans_poisson.so")


def _source_digest() -> str:
    """SHA-256 over the names and contents of every file the library is built from (csrc/*, include/*) and the flags."""
    h = hashlib.sha256(" ".join(NVCC_FLAGS[:-1]).encode())
    for d in (CSRC, os.path.join(ROOT, "include")):
        for fn in sorted(os.listdir(d)):
            p = os.path.join(d, fn)
            if os.path.isfile(p):
                h.update(fn.encode())
                with open(p, "rb") as fh:
                    h.update(fh.read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    """Rebuild unless the library exists and was built from exactly these sources (a digest of their contents, kept beside
    the objects -- modification times say nothing after a checkout)."""
    digest = _source_digest()
    stamp = os.path.join(CSRC, "build", "sources.sha256")
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read().strip() == digest:
        return LIB
    nvcc = _nvcc()
    bdir = os.path.join(CSRC, "build")
    os.makedirs(bdir, exist_ok=True)
    keep = {src.replace(".cu", ".o") for src in SOURCES}
    for fn in os.listdir(bdir):             # objects and logs of sources that no longer exist
        if (fn.endswith(".o") and fn not in keep) or (fn.endswith(".o.log") and fn[:-4] not in keep):
            os.remove(os.path.join(bdir, fn))
    if os.path.exists(stamp):
        os.remove(stamp)

    def compile_one(src):
        obj = os.path.join(bdir, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        with open(obj + ".log", "w") as fh:
            fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
        return obj

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    cmd = [nvcc, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    with open(stamp, "w") as fh:
        fh.write(digest + "\n")
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
