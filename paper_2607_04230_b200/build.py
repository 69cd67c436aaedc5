"""Builds csrc/libhair.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2607_04230_b200.build [--force] [--verbose]

HAIR_CFLAGS (environment) appends flags to the nvcc compile lines, e.g. "-DRAS_MIN_BLOCKS=4" to
try another tuning constant; such a build is for measurement only.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
SO = os.path.join(CSRC, "libhair.so")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
SOURCES = ["hair_api.cu", "k_lod.cu", "k_generate.cu", "k_raster.cu", "k_shade_filter.cu", "k_microbench.cu", "k_scan_noalloc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]


def _nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    raise RuntimeError("nvcc not found")


def _stale(target: str, deps: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    headers = [os.path.join(CSRC, "hair_internal.cuh"), os.path.join(CSRC, "gen_device.cuh"), os.path.join(INCLUDE, "hair.h")]
    nvcc = _nvcc()
    objs, jobs = [], []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(CSRC, s.replace(".cu", ".o"))
        objs.append(obj)
        if force or _stale(obj, [src] + headers):
            cmd = ([nvcc] + NVCC_FLAGS + os.environ.get("HAIR_CFLAGS", "").split()
                   + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj])
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        return r.stderr

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        for log in ex.map(run, jobs):
            if verbose and log:
                print(log)
    if force or jobs or _stale(SO, objs):
        run([nvcc, "-shared", "-o", SO] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
