"""Build libg6b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_0902_4463_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libg6b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "--shared", "-Xcompiler", "-fPIC,-O3,-Wall,-Wno-unused-function", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cpp")))


def deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")) + \
        glob.glob(os.path.join(HERE, "..", "include", "*.h"))


def build(force: bool = False, verbose: bool = False) -> str:
    stale = force or not os.path.exists(OUT) or any(os.path.getmtime(d) > os.path.getmtime(OUT) for d in deps())
    if stale:
        cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + sources() + ["-o", OUT + ".tmp"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed building libg6b200.so")
        os.replace(OUT + ".tmp", OUT)
    return OUT


# ---- the parity-test hook (csrc/debug/g6_debug_dx.cu): the production kernels with their DBG template flag, as a
# separate small library so that libg6b200.so carries no debug entry point
DBG_SRC = os.path.join(CSRC, "debug", "g6_debug_dx.cu")
DBG_OUT = os.path.join(HERE, "libg6b200_dbg.so")


# ---- bench.py's measurement aids (csrc/bench/g6_bench_probe.cu): instruction-rate and read-pass probes, their own library
PROBE_SRC = os.path.join(CSRC, "bench", "g6_bench_probe.cu")
PROBE_OUT = os.path.join(HERE, "libg6b200_probe.so")


def _build_side(src: str, out: str, force: bool) -> str:
    stale = force or not os.path.exists(out) or any(os.path.getmtime(d) > os.path.getmtime(out) for d in deps() + [src])
    if stale:
        r = subprocess.run([NVCC] + FLAGS + [src, "-o", out + ".tmp"], capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed building " + os.path.basename(out))
        os.replace(out + ".tmp", out)
    return out


def build_debug(force: bool = False) -> str:
    return _build_side(DBG_SRC, DBG_OUT, force)


def build_probe(force: bool = False) -> str:
    return _build_side(PROBE_SRC, PROBE_OUT, force)


def build_all(force: bool = False, verbose: bool = False):
    return [build(force, verbose), build_debug(force), build_probe(force)]


if __name__ == "__main__":
    for path in build_all(force="--force" in sys.argv, verbose="--verbose" in sys.argv):
        print(path)
