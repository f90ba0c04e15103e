"""Build libc8ph.so in-tree with nvcc for sm_100a (no GPU needed: nvcc cross-compiles).

    python -m paper_2405_04229_b200.build [--force] [--define NAME=VALUE ...] [--out PATH] [--prod-only]

--define / --out make an A/B build of the same sources with other compile-time choices (the knobs are
listed at the top of csrc/c8ph_kernels.cu; profiles/ records what each one measured); select it at
run time with the environment variable C8PH_LIB=PATH.  --prod-only instantiates only the kernel
variants bench.py's headline needs (seconds instead of a minute; A/B builds only).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libc8ph.so")
SOURCES = ("c8ph_host.cu", "c8ph_kernels.cu", "c8ph_substep.cu")
HEADERS = ("c8ph_device.cuh", "c8ph_philox.cuh", os.path.join("..", "..", "include", "c8ph.h"))
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _stale(lib: str) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=(), out: str | None = None) -> str:
    lib = os.path.abspath(out) if out else LIB
    if not force and not defines and not _stale(lib):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tag = "" if lib == LIB else "." + os.path.basename(lib).replace(".so", "")
    objs, procs = [], []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", tag + ".o"))
        cmd = [nvcc, *NVCC_FLAGS, *[f"-D{d}" for d in defines], "-c", os.path.join(CSRC, s), "-o", o]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(o)
    for cmd, p in procs:
        txt = p.communicate()[0]
        if verbose or p.returncode:
            sys.stderr.write(txt)
        if p.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    tmp = lib + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, "-shared", "-o", tmp, *objs, "-lcudart"])
    os.replace(tmp, lib)
    if tag:
        for o in objs:
            os.remove(o)
    return lib


if __name__ == "__main__":
    import argparse
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--define", action="append", default=[], metavar="NAME=VALUE")
    ap.add_argument("--out", default=None)
    ap.add_argument("--prod-only", action="store_true")
    ap.add_argument("--quiet", action="store_true")
    a = ap.parse_args()
    d = list(a.define) + (["C8PH_PROD_ONLY=1"] if a.prod_only else [])
    print(build(force=a.force or bool(d), verbose=not a.quiet, defines=d, out=a.out))
