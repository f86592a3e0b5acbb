"""Build libstreams.so (sm_100a) in-tree with nvcc.

    python -m paper_2304_05494_b200.build [--force] [--verbose] [--define NAME[=VALUE] ...] [--tag TAG]

--define adds -DNAME[=VALUE] to every translation unit and --tag TAG writes the result to lib_TAG/libstreams.so instead
of lib/ (builds with another tuning constant, e.g. --define STREAMS_MARCH_NSLOT=3 --tag nslot3; select one at run time
with STREAMS_LIB=<path>).

streams_canon.cu is compiled with -fmad=false (canonical, contraction-free evaluation of the
sensor path); the other translation units use the default FMA contraction.
The translation units compile in parallel (the two heavy ones, streams_march.cu and streams_weno.cu, first).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "lib")
LIB = os.path.join(OUT, "libstreams.so")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", *ARCH]
UNITS = [("streams_march.cu", []), ("streams_weno.cu", []), ("streams_canon.cu", ["-fmad=false"]), ("streams_fill.cu", []),
         ("streams_api.cu", []), ("streams_static.cu", [])]


def _newest_source() -> float:
    t = 0.0
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for f in os.listdir(root):
            t = max(t, os.path.getmtime(os.path.join(root, f)))
    return t


def build(force: bool = False, verbose: bool = False, defines=(), tag: str = "") -> str:
    out_dir = OUT if not tag else os.path.join(HERE, "lib_" + tag)
    lib = os.path.join(out_dir, "libstreams.so")
    os.makedirs(out_dir, exist_ok=True)
    if not force and not defines and os.path.exists(lib) and os.path.getmtime(lib) >= _newest_source():
        return lib
    nvcc = os.environ.get("NVCC", "nvcc")
    objs = []
    procs = []
    for src, extra in UNITS:
        obj = os.path.join(out_dir, src.replace(".cu", ".o"))
        cmd = [nvcc, *COMMON, *extra, *["-D" + d for d in defines], "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd))
        procs.append((cmd, subprocess.Popen(cmd)))
        objs.append(obj)
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    subprocess.check_call([nvcc, "-shared", *ARCH, "-o", lib, *objs])
    return lib


if __name__ == "__main__":
    argv = sys.argv[1:]
    defs = [argv[i + 1] for i, a in enumerate(argv) if a == "--define" and i + 1 < len(argv)]
    tags = [argv[i + 1] for i, a in enumerate(argv) if a == "--tag" and i + 1 < len(argv)]
    print(build(force="--force" in argv, verbose="--verbose" in argv, defines=defs, tag=tags[0] if tags else ""))
