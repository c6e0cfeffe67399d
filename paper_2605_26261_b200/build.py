"""Build libftlm.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2605_26261_b200.build [--force] [--verbose] [--checked]

--checked builds libftlm_checked.so from the same sources with -DFTLM_CHECKED: every computed address of
every kernel is range- and alignment-checked on the device, violations are suppressed and counted
(csrc/ftlm_access.cuh).  The binding loads it when FTLM_CHECKED=1 is set in the environment; the -m gpu test
session runs the suite through it first (tests/conftest.py).
"""
from __future__ import annotations

import glob
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libftlm.so")
SO_CHECKED = os.path.join(HERE, "libftlm_checked.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "--use_fast_math=false", "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _digest(checked: bool) -> str:
    """Hash of everything the library is built from (sources, headers, flags): the staleness test must not
    depend on file times, which a copy of the tree to another machine does not keep."""
    h = hashlib.sha256()
    deps = sources() + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [os.path.join(HERE, "..", "include", "ftlm.h")]
    for d in deps:
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    h.update(" ".join(FLAGS).encode() + (b" checked" if checked else b""))
    return h.hexdigest()


def stale(so: str = SO) -> bool:
    if not os.path.exists(so) or not os.path.exists(so + ".digest"):
        return True
    with open(so + ".digest") as f:
        return f.read().strip() != _digest(so == SO_CHECKED)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    so = SO_CHECKED if checked else SO
    if not force and not stale(so):
        return so
    objs = []
    procs = []
    for src in sources():
        obj = src[:-3] + (".chk.o" if checked else ".o")
        cmd = [NVCC, *[f for f in FLAGS if f != "--use_fast_math=false"], *(["-DFTLM_CHECKED"] if checked else []),
               "-c", src, "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((subprocess.Popen(cmd), cmd))
        objs.append(obj)
    for p, cmd in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    subprocess.check_call([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", *objs, "-o", so])
    with open(so + ".digest", "w") as f:
        f.write(_digest(checked))
    return so


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, checked="--checked" in sys.argv))
