"""TEST INFRASTRUCTURE: compile the library's kernel sources for the HOST against the SIMT
emulation layer (cuda_emu.h) into tests/emu/libftlm_emu.so.  Only `-m "not gpu"` tests load it
(through tests/emu/emu_harness.py); the product binding never does.

    python tests/emu/build_emu.py [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_2605_26261_b200", "csrc")
SO = os.path.join(HERE, "libftlm_emu.so")
CXX = os.environ.get("CXX", "g++")
FLAGS = ["-std=c++17", "-O1", "-g", "-fPIC", "-DFTLM_EMU", "-I", HERE, "-Wno-attributes", "-Wno-unknown-pragmas"]


def deps():
    return (sorted(glob.glob(os.path.join(CSRC, "*.cu"))) + glob.glob(os.path.join(CSRC, "*.cuh"))
            + glob.glob(os.path.join(HERE, "cuda_emu.*")) + [os.path.join(ROOT, "include", "ftlm.h")])


def build(force: bool = False) -> str:
    if not force and os.path.exists(SO) and all(os.path.getmtime(d) <= os.path.getmtime(SO) for d in deps()):
        return SO
    objs, procs = [], []
    for src in sorted(glob.glob(os.path.join(CSRC, "*.cu"))) + [os.path.join(HERE, "cuda_emu.cpp")]:
        obj = os.path.join(HERE, os.path.basename(src) + ".emu.o")
        cmd = [CXX, *FLAGS, "-x", "c++", "-c", src, "-o", obj]
        procs.append((subprocess.Popen(cmd), cmd))
        objs.append(obj)
    for p, cmd in procs:
        if p.wait() != 0:
            raise RuntimeError("emu compile failed: " + " ".join(cmd))
    subprocess.check_call([CXX, "-shared", *objs, "-o", SO])
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
