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
FLAGS = ["-std=c++17", "-O1", "-g", "-fPIC", "-pthread", "-DFTLM_EMU", "-I", HERE, "-Wno-attributes", "-Wno-unknown-pragmas"]


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
    subprocess.check_call([CXX, "-shared", "-pthread", *objs, "-o", SO])
    return SO


def build_negative(k: int) -> str:
    """A deliberately broken copy of the library for the negative tests of the emulation itself: -DFTLM_NEG_TEST=k
    removes one synchronisation from one kernel (1: the cp.async wait of PASS-B's staging phase, ftlm_passb.cu;
    2: the __syncwarp between building and reading the per-column descriptor lists, ftlm_tml.cu;
    3: the mbarrier wait after the bulk copy of TMLR's tile, ftlm_tmlr.cu).  A run through it
    must be killed by the emulation (tests/test_emu_kernels.py::test_emu_detects_removed_synchronisation)."""
    build()
    so = os.path.join(HERE, f"libftlm_emu_neg{k}.so")
    victim = {1: "ftlm_passb.cu", 2: "ftlm_tml.cu", 3: "ftlm_tmlr.cu"}[k]
    if os.path.exists(so) and all(os.path.getmtime(d) <= os.path.getmtime(so) for d in deps()):
        return so
    objs = []
    for src in sorted(glob.glob(os.path.join(CSRC, "*.cu"))) + [os.path.join(HERE, "cuda_emu.cpp")]:
        obj = os.path.join(HERE, os.path.basename(src) + ".emu.o")
        if os.path.basename(src) == victim:
            obj = os.path.join(HERE, os.path.basename(src) + f".neg{k}.emu.o")
            subprocess.check_call([CXX, *FLAGS, f"-DFTLM_NEG_TEST={k}", "-x", "c++", "-c", src, "-o", obj])
        objs.append(obj)
    subprocess.check_call([CXX, "-shared", "-pthread", *objs, "-o", so])
    return so


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
