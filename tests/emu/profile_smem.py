"""TEST INFRASTRUCTURE: shared-memory wavefront profile of one pass of a full-size sector in the host emulation.

    FTLM_EMU_PROFILE=/tmp/p.json python tests/emu/profile_smem.py '{"config": 4, "mode": "cr", "pass": 0, "tmlr": 1, "item": "mid"}'

Runs ONE tile (pass 0: the in-tile pass, TML or TMLR) or ONE item of PASS-B window `pass - 1` of a BASELINE sector
through the emulation with FTLM_EMU_PROFILE set: the emulation groups the shared-memory accesses of each warp
instruction (source line, occurrence) and counts its wavefronts = the largest number of distinct 4-byte words that fall
into one bank.  Prints one JSON line: rows written, warp instructions, wavefronts, the conflict-free minimum, and the
source lines with the most wavefronts.  Counts only; it says nothing about time."""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, HERE)

import emu_harness as E  # noqa: E402
from paper_2605_26261_b200 import workloads as W  # noqa: E402


def main():
    spec = json.loads(sys.argv[1])
    path = os.environ["FTLM_EMU_PROFILE"]
    w = W.baseline_config(spec["config"])
    n_up = w.sectors[0]
    prec = spec.get("prec", "fp32")
    rng = np.random.default_rng(1)
    opts = [("passb", 1), ("kernel", 3), ("tmlr", int(spec.get("tmlr", 0)))] + [tuple(o) for o in spec.get("options", ())]
    with E.EmuCtx(w, n_up, spec.get("mode", "cr"), prec, options=opts) as c:
        D = c.dim
        v = rng.standard_normal(D).astype(E.NDT[prec])
        y = np.zeros(D, dtype=E.NDT[prec])
        ps = int(spec["pass"])
        n = c.get("tml_tiles") if ps == 0 else c.get(f"passb_items{ps - 1}")
        item = {"mid": n // 2 - 1, "third": n // 3}.get(spec.get("item", "mid"), spec.get("item"))
        c.set("debug_pass_mask", 1 << ps)
        c.set("debug_item_first", int(item))
        c.set("debug_item_count", 1)
        c.apply_into(v, y)
        rows = int(np.count_nonzero(y))
        info = {"tml": [c.get("tml_w"), c.get("tml_m")], "windows": c.get("passb_windows"), "tmlr": [c.get("tmlr"), c.get("tmlr_available")]}
    E.lib()                                                      # the profile is written when the process exits
    import ctypes
    ctypes.CDLL(None).fflush(None)
    print(json.dumps({"spec": spec, "rows": rows, "items": n, "item": int(item), "plan": info, "profile_file": path}))


if __name__ == "__main__":
    main()
