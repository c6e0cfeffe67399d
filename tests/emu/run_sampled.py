"""TEST INFRASTRUCTURE: sampled tiles / items of a FULL-SIZE sector run through the host emulation.

    python tests/emu/run_sampled.py '{"config": 4, "mode": "cr", "samples": 3, "seed": 1}'

The TML pass and every PASS-B window are run one at a time (option debug_pass_mask) on a few
tiles / items (debug_item_first / debug_item_count) of the real BASELINE sector, with the real
run starts, offsets and vector size.  The rows a pass wrote are found by comparing y with its
initial content; they must be exactly the rows the oracle expects to change, with the oracle's
values (H restricted to the pass's bonds, in swap form: (J_b/2)(v[P_b n] - v[n]) = H_b v - J_b/4 v).
Out-of-bounds accesses hit the emulation's guard pages.  Prints one JSON line.
"""
from __future__ import annotations

import ctypes as C
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, HERE)

import emu_harness as E  # noqa: E402
from oracle import c_oracle as co  # noqa: E402
from paper_2605_26261_b200 import workloads as W  # noqa: E402


def runs_of(idx):
    """sorted row indices -> list of (start, length) of maximal contiguous runs"""
    if idx.size == 0:
        return []
    cut = np.flatnonzero(np.diff(idx) != 1) + 1
    starts = np.concatenate(([0], cut))
    ends = np.concatenate((cut, [idx.size]))
    return [(int(idx[a]), int(b - a)) for a, b in zip(starts, ends)]


def main():
    spec = json.loads(sys.argv[1])
    w = W.baseline_config(spec["config"]) if "config" in spec else None
    n_up = w.sectors[0]
    mode, prec = spec.get("mode", "cr"), spec.get("prec", "fp32")
    rng = np.random.default_rng(spec.get("seed", 1))
    basis = co.enumerate_basis(w.N, n_up)
    D = basis.shape[0]
    if spec.get("lowmem"):                               # generated in blocks: no float64 temporary of the whole vector
        v = np.empty(D, dtype=E.NDT[prec])
        for a in range(0, D, 1 << 26):
            v[a:a + (1 << 26)] = rng.standard_normal(min(1 << 26, D - a))
    else:
        v = rng.standard_normal(D).astype(E.NDT[prec])
    v64 = v.astype(np.float64)
    res = {"ok": True, "dim": D, "passes": []}
    tol = 1e-5 if prec == "fp32" else 1e-12
    with E.EmuCtx(w, n_up, mode, prec, options=[("passb", 1)] + [tuple(o) for o in spec.get("options", ())]) as c:
        assert c.dim == D
        nwin = max(c.get("passb_windows"), 0)
        res["kernel"] = c.get("kernel")
        res["windows"] = nwin
        bclass = c.bond_classes()
        touched = {}
        plist = list(range(nwin + 1)) + ([-1] if spec.get("tmlr_both") else [])   # -1: pass 0 again with the other in-tile kernel
        for ps in plist:
            if ps == -1:
                c.set("tmlr", 0 if c.get("tmlr") else 1)
                ps = 0
            if ps == 0:
                nitems = c.get("tml_tiles")
                bonds = [b for b in range(w.n_bonds) if bclass[b][0] != 6]
            else:
                nitems = c.get(f"passb_items{ps - 1}")
                bonds = [b for b in range(w.n_bonds) if bclass[b] == (6, ps - 1)]
            bi, bj, J = w.bond_i[bonds], w.bond_j[bonds], w.J[bonds]
            shift = float(np.sum(J)) / 4.0
            picks = sorted(set([0, nitems - 1] + [int(x) for x in rng.integers(0, nitems, spec.get("samples", 2))]))
            if ps == 0:                                  # tiles near the middle hold the long rows
                picks = sorted(set(picks + [nitems // 2 - 1, nitems // 3]))
            c.set("debug_pass_mask", 1 << ps)
            c.set("debug_item_count", 1)
            for it in picks:
                c.set("debug_item_first", it)
                if spec.get("lowmem"):                   # N = 34: y starts as (lazily allocated) zeros
                    y0 = None
                    y = np.zeros(D, dtype=E.NDT[prec])
                else:
                    y0 = rng.standard_normal(D).astype(E.NDT[prec])
                    y = y0.copy()
                c.apply_into(v, y)
                rows = np.flatnonzero(y != y0) if y0 is not None else np.flatnonzero(y)
                err2 = ref2 = 0.0
                nrows = 0
                for r0, n in runs_of(rows):
                    ref = co.apply_rows(w.N, bi, bj, J, 0.0, n_up, basis, v64, r0, n)
                    if ps == 0:
                        exp = ref + (c.diag0() - float(np.sum(J)) / 4.0) * v64[r0:r0 + n]
                        got = y[r0:r0 + n].astype(np.float64)
                    else:
                        exp = ref - shift * v64[r0:r0 + n]
                        got = y[r0:r0 + n].astype(np.float64) - (y0[r0:r0 + n].astype(np.float64) if y0 is not None else 0.0)
                    err2 += float(np.sum((got - exp) ** 2))
                    ref2 += float(np.sum(exp ** 2))
                    nrows += n
                rel = (err2 / ref2) ** 0.5 if ref2 > 0 else 0.0
                ok = rel <= (tol if ps == 0 else 20 * tol)   # windows: y0 + delta rounds in the width of y0
                res["passes"].append({"pass": ps, "tmlr": c.get("tmlr") if ps == 0 else None, "item": it, "rows": nrows, "relerr": rel, "ok": bool(ok)})
                res["ok"] = res["ok"] and bool(ok)
                touched[ps] = max(touched.get(ps, 0), nrows)
        # an item of a window class without antiparallel bonds (all window bits equal) changes nothing; every pass
        # must have changed rows in at least one sampled item
        res["ok"] = res["ok"] and all(n > 0 for n in touched.values())
        c.set("debug_pass_mask", 0)
        c.set("debug_item_count", 0)
    print(json.dumps(res))


if __name__ == "__main__":
    main()
