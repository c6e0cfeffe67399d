"""One CHECKED-build case in its own process: sampled tiles / items of a full-size BASELINE sector on the device.

    FTLM_CHECKED=1 python tests/gpu_sampled.py '{"config": 4, "mode": "clt", "tmlr": 1, "samples": 2}'

The in-tile pass and every PASS-B window are run one at a time (checked-build option debug_pass_mask) on a few tiles /
items (debug_item_first / debug_item_count: the first, the last, one near the middle and random ones) of the real
sector - real run starts, real offsets, real vector size, rows beyond 2^31 at config 5 - in libftlm_checked.so, where
every computed address is range- and alignment-checked on the device and a bad one is suppressed and counted.  The
rows a pass changed are found by comparing y with its initial content; their values must be the oracle's (sampled-row
form of Eq. 12 restricted to the pass's bonds, in swap form (J_b/2)(v[P_b n] - v[n]) = H_b v - (J_b/4) v), a tile must
be exactly the contiguous rows the oracle's rank gives, and the violation counter must stay at zero.
Prints one JSON line with "ok"."""
import json
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import torch  # noqa: E402

from oracle import ftlm_oracle as fo  # noqa: E402
from paper_2605_26261_b200 import ftlm  # noqa: E402
from paper_2605_26261_b200 import workloads as W  # noqa: E402
from gpu_util import MODES  # noqa: E402


def main():
    spec = json.loads(sys.argv[1])
    assert ftlm.CHECKED, "gpu_sampled.py needs FTLM_CHECKED=1 (the item hooks exist only in the checked build)"
    w = W.baseline_config(spec["config"])
    n_up = w.sectors[0]
    mode = spec.get("mode", "cr")
    torch.cuda.set_device(0)
    ctx = ftlm.ftlm_create(w.N, w.bond_i, w.bond_j, w.J, n_up, MODES[mode], ftlm.FP32, 0.0)
    for k, val in [("passb", 1), ("kernel", 3), ("tmlr", int(spec.get("tmlr", 0)))] + [tuple(o) for o in spec.get("options", ())]:
        ftlm.ftlm_set_option(ctx, k, val)
    D = ftlm.ftlm_dim(ctx)
    assert D == math.comb(w.N, n_up)
    res = {"ok": True, "dim": D, "passes": [], "windows": max(ftlm.ftlm_get_option(ctx, "passb_windows"), 0),
           "tmlr": [ftlm.ftlm_get_option(ctx, "tmlr"), ftlm.ftlm_get_option(ctx, "tmlr_available")]}
    gen = torch.Generator(device="cuda").manual_seed(spec.get("seed", 1))
    v = torch.randn(D, generator=gen, device="cuda", dtype=torch.float32)
    y0 = torch.randn(D, generator=gen, device="cuda", dtype=torch.float32)
    y = y0.clone()

    def v_of(idx):
        return v[torch.from_numpy(np.ascontiguousarray(idx, dtype=np.int64)).cuda()].cpu().numpy().astype(np.float64)

    bclass = []
    for b in range(w.n_bonds):
        x = ftlm.ftlm_get_option(ctx, f"tml_bclass:{b}")
        bclass.append((x & 0xff, x >> 8))
    mw = ftlm.ftlm_get_option(ctx, "tml_w") + ftlm.ftlm_get_option(ctx, "tml_m")
    rng = np.random.default_rng(spec.get("seed", 1))
    diag0 = float(np.sum(w.J)) / 4.0
    touched = {}
    for ps in range(res["windows"] + 1):
        if ps == 0:
            nitems = ftlm.ftlm_get_option(ctx, "tml_tiles")
            bonds = [b for b in range(w.n_bonds) if bclass[b][0] != 6]
        else:
            nitems = ftlm.ftlm_get_option(ctx, f"passb_items{ps - 1}")
            bonds = [b for b in range(w.n_bonds) if bclass[b] == (6, ps - 1)]
        bi, bj, J = w.bond_i[bonds], w.bond_j[bonds], w.J[bonds]
        picks = set([0, nitems - 1] + [int(x) for x in rng.integers(0, nitems, spec.get("samples", 2))])
        if ps == 0:                                      # tiles near the middle hold the long rows
            picks |= {nitems // 2 - 1, nitems // 3}
        ftlm.ftlm_set_option(ctx, "debug_pass_mask", 1 << ps)
        ftlm.ftlm_set_option(ctx, "debug_item_count", 1)
        for it in sorted(picks):
            ftlm.ftlm_set_option(ctx, "debug_item_first", it)
            ftlm.ftlm_apply_H(ctx, v, y)
            torch.cuda.synchronize()
            rows_t = torch.nonzero(y != y0).flatten()
            rows = rows_t.cpu().numpy()
            ok, rel = True, 0.0
            if rows.size:
                ref = fo.apply_H_sampled_rows(w.N, bi, bj, J, 0.0, n_up, rows, v_of)
                vr = v_of(rows)
                got = y[rows_t].cpu().numpy().astype(np.float64)
                if ps == 0:
                    exp = ref + (diag0 - float(np.sum(J)) / 4.0) * vr
                else:
                    exp = ref - float(np.sum(J)) / 4.0 * vr
                    got = got - y0[rows_t].cpu().numpy().astype(np.float64)
                den = float(np.linalg.norm(exp))
                rel = float(np.linalg.norm(got - exp)) / (den if den > 0 else 1.0)
                ok = rel <= (1e-5 if ps == 0 else 2e-4)   # windows: y0 + delta rounds in the width of y0
                y[rows_t] = y0[rows_t]
            if ps == 0:                                  # a tile = the contiguous rows of top part T = it
                kT = n_up - bin(it).count("1")
                n_exp = math.comb(mw, kT) if 0 <= kT <= mw else 0
                if n_exp:
                    first = fo.rank_by_counting((it << mw) | ((1 << kT) - 1), w.N, n_up)
                    ok = ok and rows.size == n_exp and int(rows[0]) == first and int(rows[-1]) == first + n_exp - 1
                else:
                    ok = ok and rows.size == 0
            res["passes"].append({"pass": ps, "item": it, "rows": int(rows.size), "relerr": rel, "ok": bool(ok)})
            res["ok"] = res["ok"] and bool(ok)
            touched[ps] = max(touched.get(ps, 0), int(rows.size))
    # an item of a window class without antiparallel bonds changes nothing; every pass must have changed rows somewhere
    res["ok"] = res["ok"] and all(n > 0 for n in touched.values())
    res["rows_beyond_2_31"] = bool(D > 2 ** 31)
    ftlm.ftlm_set_option(ctx, "debug_pass_mask", 0)
    ftlm.ftlm_set_option(ctx, "debug_item_count", 0)
    ftlm.ftlm_destroy(ctx)
    chk = ftlm.ftlm_check_info()
    res["check"] = chk
    res["ok"] = bool(res["ok"] and chk["check_build"] == 1 and chk["check_violations"] == 0)
    print(json.dumps(res))


if __name__ == "__main__":
    main()
