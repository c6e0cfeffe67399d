"""One -m gpu parity case in its own process (so that a faulting kernel cannot poison the CUDA context
of the pytest process): the CUDA path through the C ABI against the FP64 oracle.

    python tests/gpu_case.py '{"wl": "ring22j", "n_up": 11, "mode": "cr", "prec": "fp32",
                               "options": [["passb", 1]], "what": ["neighbors", "apply", "lanczos"]}'
    python tests/gpu_case.py '{"config": 4, "mode": "clt", "autotune": true, "what": ["sampled"]}'
Prints one JSON line with "ok".
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import torch  # noqa: E402

from oracle import c_oracle as co  # noqa: E402
from oracle import ftlm_oracle as fo  # noqa: E402
from paper_2605_26261_b200 import ftlm  # noqa: E402
from paper_2605_26261_b200 import workloads as W  # noqa: E402
from gpu_util import MODES, NDT, PRECS, TDT, elem_bound  # noqa: E402


def workload(spec):
    if "config" in spec:
        return W.baseline_config(spec["config"])
    name = spec["wl"]
    if name.startswith("fring"):                         # ring with folded site order (no long wrap bonds)
        j2 = name.endswith("j")
        n = int(name[5:-1] if j2 else name[5:])
        return W.relabel(W.ring(n, 1.0, 0.5 if j2 else None), W.fold_order(n))
    if name.startswith("ring"):
        j2 = name.endswith("j")
        return W.ring(int(name[4:-1] if j2 else name[4:]), 1.0, 0.5 if j2 else None)
    if name.startswith("square"):
        a, b = name[6:].split("x")
        return W.square(int(a), int(b))
    if name.startswith("tri"):
        a, b = name[3:].split("x")
        return W.triangular(int(a), int(b))
    if name in ("dodecahedron", "ring20"):
        return W.paper_workload(name)
    if name.startswith("rand"):                          # randN_E_seed: random graph, random J
        n, e, s = (int(x) for x in name[4:].split("_"))
        rng = np.random.default_rng(s)
        pairs = set()
        while len(pairs) < e:
            a, b = rng.integers(0, n, 2)
            if a != b:
                pairs.add((int(min(a, b)), int(max(a, b))))
        pairs = sorted(pairs)
        return W._mk(name, n, pairs, rng.uniform(0.5, 1.5, len(pairs)))
    raise ValueError(name)


def run_variants(spec):
    """Whole-vector parity of several kernel configurations of ONE workload in one process: the basis, the input
    vector, the oracle's y = H v and the oracle's Lanczos coefficients are computed once (they do not depend on the
    index mode or the kernel), then every variant {"mode", "options", "steps"} is run through the C ABI and compared."""
    w = workload(spec)
    n_up = spec.get("n_up", w.sectors[0])
    prec = spec.get("prec", "fp32")
    tol = 1e-5 if prec == "fp32" else 1e-12
    torch.cuda.set_device(0)
    basis = co.enumerate_basis(w.N, n_up)
    D = basis.shape[0]
    rng = np.random.default_rng(spec.get("seed", 1))
    v = rng.standard_normal(D).astype(NDT[prec])
    ref = co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v.astype(np.float64), 0, D)
    ref_norm = float(np.linalg.norm(ref))
    bound = elem_bound(v, w.J, 0.0, w.N, prec)
    max_steps = max([int(x.get("steps", 0)) for x in spec["variants"]] + [0])
    a_ref = b_ref = None
    if max_steps:
        q1 = fo.start_vector(W.SEED_VECTORS, n_up, 0, D)
        a_ref, b_ref = co.lanczos(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, q1, max_steps)[:2]
        a_ref, b_ref = np.asarray(a_ref), np.asarray(b_ref)
    dv = torch.from_numpy(v).cuda()
    res = {"ok": True, "dim": D, "variants": []}
    for var in spec["variants"]:
        ctx = ftlm.ftlm_create(w.N, w.bond_i, w.bond_j, w.J, n_up, MODES[var["mode"]], PRECS[prec], 0.0)
        for k, val in var.get("options", ()):
            ftlm.ftlm_set_option(ctx, k, val)
        r = {"mode": var["mode"], "options": var.get("options", []), "kernel": ftlm.ftlm_get_option(ctx, "kernel"),
             "windows": ftlm.ftlm_get_option(ctx, "passb_windows"),
             "tmlr": [ftlm.ftlm_get_option(ctx, "tmlr"), ftlm.ftlm_get_option(ctx, "tmlr_available")]}
        dy = torch.full_like(dv, float("nan"))
        ftlm.ftlm_apply_H(ctx, dv, dy)
        torch.cuda.synchronize()
        y = dy.cpu().numpy().astype(np.float64)
        del dy
        r["hv_relerr"] = float(np.linalg.norm(y - ref)) / ref_norm
        r["hv_maxabs"], r["hv_elem_bound"] = float(np.max(np.abs(y - ref))), bound
        ok = bool(np.isfinite(y).all()) and r["hv_relerr"] <= tol and r["hv_maxabs"] <= bound
        m = int(var.get("steps", 0))
        if m:
            out = ftlm.ftlm_lanczos(ctx, W.SEED_VECTORS, 1, m)
            k = min(int(out["m_eff"][0]), m, 6)
            ltol = 1e-9 if prec == "fp64" else 2e-4
            r["lanczos_dalpha"] = float(np.max(np.abs(out["alpha"][0][:k] - a_ref[:k])))
            r["lanczos_dbeta"] = float(np.max(np.abs(out["beta"][0][:k - 1] - b_ref[:k - 1]))) if k > 1 else 0.0
            th_ref, _ = fo.ritz(a_ref[:m], b_ref[:m - 1])
            th = out["theta"][0][:m]
            rtol = (1e-9 if prec == "fp64" else 5e-4) * max(1.0, float(np.abs(th_ref).max()))
            r["ritz_dmin"], r["ritz_dmax"] = float(abs(th.min() - th_ref.min())), float(abs(th.max() - th_ref.max()))
            r["wsum"] = float(out["weight"][0][:m].sum())
            ok = (ok and int(out["m_eff"][0]) == m and r["lanczos_dalpha"] <= ltol and r["lanczos_dbeta"] <= ltol
                  and r["ritz_dmin"] <= rtol and r["ritz_dmax"] <= rtol and abs(r["wsum"] - 1.0) <= 1e-6)
        ftlm.ftlm_destroy(ctx)
        r["ok"] = bool(ok)
        res["variants"].append(r)
        res["ok"] = res["ok"] and bool(ok)
    chk = ftlm.ftlm_check_info()
    res["check"] = chk
    if ftlm.CHECKED:
        res["ok"] = res["ok"] and chk["check_build"] == 1 and chk["check_violations"] == 0
    res["ok"] = bool(res["ok"])
    print(json.dumps(res))


def main():
    spec = json.loads(sys.argv[1])
    if "variants" in spec:
        run_variants(spec)
        return
    w = workload(spec)
    n_up = spec.get("n_up", w.sectors[0])
    mode, prec = spec.get("mode", "cr"), spec.get("prec", "fp32")
    tol = 1e-5 if prec == "fp32" else 1e-12
    res = {"ok": True}
    torch.cuda.set_device(0)
    ctx = ftlm.ftlm_create(w.N, w.bond_i, w.bond_j, w.J, n_up, MODES[mode], PRECS[prec], 0.0)
    for k, v in spec.get("options", ()):
        ftlm.ftlm_set_option(ctx, k, v)
    D = ftlm.ftlm_dim(ctx)
    if spec.get("autotune"):
        rep = ftlm.ftlm_autotune(ctx, 2)
        res["autotune"] = rep
        res["ok"] = res["ok"] and all(r["valid"] for r in rep)
    res["kernel"] = ftlm.ftlm_get_option(ctx, "kernel")
    res["windows"] = ftlm.ftlm_get_option(ctx, "passb_windows")
    res["dim"] = D
    res["tmlr"] = [ftlm.ftlm_get_option(ctx, "tmlr"), ftlm.ftlm_get_option(ctx, "tmlr_available")]
    what = spec.get("what", ["apply"])
    basis = co.enumerate_basis(w.N, n_up)
    rng = np.random.default_rng(spec.get("seed", 1))
    if "neighbors" in what:
        out = torch.empty(D * w.n_bonds, dtype=torch.int64, device="cuda")
        ftlm.ftlm_neighbors(ctx, 0, D, out)
        torch.cuda.synchronize()
        nb = out.cpu().numpy().reshape(D, w.n_bonds)
        ref = co.neighbors_rows(w.N, w.bond_i, w.bond_j, basis, np.arange(D, dtype=np.int64))
        res["neighbors_bad"] = int(np.count_nonzero(nb != ref))
        res["ok"] = res["ok"] and res["neighbors_bad"] == 0
    if "apply" in what or "sampled" in what:
        v = rng.standard_normal(D).astype(NDT[prec])
        dv = torch.from_numpy(v).cuda()
        dy = torch.full_like(dv, float("nan"))
        ftlm.ftlm_apply_H(ctx, dv, dy)
        torch.cuda.synchronize()
        y = dy.cpu().numpy().astype(np.float64)
        res["finite"] = bool(np.isfinite(y).all())
        v64 = v.astype(np.float64)
        if "apply" in what:
            ranges = [(0, D)]
        else:                                            # head, tail and random interior blocks of 2^16 rows
            n = 1 << 16
            starts = [0, D - n] + [int(x) for x in rng.integers(0, D - n, spec.get("blocks", 6))]
            ranges = [(s, n) for s in starts]
        err2 = ref2 = worst = 0.0
        for r0, n in ranges:
            ref = co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v64, r0, n)
            err2 += float(np.sum((y[r0:r0 + n] - ref) ** 2))
            ref2 += float(np.sum(ref ** 2))
            worst = max(worst, float(np.max(np.abs(y[r0:r0 + n] - ref))) if n else 0.0)
        res["hv_relerr"] = (err2 / ref2) ** 0.5 if ref2 > 0 else 0.0
        res["hv_maxabs"], res["hv_elem_bound"] = worst, elem_bound(v, w.J, 0.0, w.N, prec)   # element-wise criterion beside the norm
        res["ok"] = res["ok"] and res["finite"] and res["hv_relerr"] <= tol and worst <= res["hv_elem_bound"]
    if "lanczos" in what:
        m = min(spec.get("steps", 8), D)
        out = ftlm.ftlm_lanczos(ctx, W.SEED_VECTORS, 1, m)
        q1 = fo.start_vector(W.SEED_VECTORS, n_up, 0, D)
        a, b = co.lanczos(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, q1, m)[:2]
        k = min(int(out["m_eff"][0]), len(a), 6)
        ltol = 1e-9 if prec == "fp64" else 2e-4
        da = float(np.max(np.abs(out["alpha"][0][:k] - np.asarray(a)[:k]))) if k else 0.0
        kb = max(k - 1, 0)
        db = float(np.max(np.abs(out["beta"][0][:kb] - np.asarray(b)[:kb]))) if kb else 0.0
        res["lanczos_dalpha"], res["lanczos_dbeta"] = da, db
        res["m_eff"] = int(out["m_eff"][0])
        # extremal Ritz values of the whole run (converge first, L246) and the weight sum rule
        th_ref, _ = fo.ritz(np.asarray(a), np.asarray(b))
        th = out["theta"][0][: res["m_eff"]]
        res["ritz_dmin"], res["ritz_dmax"] = float(abs(th.min() - th_ref.min())), float(abs(th.max() - th_ref.max()))
        res["wsum"] = float(out["weight"][0][: res["m_eff"]].sum())
        rtol = (1e-9 if prec == "fp64" else 5e-4) * max(1.0, float(np.abs(th_ref).max()))
        res["ok"] = (res["ok"] and da <= ltol and db <= ltol and res["m_eff"] == m and res["ritz_dmin"] <= rtol
                     and res["ritz_dmax"] <= rtol and abs(res["wsum"] - 1.0) <= 1e-6)
    ftlm.ftlm_destroy(ctx)
    chk = ftlm.ftlm_check_info()                             # checked build (FTLM_CHECKED=1): no suppressed access
    res["check"] = chk
    if ftlm.CHECKED:
        res["ok"] = res["ok"] and chk["check_build"] == 1 and chk["check_violations"] == 0
    res["ok"] = bool(res["ok"])
    print(json.dumps(res))


if __name__ == "__main__":
    main()
