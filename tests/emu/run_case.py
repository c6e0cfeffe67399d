"""TEST INFRASTRUCTURE: run ONE emulated parity case and print a JSON result line.

    python tests/emu/run_case.py '<json spec>'

spec = {"wl": "ring12j"|..., "n_up": k, "mode": "cr"|"clt", "prec": "fp32"|"fp64", "options": [[key, value], ...],
        "what": ["neighbors", "apply", "lanczos"], "h": 0.0, "randJ": false}
Compares the emulated CUDA path (kernel sources compiled for the host, tests/emu/cuda_emu.h) with the
FP64 oracle on the same seeded inputs: neighbour indices bit-exactly, H.v in the norm-relative error,
Lanczos alpha/beta (FP64) element-wise for the first steps.
"""
from __future__ import annotations

import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, HERE)

from oracle import ftlm_oracle as fo  # noqa: E402
from paper_2605_26261_b200 import workloads as W  # noqa: E402
import emu_harness as E  # noqa: E402
sys.path.insert(0, os.path.join(ROOT, "tests"))
from hv_bound import elem_bound  # noqa: E402


def workload(name):
    if name.startswith("fring"):                     # ring with folded site order (no long wrap bonds)
        j2 = name.endswith("j")
        n = int(name[5:-1] if j2 else name[5:])
        return W.relabel(W.ring(n, 1.0, 0.5 if j2 else None), W.fold_order(n))
    if name.startswith("ring"):
        j2 = name.endswith("j")
        n = int(name[4:-1] if j2 else name[4:])
        return W.ring(n, 1.0, 0.5 if j2 else None)
    if name.startswith("square"):
        a, b = name[6:].split("x")
        return W.square(int(a), int(b))
    if name.startswith("tri"):
        a, b = name[3:].split("x")
        return W.triangular(int(a), int(b))
    if name == "icosahedron":
        return W.icosahedron()
    if name in ("dodecahedron", "ring20"):
        return W.paper_workload(name)
    if name.startswith("rand"):                      # randN_E_seed : random graph, random J
        n, e, s = (int(x) for x in name[4:].split("_"))
        rng = np.random.default_rng(s)
        pairs = set()
        while len(pairs) < e:
            a, b = rng.integers(0, n, 2)
            if a != b:
                pairs.add((min(a, b), max(a, b)))
        pairs = sorted(pairs)
        J = rng.uniform(0.5, 1.5, len(pairs))
        return W._mk(name, n, pairs, J)
    raise ValueError(name)


def main():
    spec = json.loads(sys.argv[1])
    w = workload(spec["wl"])
    n_up = spec["n_up"]
    h = spec.get("h", 0.0)
    mode, prec = spec.get("mode", "cr"), spec.get("prec", "fp64")
    res = {"ok": True}
    basis = fo.sector_basis(w.N, n_up)
    D = basis.shape[0]
    with E.EmuCtx(w, n_up, mode, prec, h=h, options=spec.get("options", ())) as c:
        res["kernel"] = c.get("kernel")
        res["dim"] = c.dim
        res["passb"] = [c.get("passb_windows"), c.get("passb_bonds"), c.get("passb_lo"), c.get("passb_s")]
        res["tml"] = [c.get("tml_w"), c.get("tml_m")]
        res["tmlr"] = [c.get("tmlr"), c.get("tmlr_available")]
        res["persistent"] = [c.get("persistent"), c.get("persistent_fits")]
        assert c.dim == D
        what = spec.get("what", ["neighbors", "apply"])
        if "neighbors" in what:
            nb = c.neighbors(0, D)
            ref = fo.neighbor_indices(basis, w.bond_i, w.bond_j, np.arange(D))
            bad = int(np.count_nonzero(nb != ref))
            res["neighbors_bad"] = bad
            if bad:
                r, b = np.argwhere(nb != ref)[0]
                res["first_bad"] = [int(r), int(b), int(nb[r, b]), int(ref[r, b])]
                res["ok"] = False
        if "apply" in what:
            rng = np.random.default_rng(spec.get("seed", 1))
            v = rng.standard_normal(D).astype(E.NDT[prec])
            y = c.apply(v, spec.get("shift", 0))
            ref = fo.apply_H(basis, w.N, w.bond_i, w.bond_j, w.J, h, n_up, v.astype(np.float64))
            den = np.linalg.norm(ref)
            err = float(np.linalg.norm(y.astype(np.float64) - ref) / (den if den > 0 else 1.0))
            res["hv_relerr"] = err
            res["hv_maxabs"] = float(np.max(np.abs(y.astype(np.float64) - ref))) if D else 0.0
            res["hv_elem_bound"] = elem_bound(v, w.J, h, w.N, prec)       # element-wise criterion beside the norm
            res["ok"] = (res["ok"] and bool(np.isfinite(y).all()) and err <= (1e-5 if prec == "fp32" else 1e-12)
                         and res["hv_maxabs"] <= res["hv_elem_bound"])
        if "lanczos" in what:
            m = min(spec.get("steps", 12), D)
            out = c.lanczos(W.SEED_VECTORS, 1, m)
            q1 = fo.start_vector(W.SEED_VECTORS, n_up, 0, D)
            a, b = fo.lanczos(lambda x: fo.apply_H(basis, w.N, w.bond_i, w.bond_j, w.J, h, n_up, x), q1, m)[:2]
            k = min(int(out["m_eff"][0]), len(a), 8)
            tol = 1e-9 if prec == "fp64" else 2e-4
            da = float(np.max(np.abs(out["alpha"][0][:k] - np.asarray(a)[:k]))) if k else 0.0
            kb = max(k - 1, 0)
            db = float(np.max(np.abs(out["beta"][0][:kb] - np.asarray(b)[:kb]))) if kb else 0.0
            res["lanczos_dalpha"], res["lanczos_dbeta"] = da, db
            res["m_eff"] = int(out["m_eff"][0])
            res["ok"] = res["ok"] and da <= tol and db <= tol
            if spec.get("chains", 1) > 1:                  # several chains in one call (persistent kernel: one CTA each)
                Rn = spec["chains"]
                outR = c.lanczos(W.SEED_VECTORS, Rn, m)
                worst = 0.0
                for r in range(Rn):
                    q1 = fo.start_vector(W.SEED_VECTORS, n_up, r, D)
                    ar, br = fo.lanczos(lambda x: fo.apply_H(basis, w.N, w.bond_i, w.bond_j, w.J, h, n_up, x), q1, m)[:2]
                    kk = min(int(outR["m_eff"][r]), len(ar), 8)
                    if kk:
                        worst = max(worst, float(np.max(np.abs(outR["alpha"][r][:kk] - np.asarray(ar)[:kk]))))
                    if kk > 1:
                        worst = max(worst, float(np.max(np.abs(outR["beta"][r][:kk - 1] - np.asarray(br)[:kk - 1]))))
                    worst = max(worst, abs(float(outR["weight"][r][: int(outR["m_eff"][r])].sum()) - 1.0))
                res["chains_worst"] = worst
                res["chains_m_eff"] = [int(x) for x in outR["m_eff"]]
                res["ok"] = res["ok"] and worst <= max(tol, 1e-6)
        if "batch" in spec:
            # batched chains (L207, L309): R chains in groups of B on interleaved vectors; every chain must be
            # bit-identical to the same chain run alone (same kernel, same tile split) and agree with the oracle
            R, B = spec["batch"]
            m = min(spec.get("steps", 10), D)
            c.set("plan_batch", B)                      # same tiles and windows for the single chains: bit-identical sums
            c.set("batch", 1)
            one = c.lanczos(W.SEED_VECTORS, R, m)
            c.set("batch", B)
            res["batch_split"] = [c.get("tml_w"), c.get("tml_m"), c.get("kernel"), c.get("passb_windows")]
            many = c.lanczos(W.SEED_VECTORS, R, m)
            same = all(np.array_equal(one[k], many[k]) for k in ("alpha", "beta", "m_eff", "theta", "weight"))
            res["batch_identical"] = bool(same)
            res["batch_m_eff"] = [int(x) for x in many["m_eff"]]
            worst = 0.0
            tol = 1e-9 if prec == "fp64" else 2e-4
            for r in range(R):
                q1 = fo.start_vector(W.SEED_VECTORS, n_up, r, D)
                a, b = fo.lanczos(lambda x: fo.apply_H(basis, w.N, w.bond_i, w.bond_j, w.J, h, n_up, x), q1, m)[:2]
                k = min(int(many["m_eff"][r]), len(a), 6)
                if k:
                    worst = max(worst, float(np.max(np.abs(many["alpha"][r][:k] - np.asarray(a)[:k]))))
                if k > 1:
                    worst = max(worst, float(np.max(np.abs(many["beta"][r][:k - 1] - np.asarray(b)[:k - 1]))))
            res["batch_vs_oracle"] = worst
            res["ok"] = res["ok"] and same and worst <= tol
            c.set("batch", 1)
            c.set("plan_batch", 0)
    res["ok"] = bool(res["ok"])
    print(json.dumps(res))


if __name__ == "__main__":
    main()
