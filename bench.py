#!/usr/bin/env python
"""bench.py - FTLM hot path on B200: fused Lanczos steps/s at D = 1.55e8 (BASELINE config 4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 4] [--mode clt|cr] [--kernel auto|row|tile] [--no-cpu-baseline]

A "step" is one fused Lanczos step (row states, diagonal, gather with
CLT or CR indexing, fused recurrence + FP64 reductions, normalisation pass) on the S^z = 0
sector of the N = 30 icosidodecahedron in FP32; the one-time tables (A0/A1) are built before
the timed region and the host parts (A8/A9) run once per chain inside the e2e measurement.
Prints ONE JSON line (rank 0).  N > 1: one independent chain (replica) per GPU, no data-path
collective ("scaling": "weak"); timing = max over ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "lanczos_steps_per_s"
UNIT = "steps/s"


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_traffic(kernel_key):
    """dram bytes/launch of the dominant kernel from the committed ncu --set full capture."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)).get(kernel_key)
        except Exception:
            return None
    return None


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 6:
                    self.rows.append(f)
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[2 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows)}


def oracle_hv_rate(w, n_up, budget_s=15.0):
    """Time the C oracle's H.v (as it stands) on a bounded sample of rows of the same sector."""
    from oracle import c_oracle as co
    t0 = time.time()
    basis = co.enumerate_basis(w.N, n_up)
    t_enum = time.time() - t0
    D = basis.shape[0]
    rng = np.random.default_rng(0)
    v = rng.standard_normal(D)
    rows = min(D, 1 << 18)
    t0 = time.time()
    co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v, 0, rows)
    dt = max(time.time() - t0, 1e-6)
    rows2 = int(min(D, max(rows, rows * budget_s / dt)))
    row0 = (D - rows2) // 2                       # middle of the sector: typical rows
    t0 = time.time()
    co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v, row0, rows2)
    dt = time.time() - t0
    return dict(rows_per_s=rows2 / dt, rows=rows2, row0=row0, seconds=dt, enum_seconds=t_enum,
                cores=co.threads(), D=D)


def run_reference(args, w, n_up):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import c_oracle as co
    basis = co.enumerate_basis(w.N, n_up)
    D = basis.shape[0]
    rng = np.random.default_rng(0)
    v = rng.standard_normal(D)
    # size one "step" = a bounded slice of rows so that K + W steps finish within ~2 minutes
    t0 = time.time()
    co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v, D // 2, 1 << 18)
    per_row = (time.time() - t0) / (1 << 18)
    rows = int(min(D, max(1 << 16, 100.0 / max(args.steps + args.warmup, 1) / per_row)))
    row0 = (D - rows) // 2
    for _ in range(args.warmup):
        co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v, row0, rows)
    t0 = time.time()
    for _ in range(args.steps):
        co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v, row0, rows)
    dt = time.time() - t0
    value = (rows * args.steps / dt) / D
    sample = (f"FP64 C/OpenMP oracle H.v on rows [{row0}, {row0 + rows}) of the D={D} sector per step; "
              f"steps/s = rows/s / D (vector updates of the recurrence not included)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": f"config{args.config}:{w.name}", "N": w.N, "N_up": n_up, "dim": D,
                                            "n_bonds": w.n_bonds, "sample_rows_per_step": rows},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": co.threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# name -> option settings, in order (the candidates of ftlm_autotune, include/ftlm.h)
CANDIDATES = {
    "row": [("lazy_norm", 0), ("tmlr", 0), ("kernel", 1)],
    "rowg": [("lazy_norm", 0), ("tmlr", 0), ("kernel", 2)],
    "tml": [("lazy_norm", 0), ("tmlr", 0), ("tml_split", 0), ("passb", 0), ("kernel", 3)],
    "tml+passb": [("tmlr", 0), ("tml_split", 0), ("passb_smax", 0), ("passb_ctas", 0), ("passb", 1), ("kernel", 3)],
    "tml+passb_1cta": [("tmlr", 0), ("tml_split", 0), ("passb_smax", 0), ("passb_ctas", 1), ("passb", 1), ("kernel", 3)],
    "tml+passb_s11": [("tmlr", 0), ("tml_split", 0), ("passb_smax", 11), ("passb_ctas", 0), ("passb", 1), ("kernel", 3)],
    "tml+passb_s10": [("tmlr", 0), ("tml_split", 0), ("passb_smax", 10), ("passb_ctas", 0), ("passb", 1), ("kernel", 3)],
    "tmlr+passb": [("tml_split", 0), ("passb_smax", 0), ("passb_ctas", 0), ("passb", 1), ("kernel", 3), ("tmlr", 1)],
    "tmlr+passb_s11": [("tml_split", 0), ("passb_smax", 11), ("passb_ctas", 0), ("passb", 1), ("kernel", 3), ("tmlr", 1)],
    "tmlr+passb_lazy": [("tml_split", 0), ("passb_smax", 0), ("passb_ctas", 0), ("passb", 1), ("kernel", 3), ("tmlr", 1), ("lazy_norm", 1)],
    "tmlr+passb_s11_lazy": [("tml_split", 0), ("passb_smax", 11), ("passb_ctas", 0), ("passb", 1), ("kernel", 3), ("tmlr", 1), ("lazy_norm", 1)],
    "tml_w9m7": [("lazy_norm", 0), ("tmlr", 0), ("tml_split", 9 | (7 << 8)), ("passb", 0), ("kernel", 3)],
    "tml_w9m7+passb": [("lazy_norm", 0), ("tmlr", 0), ("tml_split", 9 | (7 << 8)), ("passb_smax", 0), ("passb_ctas", 0), ("passb", 1), ("kernel", 3)],
}
SAFE_CHOICE = "row"          # thread-per-row kernel: parity-green on B200 in round 1 and the on-device reference of every candidate


def run_probe(args):
    """Child process: ftlm_autotune on the bench sector; prints one JSON line.
    stage "checked" (FTLM_CHECKED=1 in the environment: the binding loads libftlm_checked.so, in which every computed
    address is range- and alignment-checked on the device and a violation is suppressed and counted, never a fault):
    every candidate computes H.v and three fused steps and is compared on the device with the thread-per-row kernel;
    stage "release": the candidates named by --mask (those that passed the checked stage with zero violations) are
    timed in the release library and the fastest is chosen."""
    import torch
    from paper_2605_26261_b200 import ftlm, workloads as W
    w = W.baseline_config(args.config)
    n_up = w.sectors[0]
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    mode = ftlm.INDEX_CR if (args.mode == "cr" or w.N > 32) else ftlm.INDEX_CLT
    ctx = ftlm.ftlm_create(w.N, w.bond_i, w.bond_j, w.J, n_up, mode, ftlm.FP32, 0.0, torch.cuda.current_device())
    ftlm.ftlm_set_option(ctx, "allow_unverified", 1)
    if args.probe_stage in ("batchcheck", "batchtime"):
        # batch > 1.  "batchcheck" (checked library): three fused steps of `batch` interleaved chains through each batched
        # configuration (TML in-tile pass + PASS-B windows; TML with global reads) against the same chains through
        # the thread-per-row kernel one at a time; zero suppressed accesses.  "batchtime" (release library): times the
        # configurations named by --names over whole fused steps.
        B = args.batch
        names = [n for n in (args.names.split(",") if args.names else ["tml+passb", "tml"])]
        out = {}
        if args.probe_stage == "batchcheck":
            assert ftlm.CHECKED, "checked probe stage needs FTLM_CHECKED=1"
            ftlm.ftlm_set_option(ctx, "kernel", 1)
            ref = ftlm.ftlm_lanczos(ctx, W.SEED_VECTORS, B, 3)
        else:
            assert not ftlm.CHECKED
        ftlm.ftlm_set_option(ctx, "batch", B)
        for name in names:
            try:
                for key, val in CANDIDATES[name]:
                    ftlm.ftlm_set_option(ctx, key, val)
                if args.probe_stage == "batchcheck":
                    got = ftlm.ftlm_lanczos(ctx, W.SEED_VECTORS, B, 3)
                    out[name] = bool(np.abs(got["alpha"] - ref["alpha"]).max() <= 1e-4 and np.abs(got["beta"] - ref["beta"]).max() <= 1e-4)
                else:
                    ftlm.ftlm_chain_begin_batch(ctx, W.SEED_VECTORS, 0, B)
                    ftlm.ftlm_chain_steps(ctx, 2)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    ftlm.ftlm_chain_steps(ctx, 5)
                    e1.record()
                    torch.cuda.synchronize()
                    out[name] = e0.elapsed_time(e1) / 5
            except ftlm.FtlmError:
                out[name] = False
        info = ftlm.ftlm_check_info()
        ftlm.ftlm_destroy(ctx)
        print(json.dumps({"stage": args.probe_stage, "result": out, "check": info}), flush=True)
        return
    if args.probe_stage == "checked":
        assert ftlm.CHECKED, "checked probe stage needs FTLM_CHECKED=1"
        rep = ftlm.ftlm_autotune(ctx, 1)
        info = ftlm.ftlm_check_info()
        ftlm.ftlm_destroy(ctx)
        print(json.dumps({"stage": "checked", "report": rep, "check": info}), flush=True)
        return
    assert not ftlm.CHECKED
    ftlm.ftlm_set_option(ctx, "autotune_mask", args.mask)
    rep = ftlm.ftlm_autotune(ctx, 3)
    valid = [r for r in rep if r["valid"]]
    best = min(valid, key=lambda r: r["ms"])["name"] if valid else None
    ftlm.ftlm_destroy(ctx)
    print(json.dumps({"stage": "release", "choice": best, "report": rep}), flush=True)


def _child_json(cmd, env, timeout):
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env)
    for ln in reversed(out.stdout.strip().splitlines()):
        if ln.startswith("{"):
            return json.loads(ln), None
    return None, f"rc={out.returncode}: {out.stderr.strip()[-300:]}"


def probe_batch(args):
    """batch > 1: a batched configuration is timed only after the checked library ran it on this device without a
    suppressed access and in agreement with the thread-per-row kernel; else the batched thread-per-row kernel."""
    cmd = [sys.executable, os.path.abspath(__file__), "--probe", "--config", str(args.config), "--mode", args.mode, "--batch", str(args.batch)]
    try:
        from paper_2605_26261_b200 import build
        build.build(checked=True)
        d, err = _child_json(cmd + ["--probe-stage", "batchcheck"], dict(os.environ, FTLM_CHECKED="1"), 1800)
        if not d or d["check"].get("check_violations") != 0:
            return "row", None, f"batch check: {err or d}"
        ok = [n for n, v in d["result"].items() if v is True]
        if not ok:
            return "row", d, "batch check: no valid batched configuration"
        env = dict(os.environ)
        env.pop("FTLM_CHECKED", None)
        d2, err = _child_json(cmd + ["--probe-stage", "batchtime", "--names", ",".join(ok)], env, 900)
        if not d2:
            return "row", d, "batch timing " + str(err)
        timed = {n: v for n, v in d2["result"].items() if v is not False}
        if not timed:
            return "row", d2, "batch timing: nothing ran"
        return min(timed, key=timed.get), {"checked": d["result"], "release_ms": d2["result"]}, None
    except Exception as e:
        return "row", None, f"batch check failed: {e!r}"


def probe_choice(args):
    """Kernel configuration of the default run.  No candidate is timed in the release library before the SAME candidate
    has run on THIS device in the checked library with zero address violations and agreed with the thread-per-row
    kernel; if any stage fails the bench times the thread-per-row kernel."""
    cmd = [sys.executable, os.path.abspath(__file__), "--probe", "--config", str(args.config), "--mode", args.mode]
    try:
        from paper_2605_26261_b200 import build
        build.build(checked=True)                      # no-op when libftlm_checked.so is up to date
        d, err = _child_json(cmd + ["--probe-stage", "checked"], dict(os.environ, FTLM_CHECKED="1"), 1800)
        if d is None:
            return SAFE_CHOICE, None, "checked probe " + err
        chk, rep = d["check"], d["report"]
        if chk.get("check_build") != 1 or chk.get("check_violations") != 0:
            return SAFE_CHOICE, rep, f"checked probe: address violations on the device: {chk}"
        mask = 0
        for r in rep:
            if r["valid"] and r["name"] in CANDIDATES:
                mask |= 1 << int(r["index"])
        if mask == 0:
            return SAFE_CHOICE, rep, "checked probe: no valid candidate"
        env = dict(os.environ)
        env.pop("FTLM_CHECKED", None)
        d2, err = _child_json(cmd + ["--probe-stage", "release", "--mask", str(mask)], env, 900)
        if d2 is None or d2.get("choice") not in CANDIDATES:
            return SAFE_CHOICE, rep, "release probe " + (err or "no choice")
        return d2["choice"], {"checked": rep, "release": d2["report"]}, None
    except Exception as e:  # timeout, crash
        return SAFE_CHOICE, None, f"probe failed: {e!r}"


ALL_CASES = [  # (config, mode, extra flags): north_star "five synthetic clusters ... CLT vs CR"
    (1, "clt", []), (1, "cr", []), (1, "clt", ["--graph", "1"]), (1, "clt", ["--batch", "4", "--graph", "1"]), (1, "clt", ["--persistent", "1"]),
    (2, "clt", []), (2, "cr", []), (2, "clt", ["--graph", "1"]), (2, "clt", ["--batch", "4"]),
    (3, "clt", []), (3, "cr", []),
    (4, "clt", []), (4, "cr", []), (41, "clt", []), (40, "clt", []), (4, "clt", ["--batch", "2"]), (4, "clt", ["--batch", "4"]),
    (5, "cr", []),
]


def run_all(args):
    """Every BASELINE config (largest sector) and index mode, each in its own child bench run (own probe: no candidate
    is timed before the checked library has run it on this device); rows -> gpurun_out/bench_all.json and a table on
    stderr.  The ONE JSON line printed is the headline case (config 4, CLT, FP32, B = 1)."""
    rows, headline = [], None
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    for cfg, mode, extra in ALL_CASES:
        steps = {1: 200, 2: 200, 3: 60, 5: 20}.get(cfg, 40)
        cmd = [sys.executable, os.path.abspath(__file__), "--config", str(cfg), "--mode", mode, "--steps", str(steps),
               "--warmup", "3"] + extra
        if cfg == 5:
            cmd.append("--no-cpu-baseline")               # the oracle cannot enumerate this basis; its sampled-row form is a test tool
        if not (cfg == 4 and mode == "clt" and not extra):
            cmd.append("--no-e2e")
        try:
            d, err = _child_json(cmd, dict(os.environ), 3600)
        except Exception as e:
            d, err = None, repr(e)
        if d is None:
            rows.append({"config": cfg, "mode": mode, "flags": extra, "error": err})
            continue
        r = d["roofline"]
        rows.append({"config": cfg, "workload": d["config"]["workload"], "mode": mode, "flags": extra, "dim": d["config"]["dim"],
                     "kernel": d["config"]["candidate"], "hv_passes": d["config"]["hv_passes"], "steps_per_s": d["value"],
                     "ms_per_step": d["ms_per_step"], "hv_rows_per_s": d["hv_rows_per_s"], "hv_gelem_per_s": d["hv_gelem_per_s"],
                     "hv_ms": r.get("ms_per_launch"), "floorA_GBps": r["achieved"], "frac_of_measured_hbm": r["frac"],
                     "norm_GBps": r.get("norm_kernel_GBps"), "oracle_rows_per_s": (d.get("cpu_baseline") or {}).get("rows_per_s"),
                     "oracle_cores": (d.get("cpu_baseline") or {}).get("cores"), "clocks": d.get("clocks"),
                     "site_numbering": d["config"].get("site_numbering"), "probe_note": d["config"].get("probe_note")})
        if cfg == 4 and mode == "clt" and not extra:
            headline = d
        with open(os.path.join(ROOT, "gpurun_out", "bench_all.json"), "w") as f:
            json.dump(rows, f, indent=1)
    sys.stderr.write("| config | mode | flags | kernel | passes | steps/s | H.v rows/s | Gelem/s | floor-A GB/s | frac | oracle rows/s |\n|---|---|---|---|---|---|---|---|---|---|---|\n")
    for r in rows:
        if "error" in r:
            sys.stderr.write(f"| {r['config']} | {r['mode']} | {' '.join(r['flags'])} | ERROR {r['error']} |\n")
        else:
            sys.stderr.write(f"| {r['workload']} | {r['mode']} | {' '.join(r['flags'])} | {r['kernel']} | {r['hv_passes']} | {r['steps_per_s']:.1f} | "
                             f"{r['hv_rows_per_s']:.3e} | {(r['hv_gelem_per_s'] or 0):.2f} | {r['floorA_GBps']:.1f} | {r['frac_of_measured_hbm']:.4f} | "
                             f"{(r['oracle_rows_per_s'] or 0):.3e} |\n")
    if headline is not None:
        headline["config"]["all_cases_file"] = "gpurun_out/bench_all.json"
        print(json.dumps(headline), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--probe", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--probe-stage", default="checked", choices=["checked", "release", "batchcheck", "batchtime"], help=argparse.SUPPRESS)
    ap.add_argument("--names", default="", help=argparse.SUPPRESS)
    ap.add_argument("--mask", type=int, default=0, help=argparse.SUPPRESS)
    ap.add_argument("--candidate", default="", help="one of " + ", ".join(CANDIDATES))
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--mode", default="clt", choices=["clt", "cr"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "row", "tml"])
    ap.add_argument("--low-bits", type=int, default=0)
    ap.add_argument("--tml-low-bits", type=int, default=0)
    ap.add_argument("--tml-mid-bits", type=int, default=0)
    ap.add_argument("--batch", type=int, default=1, choices=[1, 2, 4], help="chains advanced together (L207); value counts chain-steps")
    ap.add_argument("--graph", type=int, default=0, choices=[0, 1], help="replay steps from a CUDA graph")
    ap.add_argument("--persistent", type=int, default=0, choices=[0, 1], help="small sectors: all chains of the sector in one launch (csrc/ftlm_chain.cu); times ftlm_lanczos(R, steps)")
    ap.add_argument("--all", action="store_true", help="every BASELINE config and index mode (children), table in gpurun_out/bench_all.json")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    from paper_2605_26261_b200 import workloads as W
    w = W.baseline_config(args.config)
    n_up = w.sectors[0]
    if args.impl == "reference":
        run_reference(args, w, n_up)
        return
    if args.all:
        run_all(args)
        return
    if args.probe:
        run_probe(args)
        return

    import torch
    from paper_2605_26261_b200 import ftlm, replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    mode = ftlm.INDEX_CLT if args.mode == "clt" else ftlm.INDEX_CR
    if w.N > 32:
        mode, args.mode = ftlm.INDEX_CR, "cr"
    ctx = ftlm.ftlm_create(w.N, w.bond_i, w.bond_j, w.J, n_up, mode, ftlm.FP32, 0.0, local)
    autotune_report, probe_note = None, None
    B = args.batch
    if args.candidate:
        choice = args.candidate
    elif B > 1:
        choice, autotune_report, probe_note = probe_batch(args) if rank == 0 else ("row", None, None)
        choice = replicas.broadcast_choice(choice, dist)
    elif args.kernel == "auto":
        # rank 0 probes in a child process; every rank applies the same choice
        choice, autotune_report, probe_note = probe_choice(args) if rank == 0 else (SAFE_CHOICE, None, None)
        choice = replicas.broadcast_choice(choice, dist)
    else:
        choice = {"row": "row", "tml": "tml"}[args.kernel]
    for key, val in CANDIDATES[choice]:
        ftlm.ftlm_set_option(ctx, key, val)
    if args.tml_low_bits:                                        # explicit split flags win over the candidate's
        ftlm.ftlm_set_option(ctx, "tml_low_bits", args.tml_low_bits)
    if args.tml_mid_bits:
        ftlm.ftlm_set_option(ctx, "tml_mid_bits", args.tml_mid_bits)
    if B > 1:                                                    # batched chains: TML in-tile pass (+ windows), or ROW
        for key in ("lazy_norm", "tmlr"):
            ftlm.ftlm_set_option(ctx, key, 0)
        ftlm.ftlm_set_option(ctx, "batch", B)
    ftlm.ftlm_set_option(ctx, "graph", args.graph)
    kernel_used = {1: "row", 2: "rowg", 3: "tml"}[ftlm.ftlm_get_option(ctx, "kernel")]
    if kernel_used == "tml" and ftlm.ftlm_get_option(ctx, "tmlr") == 1 and ftlm.ftlm_get_option(ctx, "tmlr_available") == 1:
        kernel_used = "tmlr"
    n_windows = max(ftlm.ftlm_get_option(ctx, "passb_windows"), 0) if kernel_used in ("tml", "tmlr") else 0
    ftlm_lazy = (kernel_used == "tmlr" and ftlm.ftlm_get_option(ctx, "lazy_norm") == 1
                 and ftlm.ftlm_get_option(ctx, "lazy_norm_ok") == 1)
    D = ftlm.ftlm_dim(ctx)
    K, Wm = args.steps, args.warmup
    assert 1 <= K and K + Wm <= ftlm.MAX_STEPS, "steps + warmup must be <= 1024 (one chain)"

    if args.persistent:
        # small sectors: ONE launch runs all R chains of the sector, one CTA per chain, vectors in shared
        # memory; the unit is still a fused chain-step, timed over whole ftlm_lanczos calls (device events)
        ftlm.ftlm_set_option(ctx, "persistent", 1)
        assert ftlm.ftlm_get_option(ctx, "persistent_fits") == 1, "--persistent: this sector does not fit shared memory"
        Rp = max(w.R, 1)
        for _ in range(max(Wm, 3)):
            ftlm.ftlm_lanczos(ctx, W.SEED_VECTORS, Rp, K)
        barrier()
        sampler = ClockSampler(local)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 5
        e0.record()
        for _ in range(reps):
            out = ftlm.ftlm_lanczos(ctx, W.SEED_VECTORS, Rp, K)
        e1.record()
        barrier()
        ms = replicas.max_over_ranks(e0.elapsed_time(e1), dist, device="cuda")
        sampler.stop_flag = True
        steps_done = int(out["m_eff"].sum())
        table_bytes = (8 * ((1 << w.N) // 32)) if mode == ftlm.INDEX_CLT else 0
        line = {"metric": METRIC, "value": world * reps * steps_done / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
                "ms_per_step": ms / (reps * max(steps_done, 1)), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": f"config{args.config}:{w.name}", "N": w.N, "N_up": n_up, "dim": D, "n_bonds": w.n_bonds,
                           "index_mode": args.mode, "kernel": "persistent_chain", "candidate": "persistent", "hv_passes": 1, "chains_per_launch": Rp,
                           "l2": "vectors resident in shared memory for the whole chain", "parallelism": f"replicas x{world}",
                           "note": "one launch = R chains x steps (start vectors, H.v, reductions, normalisation); includes the host tridiagonal solves of ftlm_lanczos"},
                "roofline": {"bound": "hbm", "achieved": (12 * D + table_bytes) * reps * steps_done / (ms * 1e-3) / 1e9, "peak": measured_peak()[0], "unit": "GB/s",
                             "frac": (12 * D + table_bytes) * reps * steps_done / (ms * 1e-3) / 1e9 / measured_peak()[0], "traffic": None,
                             "kernel": "lanczos_chain_kernel", "note": "launch-bound sector: the byte floor is not what bounds it (SURVEY H7)"},
                "cpu_baseline": None, "e2e": None, "gpu_launches": reps, "clocks": sampler.summary(),
                "hv_rows_per_s": world * D * reps * steps_done / (ms * 1e-3), "hv_gelem_per_s": None}
        ftlm.ftlm_destroy(ctx)
        if rank == 0:
            print(json.dumps(line), flush=True)
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- device-resident timing: `value` ---------------------------------------------------
    def begin():
        if B > 1:
            ftlm.ftlm_chain_begin_batch(ctx, W.SEED_VECTORS, rank * B, B)   # B replica chains per rank, interleaved
        else:
            ftlm.ftlm_chain_begin(ctx, None, W.SEED_VECTORS, rank)       # one replica chain per rank

    begin()
    ftlm.ftlm_chain_steps(ctx, Wm)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    ftlm.ftlm_chain_steps(ctx, K)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    sampler.stop_flag = True
    if B > 1:
        a, b, m_effs = ftlm.ftlm_chain_end_batch(ctx, B)
        m_eff = int(m_effs.min())
        assert int(m_effs.max()) == m_eff
    else:
        a, b, m_eff = ftlm.ftlm_chain_end(ctx)
    assert m_eff == min(K + Wm, D) and np.isfinite(a).all() and np.isfinite(b).all(), (m_eff, K + Wm)
    ms = replicas.max_over_ranks(ms, dist, device="cuda")
    value = world * B * K / (ms * 1e-3)                          # chain-steps per second (B = 1: steps per second)

    # ---- per-kernel timing for the roofline of the dominant kernel --------------------------
    begin()
    ftlm.ftlm_chain_steps(ctx, 3)
    ms_hv, ms_norm = ftlm.ftlm_chain_profile(ctx, min(K, 30))
    table_bytes = (8 * ((1 << w.N) // 32)) if mode == ftlm.INDEX_CLT else 0
    alg_bytes = 12 * B * D + table_bytes         # floor A of SURVEY 8(d): v, v_prev, y (x B chains) + table
    peak, peak_src = measured_peak()
    achieved = alg_bytes / (ms_hv * 1e-3) / 1e9
    kname = f"hv_{kernel_used}_{args.mode}_fp32_fused" + (f"+passb{n_windows}" if n_windows else "")
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": recorded_traffic(kname), "kernel": kname, "ms_per_launch": ms_hv,
                "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src,
                "norm_kernel_ms": ms_norm, "norm_kernel_GBps": 12 * D / (ms_norm * 1e-3) / 1e9 if ms_norm > 0 else None}

    # ---- end-to-end through the host-buffer ABI call ---------------------------------------
    e2e = None
    if not args.no_e2e:
        hq = torch.empty((B, D), dtype=torch.float32).pin_memory()
        hq.normal_(generator=torch.Generator().manual_seed(1234 + rank))
        hq_np = hq.numpy()
        ke = min(K, 100)
        ftlm.ftlm_lanczos_host(ctx, hq_np, 2)                     # warm-up of the path (B start vectors = one batch)
        barrier()
        t0 = time.perf_counter()
        out = ftlm.ftlm_lanczos_host(ctx, hq_np, ke)              # H2D start vector, ke steps, D2H alpha/beta, T eig
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        t_e = replicas.max_over_ranks(dt, dist, device="cuda")
        assert int(out["m_eff"][0]) == ke
        e2e = {"value": world * B * ke / t_e, "unit": UNIT, "h2d_bytes_per_step": 4 * B * D / ke,
               "d2h_bytes_per_step": B * (16.0 + 8.0 / ke), "steps": ke,
               "call": "ftlm_lanczos_host(pinned host start vector -> alpha, beta, theta, weight)"}

    ftlm.ftlm_destroy(ctx)
    if dist is not None:
        dist.barrier()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        o = oracle_hv_rate(w, n_up)
        cpu = {"value": o["rows_per_s"] / D, "unit": UNIT, "cores": o["cores"], "kind": "oracle",
               "sample": (f"FP64 C/OpenMP oracle H.v on rows [{o['row0']}, {o['row0'] + o['rows']}) of the D={D} "
                          f"sector ({o['seconds']:.1f} s); steps/s = rows/s / D; basis enumeration "
                          f"({o['enum_seconds']:.1f} s) excluded"),
               "rows_per_s": o["rows_per_s"]}

    nnz = D + 2 * w.n_bonds * __import__("math").comb(w.N - 2, n_up - 1)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"config{args.config}:{w.name}", "N": w.N, "N_up": n_up, "dim": D,
                       "n_bonds": w.n_bonds, "index_mode": args.mode, "kernel": kernel_used, "candidate": choice,
                       "hv_passes": 1 + n_windows, "autotune": autotune_report, "probe_note": probe_note,
                       "precision": "fp32 vectors, fp64 reductions",
                       "l2": (f"inputs_exceed_l2 (3 x {4 * D / 1e6:.0f} MB vectors)" if 12 * D > 126e6 else
                              f"inputs_fit_l2 (3 x {4 * D / 1e6:.2f} MB vectors: this workload is L2-resident by size; no flush between steps)"),
                       "site_numbering": {4: "CONFIG4_SITE_ORDER (annealed for two window passes, DESIGN.md section 3)", 40: "CONFIG4_SITE_ORDER",
                                          41: "lexicographic icosahedron edges (SURVEY 8(d))", 5: "fold_order(34)"}.get(args.config, "SURVEY 8(d)"),
                       "batch": args.batch, "graph": args.graph,
                       "parallelism": f"replicas x{world}"},
            "hv_rows_per_s": world * B * D / (ms_hv * 1e-3), "hv_gelem_per_s": world * B * nnz / (ms_hv * 1e-3) / 1e9,
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": ((1 if ftlm_lazy else 2) + n_windows) * K,
            "clocks": sampler.summary()}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
