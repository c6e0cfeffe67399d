"""Host-side execution of the CUDA kernel sources (`-m "not gpu"`).

The library's .cu files are compiled as C++ against tests/emu/cuda_emu.h (every CUDA thread a fiber,
real barrier / warp-collective rendezvous, guard pages behind every "device" allocation and behind the
dynamic shared memory) and driven through the same C ABI as on the GPU.  Each case runs in a
subprocess and is compared with the FP64 oracle: neighbour indices bit-exactly, H.v within the
north_star tolerance, the first Lanczos coefficients.  This checks index arithmetic, plan tables,
barrier placement and bounds of every kernel variant without a GPU; it says nothing about speed.
"""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
RUN = os.path.join(ROOT, "tests", "emu", "run_case.py")

K = {"row": 1, "tml": 3}


def run_case(spec, timeout=600, order=None):
    env = dict(os.environ, FTLM_EMU_ORDER=str(order)) if order is not None else None
    p = subprocess.run([sys.executable, RUN, json.dumps(spec)], capture_output=True, text=True, timeout=timeout, env=env)
    assert p.returncode == 0, f"emulated case died (rc={p.returncode}): {spec}\n{p.stderr[-2000:]}"
    res = json.loads(p.stdout.strip().splitlines()[-1])
    assert res["ok"], (spec, res)
    return res


@pytest.fixture(scope="module", autouse=True)
def _build():
    sys.path.insert(0, os.path.join(ROOT, "tests", "emu"))
    import build_emu
    build_emu.build()


@pytest.mark.parametrize("mode,prec", [("cr", "fp64"), ("clt", "fp32")])
@pytest.mark.parametrize("kernel", ["row"])
def test_emu_row_kernel(kernel, mode, prec):
    res = run_case({"wl": "ring12j", "n_up": 6, "mode": mode, "prec": prec, "options": [["kernel", K[kernel]]],
                    "what": ["neighbors", "apply", "lanczos"]})
    assert res["kernel"] == K[kernel]


@pytest.mark.parametrize("wl,n_up,w,m,mode,prec", [
    ("ring14j", 7, 5, 3, "cr", "fp64"),
    ("ring16j", 8, 6, 4, "clt", "fp32"),
    ("ring16j", 5, 7, 5, "cr", "fp32"),
    ("rand14_30_3", 7, 5, 5, "clt", "fp64"),
    ("tri4x4", 8, 8, 4, "cr", "fp32"),
])
def test_emu_tml_kernel(wl, n_up, w, m, mode, prec):
    res = run_case({"wl": wl, "n_up": n_up, "mode": mode, "prec": prec,
                    "options": [["tml_low_bits", w], ["tml_mid_bits", m], ["kernel", K["tml"]]],
                    "what": ["neighbors", "apply", "lanczos"]})
    assert res["kernel"] == K["tml"]


def test_emu_guard_pages_catch_overrun():
    """The checker itself: a read past the end of an emulated device buffer must kill the process."""
    code = ("import sys; sys.path.insert(0, %r); import numpy as np, ctypes as C, emu_harness as E; L = E.lib();"
            "p = C.c_void_p(); L.cudaMalloc = None" % os.path.join(ROOT, "tests", "emu"))
    # cudaMalloc is a C++ symbol of the emulation layer; exercise it through a tiny kernel instead:
    # apply_H with a y buffer one element short must fault on the last store.
    code = ("import sys; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
            "import numpy as np, ctypes as C, emu_harness as E\n"
            "from paper_2605_26261_b200 import workloads as W\n"
            "w = W.ring(10)\n"
            "c = E.EmuCtx(w, 5, 'cr', 'fp64', options=[('kernel', 1)])\n"
            "import mmap\n"
            "m = mmap.mmap(-1, 8192)\n"
            "buf = (C.c_char * 8192).from_buffer(m)\n"
            "base = C.addressof(buf)\n"
            "C.CDLL(None).mprotect(C.c_void_p(base + 4096), C.c_size_t(4096), C.c_int(0))\n"
            "v = np.ones(c.dim)\n"
            "y_addr = base + 4096 - 8 * (c.dim - 1)\n"      # one element short of the guard page
            "E._check(E.lib().ftlm_apply_H(c.ctx, C.c_void_p(v.ctypes.data), C.c_void_p(y_addr), C.c_void_p(0)))\n"
            "print('survived')\n" % (ROOT, os.path.join(ROOT, "tests", "emu")))
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=120)
    assert p.returncode != 0 and "survived" not in p.stdout


@pytest.mark.parametrize("wl,n_up,w,m,mode,prec,what", [
    ("ring16j", 8, 5, 3, "cr", "fp64", ["neighbors", "apply", "lanczos"]),      # one window, no frozen bits
    ("ring16j", 8, 5, 3, "clt", "fp32", ["apply", "lanczos"]),
    ("rand15_40_5", 7, 5, 2, "clt", "fp64", ["neighbors", "apply", "lanczos"]),  # random graph, random J
                             # two windows, frozen bits above the second
])
def test_emu_two_pass_tml_plus_passb(wl, n_up, w, m, mode, prec, what):
    """PASS-B (bonds among the top label bits streamed by window) + the TML pass that leaves them out."""
    res = run_case({"wl": wl, "n_up": n_up, "mode": mode, "prec": prec,
                    "options": [["passb", 1], ["tml_split", w | (m << 8)], ["kernel", K["tml"]]], "what": what, "steps": 6},
                   timeout=1500)
    assert res["kernel"] == K["tml"] and res["passb"][0] >= 1 and res["passb"][1] >= 3


@pytest.mark.parametrize("wl,n_up,split,mode,prec,opts,nwin,what", [
    # windows reach below the tile boundary (TM / TL bonds too) and need not be contiguous
    ("ring16j", 8, 5 | (3 << 8), "cr", "fp64", [["passb_lo_min", 4]], 1, ["neighbors", "apply", "lanczos"]),
    ("rand15_40_5", 7, 5 | (2 << 8), "clt", "fp64", [["passb_lo_min", 3], ["passb_smax", 6]], 2, ["neighbors", "apply", "lanczos"]),
    ("rand15_40_5", 6, 5 | (2 << 8), "cr", "fp32", [["passb_lo_min", 5], ["passb_smax", 5], ["passb_ctas", 1]], 2, ["neighbors", "apply"]),
])
def test_emu_generalised_windows(wl, n_up, split, mode, prec, opts, nwin, what):
    """PASS-B windows as arbitrary sets of label positions >= lo_min chosen by the greedy cover."""
    res = run_case({"wl": wl, "n_up": n_up, "mode": mode, "prec": prec,
                    "options": [["passb", 1]] + opts + [["tml_split", split], ["kernel", K["tml"]]], "what": what, "steps": 6},
                   timeout=1500)
    assert res["kernel"] == K["tml"] and res["passb"][0] >= nwin


@pytest.mark.parametrize("wl,n_up,split,mode,prec,opts", [
    ("fring16j", 8, 5 | (3 << 8), "cr", "fp32", [["passb_lo_min", 4]]),
    ("fring14j", 7, 5 | (3 << 8), "clt", "fp64", [["passb_lo_min", 4]]),
    ("fring15", 6, 6 | (3 << 8), "clt", "fp32", [["passb_lo_min", 4]]),
    # windows only above the tile: the bonds between M and T stay in TMLR as coalesced global reads
    ("fring16j", 7, 5 | (4 << 8), "clt", "fp64", [["passb_lo_min", 9]]),
])
def test_emu_tmlr_in_tile_pass(wl, n_up, split, mode, prec, opts):
    """TMLR (lane tables in registers, per-column descriptors) as the in-tile pass, PASS-B windows for the rest."""
    res = run_case({"wl": wl, "n_up": n_up, "mode": mode, "prec": prec,
                    "options": [["passb", 1]] + opts + [["tml_split", split], ["kernel", K["tml"]], ["tmlr", 1]],
                    "what": ["apply", "lanczos"], "steps": 6}, timeout=1500)
    assert res["tmlr"] == [1, 1] and res["passb"][0] >= 1


@pytest.mark.parametrize("shift,prec", [(1, "fp32"), (2, "fp32"), (3, "fp32"), (1, "fp64")])
def test_emu_tmlr_bulk_copy_with_unaligned_caller_vectors(shift, prec):
    """The tile's bulk copy (cp.async.bulk: 16-byte aligned source, destination, size) takes its alignment from the
    actual address of the caller's vector, which is only element-aligned (a slice of a larger buffer)."""
    res = run_case({"wl": "fring16j", "n_up": 8, "mode": "clt", "prec": prec, "shift": shift,
                    "options": [["passb", 1], ["passb_lo_min", 4], ["tml_split", 5 | (3 << 8)], ["kernel", K["tml"]], ["tmlr", 1]],
                    "what": ["apply"]})
    assert res["tmlr"] == [1, 1]


@pytest.mark.parametrize("spec", [
    {"wl": "ring12j", "n_up": 6, "mode": "cr", "prec": "fp64"},
    {"wl": "rand15_40_5", "n_up": 7, "mode": "clt", "prec": "fp32"},
    {"wl": "ring16", "n_up": 15, "mode": "lin", "prec": "fp32", "steps": 16},       # D = 16: two groups of 8, breakdown
    {"wl": "ring12", "n_up": 0, "mode": "cr", "prec": "fp64", "what": ["neighbors", "apply"]},   # D = 1, label 0
    {"wl": "ring12", "n_up": 12, "mode": "clt", "prec": "fp32", "what": ["neighbors", "apply"]},
    {"wl": "ring13", "n_up": 5, "mode": "cr", "prec": "fp32"},                        # D = 1287: ragged last group
])
def test_emu_rowg_unrank_plus_gosper_successor(spec):
    """Kernel ROWG (north_star: "row bit-states by unranking plus Gosper-style successor enumeration"): a thread unranks
    the first of 8 consecutive rows (L136) and steps through the next seven with the same-popcount successor; neighbour
    indices bit-exact, H.v and Lanczos against the oracle, in all three index modes and on the degenerate sectors."""
    res = run_case(dict({"what": ["neighbors", "apply", "lanczos"], "options": [["kernel", 2]]}, **spec))
    assert res["kernel"] == 2


def test_emu_rowg_64_bit_labels_sampled():
    code = ("import sys, json; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
            "import numpy as np, emu_harness as E\n"
            "from oracle import ftlm_oracle as fo\n"
            "from paper_2605_26261_b200 import workloads as W\n"
            "w = W.baseline_config(5)\n"
            "_, Dc = fo.cr_tables(34)\n"
            "bad = 0\n"
            "with E.EmuCtx(w, 17, 'cr', 'fp32', options=[('kernel', 2)]) as c:\n"
            "    for r0 in (0, 2**31 - 5, c.dim // 2 + 3, c.dim - 19):\n"
            "        nb = c.neighbors(int(r0), 19)\n"
            "        lab = fo.alg1_unrank_vec(np.arange(r0, r0 + 19, dtype=np.uint64), 34, 17, Dc)\n"
            "        for k in range(19):\n"
            "            for b in range(w.n_bonds):\n"
            "                m = (1 << int(w.bond_i[b])) | (1 << int(w.bond_j[b])); x = int(lab[k]) & m\n"
            "                e = -1 if x in (0, m) else fo.rank_by_counting(int(lab[k]) ^ m, 34, 17)\n"
            "                bad += int(nb[k, b] != e)\n"
            "print(json.dumps({'bad': bad}))\n" % (ROOT, os.path.join(ROOT, "tests", "emu")))
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    assert json.loads(p.stdout.strip().splitlines()[-1])["bad"] == 0


@pytest.mark.parametrize("spec,fits", [
    ({"wl": "ring12j", "n_up": 6, "mode": "cr", "prec": "fp64", "steps": 20, "chains": 3}, 1),
    ({"wl": "ring14", "n_up": 7, "mode": "clt", "prec": "fp32", "steps": 8, "chains": 5}, 1),
    ({"wl": "ring16", "n_up": 15, "mode": "lin", "prec": "fp32", "steps": 16, "chains": 2}, 1),       # breakdown at step 9
    ({"wl": "ring16", "n_up": 16, "mode": "cr", "prec": "fp64", "steps": 5}, 1),                        # D = 1
    ({"wl": "ring20", "n_up": 5, "mode": "cr", "prec": "fp32", "steps": 4}, 1),                         # D = 15 504: vectors fit, stored labels do not
    ({"wl": "ring16", "n_up": 8, "mode": "cr", "prec": "fp64", "steps": 3}, 0),                         # 3 x 12 870 doubles do not fit: ordinary path
])
def test_emu_persistent_chain_kernel(spec, fits):
    """Option "persistent": all chains of a small sector in one launch, one CTA per chain with the three
    work vectors in shared memory; alpha, beta, weights against the oracle chain by chain."""
    res = run_case(dict({"what": ["lanczos"], "options": [["persistent", 1]]}, **spec))
    assert res["persistent"] == [1, fits]


def test_emu_passb_off_keeps_top_bonds_in_tml():
    res = run_case({"wl": "ring16j", "n_up": 8, "mode": "cr", "prec": "fp64",
                    "options": [["passb", 0], ["tml_split", 5 | (3 << 8)], ["kernel", K["tml"]]],
                    "what": ["neighbors", "apply"]})
    assert res["passb"][0] == 0


def test_emu_autotune_checks_every_candidate_against_row():
    """ftlm_autotune: every candidate is compared with the ROW kernel on the (emulated) device and timed."""
    code = ("import sys, json; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
            "import emu_harness as E\n"
            "from paper_2605_26261_b200 import workloads as W\n"
            "w = W.relabel(W.ring(14, 1.0, 0.5), W.fold_order(14))\n"
            "with E.EmuCtx(w, 7, 'cr', 'fp32', options=[('passb_lo_min', 4), ('tml_split', 5 | (3 << 8))]) as c:\n"
            "    rep0 = c.autotune(1)\n"
            "    c.set('allow_unverified', 1)\n"
            "    rep = c.autotune(1)\n"
            "    c.set('autotune_mask', 1 << [r['index'] for r in rep if r['name'] == 'tmlr+passb'][0])\n"
            "    rep2 = c.autotune(1)\n"
            "    print(json.dumps({'rep0': rep0, 'rep': rep, 'rep2': rep2, 'tuned': c.get('autotuned')}))\n" % (ROOT, os.path.join(ROOT, "tests", "emu")))
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    d = json.loads(p.stdout.strip().splitlines()[-1])
    # by default only configurations with a device record are run; the full list needs the opt-in
    import re
    src = open(os.path.join(ROOT, "paper_2605_26261_b200", "csrc", "ftlm_autotune.cu")).read()
    verified = set(re.findall(r'\{"([a-z0-9_+]+)",[^}]*, 1\},', src))
    assert {r["name"] for r in d["rep0"]} == verified and "row" in verified
    names = [r["name"] for r in d["rep"]]
    assert names[0] == "row" and "tml" in names and "tml+passb" in names and "tmlr+passb" in names
    assert all(r["valid"] and r["relerr"] <= 1e-5 and r["maxabs"] <= r["elem_bound"] for r in d["rep"]) and d["tuned"] >= 1
    # "autotune_mask" (bench.py: the candidates its checked pre-flight passed): the reference and the named candidate only
    assert [r["name"] for r in d["rep2"]] == ["row", "tmlr+passb"]
    import bench
    assert set(names) <= set(bench.CANDIDATES), set(names) - set(bench.CANDIDATES)   # bench.py can apply whatever is chosen


def test_emu_config4_full_size_sampled_tiles_and_items():
    """BASELINE config 4 (D = 155 117 520) at full size, in the index mode bench.py times (CLT, 268 MB table): sampled tiles of the TML pass and sampled items of
    both PASS-B windows (in-tile pass: TMLR and TML) run through the emulation with the real run starts and offsets; the rows each
    pass writes and their values must be the oracle's (and nothing may touch a guard page)."""
    p = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "emu", "run_sampled.py"),
                        json.dumps({"config": 4, "mode": "clt", "samples": 1, "options": [["tmlr", 1]], "tmlr_both": True})],
                       capture_output=True, text=True, timeout=1500)
    assert p.returncode == 0, p.stderr[-2000:]
    d = json.loads(p.stdout.strip().splitlines()[-1])
    assert d["ok"] and d["windows"] == 2 and d["kernel"] == K["tml"], d
    assert {x["pass"] for x in d["passes"]} == {0, 1, 2} and {x.get("tmlr") for x in d["passes"] if x["pass"] == 0} == {0, 1}
    assert all(x["ok"] for x in d["passes"])


def test_emu_lazy_normalisation_matches_separate_pass():
    """Option lazy_norm: the TMLR pass forms q_{j+1} = (y_j - alpha_j q_j)/beta_j while staging its tile (no
    normalisation kernel, buffers rotate by three).  Same arithmetic, so alpha and beta must be identical."""
    code = ("import sys, json; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
            "import numpy as np, emu_harness as E\n"
            "from paper_2605_26261_b200 import workloads as W\n"
            "w = W.relabel(W.ring(14, 1.0, 0.5), W.fold_order(14))\n"
            "out = {}\n"
            "for prec, mode in (('fp32', 'clt'), ('fp64', 'cr')):\n"
            "    res = []\n"
            "    for lazy in (0, 1):\n"
            "        opts = [('passb', 1), ('passb_lo_min', 4), ('tml_split', 5 | (3 << 8)), ('kernel', 3), ('tmlr', 1), ('lazy_norm', lazy)]\n"
            "        with E.EmuCtx(w, 7, mode, prec, options=opts) as c:\n"
            "            assert c.get('lazy_norm_ok') == 1 and c.get('passb_windows') >= 1\n"
            "            res.append(c.lanczos(W.SEED_VECTORS, 2, 6))\n"
            "    out[prec] = [float(np.abs(res[0][k] - res[1][k]).max()) for k in ('alpha', 'beta')] + [int(res[1]['m_eff'].min())]\n"
            "print(json.dumps(out))\n" % (ROOT, os.path.join(ROOT, "tests", "emu")))
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    d = json.loads(p.stdout.strip().splitlines()[-1])
    for prec in ("fp32", "fp64"):
        assert d[prec][0] <= 1e-12 and d[prec][1] <= 1e-12 and d[prec][2] == 6, d


@pytest.mark.parametrize("neg,spec,expect", [
    (1, {"wl": "ring16j", "n_up": 8, "mode": "clt", "prec": "fp32",
         "options": [["passb", 1], ["tml_split", 5 | (3 << 8)], ["kernel", 3]], "what": ["apply"]}, "cp.async"),
    (2, {"wl": "ring16j", "n_up": 8, "mode": "cr", "prec": "fp32",
         "options": [["tml_low_bits", 6], ["tml_mid_bits", 4], ["kernel", 3]], "what": ["apply"]}, "shared-memory race"),
    (3, {"wl": "fring16j", "n_up": 8, "mode": "cr", "prec": "fp32",
         "options": [["passb", 1], ["passb_lo_min", 4], ["tml_split", 5 | (3 << 8)], ["kernel", 3], ["tmlr", 1]], "what": ["apply"]}, "mbarrier"),
])
def test_emu_detects_removed_synchronisation(neg, spec, expect):
    """Negative test of the checker: a copy of the library with ONE synchronisation removed (1: the cp.async wait of
    PASS-B's staging, 2: the __syncwarp between building and reading TML's descriptor lists, 3: the mbarrier wait after the bulk copy of
    TMLR's tile) must be killed by the
    emulation - by the deferred cp.async model / the shared-memory race detector - while the intact library passes
    the same case."""
    import build_emu
    assert run_case(spec)["ok"]
    so = build_emu.build_negative(neg)
    p = subprocess.run([sys.executable, RUN, json.dumps(spec)], capture_output=True, text=True, timeout=900,
                       env=dict(os.environ, FTLM_EMU_LIB=so))
    ok = p.returncode == 0 and json.loads(p.stdout.strip().splitlines()[-1])["ok"]
    assert not ok, "the emulation did not notice the removed synchronisation"
    assert expect in p.stderr or p.returncode == 0, p.stderr[-1500:]      # died for the expected reason (or produced wrong values)


@pytest.mark.parametrize("order", [5])
def test_emu_result_does_not_depend_on_thread_schedule(order):
    """The emulation resumes runnable threads in ascending order by default; descending (1) and pseudo-random (>= 2)
    orders must give the same result - a difference would be a race (missing __syncthreads / __syncwarp)."""
    spec = {"wl": "fring14j", "n_up": 7, "mode": "clt", "prec": "fp64",
            "options": [["passb", 1], ["passb_lo_min", 4], ["tml_split", 5 | (3 << 8)], ["kernel", K["tml"]], ["tmlr", 1],
                        ["lazy_norm", 1]], "what": ["apply", "lanczos"], "steps": 6}
    ref = run_case(spec)
    res = run_case(spec, order=order)
    assert res["hv_relerr"] == ref["hv_relerr"] and res["lanczos_dalpha"] == ref["lanczos_dalpha"]


@pytest.mark.parametrize("spec", [
    {"wl": "ring12j", "n_up": 6, "mode": "cr", "prec": "fp64", "options": [["kernel", 1]], "batch": [5, 4], "steps": 6},
    {"wl": "ring16", "n_up": 15, "mode": "clt", "prec": "fp32", "options": [["kernel", 1]], "batch": [4, 4], "steps": 16},   # D = 16: breakdown at step 9
    {"wl": "ring14j", "n_up": 7, "mode": "clt", "prec": "fp32", "options": [["tml_split", 5 | (4 << 8)], ["kernel", 3]], "batch": [5, 4], "steps": 5},
    # multi-pass step: TML in-tile pass + PASS-B windows on rows of B interleaved chains (remainder groups run B = 1
    # on the same window geometry: option "plan_batch")
    {"wl": "ring14j", "n_up": 7, "mode": "cr", "prec": "fp32", "options": [["passb", 1], ["passb_lo_min", 4], ["tml_split", 5 | (3 << 8)], ["kernel", 3]], "batch": [5, 4], "steps": 5},
    {"wl": "rand13_30_5", "n_up": 6, "mode": "cr", "prec": "fp64",
     "options": [["passb", 1], ["passb_lo_min", 3], ["passb_smax", 6], ["tml_split", 5 | (2 << 8)], ["kernel", 3]], "batch": [3, 2], "steps": 4},
])
def test_emu_batched_chains_are_bit_identical_to_single_chains(spec):
    """SURVEY 8(f)-1, PAPER.md L207 / L309: R chains advanced in groups of B on interleaved vectors through
    ftlm_lanczos (ROW and TML kernels): alpha, beta, m_eff, theta, weight of every chain bit-identical to the same
    chain run alone with the same kernel and split, and the first coefficients equal to the oracle's."""
    res = run_case(dict(spec, what=[]))
    assert res["batch_identical"] and len(res["batch_m_eff"]) == spec["batch"][0]
    if spec["wl"] == "ring16":
        assert max(res["batch_m_eff"]) < 16              # the Krylov space of this sector is exhausted early (reading 10)


@pytest.mark.parametrize("n_up,mode,prec,opts", [
    (3, "clt", "fp32", [["kernel", 1]]),
    (5, "cr", "fp64", [["tml_split", 7 | (6 << 8)], ["passb", 1], ["passb_lo_min", 6], ["kernel", 3]]),
])
def test_emu_dodecahedron(n_up, mode, prec, opts):
    """SURVEY 8(f)-2 (Fig. 3 e-f): sectors of the N = 20 dodecahedron through the ROW kernel, the TML
    kernel and TML + windows: neighbour indices bit-exact, H.v and the first Lanczos coefficients against the oracle."""
    run_case({"wl": "dodecahedron", "n_up": n_up, "mode": mode, "prec": prec, "options": opts,
              "what": ["neighbors", "apply", "lanczos"], "steps": 6}, timeout=1200)


def test_emu_lin_two_table_index_mode():
    """index_mode LIN through the emulated kernels: ftlm_index_of on EVERY label of the
    full space (in-sector: the oracle's sorted-search index, else -1), ftlm_state_of round trip, neighbour lists, H.v,
    Lanczos and batched chains on small sectors; N = 34 (64-bit labels, dim > 2^31) on sampled labels against Alg. 1."""
    for spec in ({"wl": "ring12j", "n_up": 6, "mode": "lin", "prec": "fp64", "what": ["neighbors", "apply", "lanczos"]},
                 {"wl": "rand15_40_5", "n_up": 7, "mode": "lin", "prec": "fp32", "what": ["neighbors", "apply", "lanczos"], "batch": [3, 2]}):
        res = run_case(spec)
        assert res["kernel"] == K["row"]
    code = ("import sys, json; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
            "import numpy as np, emu_harness as E\n"
            "from oracle import ftlm_oracle as fo\n"
            "from paper_2605_26261_b200 import workloads as W\n"
            "bad = 0\n"
            "for N, n_up in ((11, 4), (12, 6), (9, 0), (9, 9)):\n"
            "    w = W.ring(N)\n"
            "    basis = fo.sector_basis(N, n_up)\n"
            "    lab = np.arange(1 << N, dtype=np.uint64)\n"
            "    with E.EmuCtx(w, n_up, 'lin', 'fp64') as c:\n"
            "        bad += int(np.count_nonzero(c.index_of(lab) != fo.index_of_sorted(basis, lab)))\n"
            "        bad += int(np.count_nonzero(c.state_of(np.arange(c.dim)) != basis))\n"
            "w = W.ring(34, 1.0, 0.5)\n"
            "rng = np.random.default_rng(3)\n"
            "_, Dc = fo.cr_tables(34)\n"
            "with E.EmuCtx(w, 17, 'lin', 'fp32') as c:\n"
            "    idx = np.concatenate([[0, c.dim - 1, 2**31 - 1, 2**31, 2**32 - 1 if c.dim > 2**32 else c.dim - 2], rng.integers(0, c.dim, 500)]).astype(np.int64)\n"
            "    lab = fo.alg1_unrank_vec(idx.astype(np.uint64), 34, 17, Dc)\n"
            "    bad += int(np.count_nonzero(c.index_of(lab) != idx))\n"
            "    out = rng.integers(0, 2**34, 200).astype(np.uint64)\n"
            "    exp = np.where(fo.popcount(out) == 17, fo.alg1_rank_vec(out, 34, 17, Dc).astype(np.int64), -1)\n"
            "    bad += int(np.count_nonzero(c.index_of(out) != exp))\n"
            "    nb = c.neighbors(int(idx[3]), 4)\n"
            "    bad += int((nb >= c.dim).sum())\n"
            "print(json.dumps({'bad': bad}))\n" % (ROOT, os.path.join(ROOT, "tests", "emu")))
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    assert json.loads(p.stdout.strip().splitlines()[-1])["bad"] == 0


def test_bench_candidates_are_valid_option_lists():
    """Every configuration bench.py can select (its CANDIDATES table = the names ftlm_autotune reports) must be a list of
    options the library accepts, on the bench sector itself (plans only; nothing is launched)."""
    code = ("import sys, json; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
            "import emu_harness as E, bench\n"
            "from paper_2605_26261_b200 import workloads as W\n"
            "w = W.baseline_config(4)\n"
            "out = {}\n"
            "with E.EmuCtx(w, w.sectors[0], 'cr', 'fp32') as c:\n"
            "    for name, opts in bench.CANDIDATES.items():\n"
            "        for k, v in opts:\n"
            "            c.set(k, v)\n"
            "        out[name] = [c.get('kernel'), c.get('passb_windows'), c.get('tmlr'), c.get('tmlr_available'), c.get('lazy_norm'), c.get('tml_m')]\n"
            "print(json.dumps(out))\n" % (ROOT, os.path.join(ROOT, "tests", "emu")))
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stderr[-2000:]
    d = json.loads(p.stdout.strip().splitlines()[-1])
    assert d["row"][0] == K["row"] and d["tml"][:2] == [K["tml"], 0]
    assert d["tml+passb"][:2] == [K["tml"], 2] and d["tmlr+passb"][:4] == [K["tml"], 2, 1, 1]
    assert d["tmlr+passb_lazy"][4] == 1 and d["tml"][4] == 0
    assert d["tml_w9m7"][5] == 7 and d["tml"][5] == 8 and d["tml_w9m7+passb"][1] >= 1
