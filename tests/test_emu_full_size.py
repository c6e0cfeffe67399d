"""Host emulation at BASELINE's full sizes on sampled tiles / items (tests/emu/run_sampled.py), beyond the routine
config-4 CLT case of tests/test_emu_kernels.py.  These take 2-6 minutes each (basis enumeration, 268 MB CLT) and
config 5 needs ~47 GB of host memory, so they run only with FTLM_EMU_FULL=1:

    FTLM_EMU_FULL=1 python -m pytest tests/test_emu_full_size.py -q            (config 5: FTLM_EMU_FULL=2)

Results of the last run on the build container are recorded in DESIGN.md section 13."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
LEVEL = int(os.environ.get("FTLM_EMU_FULL", "0") or 0)
pytestmark = pytest.mark.skipif(LEVEL < 1, reason="set FTLM_EMU_FULL=1 (2 for config 5) to run the full-size emulation cases")


def sampled(spec, timeout=5400):
    p = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "emu", "run_sampled.py"), json.dumps(spec)],
                       capture_output=True, text=True, timeout=timeout)
    assert p.returncode == 0, p.stderr[-2000:]
    d = json.loads(p.stdout.strip().splitlines()[-1])
    assert d["ok"] and all(x["ok"] for x in d["passes"]), d
    return d


@pytest.mark.parametrize("cfg,mode,opts,both", [
    (3, "clt", [["tmlr", 1]], True), (3, "cr", [["tmlr", 1]], True),
    (4, "cr", [["tmlr", 1]], True),
    (40, "cr", [["tmlr", 1]], True),                       # config 4b: random J_b (no uniform-J fast paths)
    (41, "clt", [], False),                                # lexicographic numbering: left-over bonds stay global gathers
    (4, "clt", [["tml_split", 9 | (7 << 8)]], False),      # the 16-bit tile measured in round 1, with windows
])
def test_emu_full_size_sampled(cfg, mode, opts, both):
    d = sampled({"config": cfg, "mode": mode, "samples": 1, "options": opts, "tmlr_both": both})
    assert d["kernel"] == 3 and d["windows"] >= (0 if cfg == 41 else 1)


@pytest.mark.skipif(LEVEL < 2, reason="config 5 needs ~47 GB of host memory: FTLM_EMU_FULL=2")
@pytest.mark.parametrize("opts", [[], [["tmlr", 1]]])
def test_emu_config5_full_size_sampled(opts):
    d = sampled({"config": 5, "mode": "cr", "samples": 1, "lowmem": True, "options": opts}, timeout=3 * 3600)
    assert d["dim"] == 2333606220 and d["windows"] >= 1


def test_emu_smoke_configurations():
    """The two multi-pass configurations __graft_entry__.smoke() runs on the device (folded N = 18 ring, D = 48 620):
    TMLR + window + lazy normalisation, and a batch of 4 chains through TML + window (bit-identical to single chains)."""
    run = os.path.join(ROOT, "tests", "emu", "run_case.py")
    for spec in ({"wl": "fring18j", "n_up": 9, "mode": "clt", "prec": "fp32", "what": ["apply", "lanczos"], "steps": 6,
                  "options": [["passb", 1], ["passb_lo_min", 5], ["tml_split", 6 | (4 << 8)], ["kernel", 3], ["tmlr", 1], ["lazy_norm", 1]]},
                 {"wl": "fring18j", "n_up": 9, "mode": "cr", "prec": "fp32", "what": [], "steps": 8, "batch": [4, 4],
                  "options": [["passb", 1], ["passb_lo_min", 5], ["tml_split", 6 | (4 << 8)], ["kernel", 3]]}):
        p = subprocess.run([sys.executable, run, json.dumps(spec)], capture_output=True, text=True, timeout=3600)
        assert p.returncode == 0, p.stderr[-2000:]
        d = json.loads(p.stdout.strip().splitlines()[-1])
        assert d["ok"] and d["passb"][0] >= 1, d
        if "batch" in spec:
            assert d["batch_identical"], d
