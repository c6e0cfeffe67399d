"""-m gpu parity of the PASS-B window passes and of ftlm_autotune against the FP64
oracle.  These kernels were developed while the GPU pool was closed to this repository and are verified
in host emulation (tests/test_emu_kernels.py); on a GPU each case runs in its own process (tests/gpu_case.py)
and this file sorts last, so that the device-verified cases of test_gpu_parity.py always run first."""
import json
import os
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(spec, timeout=1800):
    p = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "gpu_case.py"), json.dumps(spec)],
                       capture_output=True, text=True, timeout=timeout)
    assert p.returncode == 0, (p.stdout[-1500:], p.stderr[-3000:])
    d = json.loads(p.stdout.strip().splitlines()[-1])
    assert d["ok"], d
    return d


@pytest.mark.parametrize("wl,n_up,mode,prec,opts,nwin", [
    ("ring16j", 8, "cr", "fp64", [["passb", 1], ["passb_lo_min", 4], ["tml_split", 5 | (3 << 8)]], 1),
    ("rand15_40_5", 7, "clt", "fp64", [["passb", 1], ["passb_lo_min", 3], ["passb_smax", 6], ["tml_split", 5 | (2 << 8)]], 2),
    ("rand15_40_5", 6, "cr", "fp32", [["passb", 1], ["passb_lo_min", 5], ["passb_smax", 5], ["passb_ctas", 1], ["tml_split", 5 | (2 << 8)]], 2),
    ("ring20j", 10, "clt", "fp32", [["passb", 1], ["passb_lo_min", 4], ["passb_smax", 7], ["tml_split", 5 | (1 << 8)]], 2),
    ("ring22j", 11, "cr", "fp32", [["passb", 1]], 1),
    ("tri4x5", 10, "clt", "fp32", [["passb", 1]], 1),
    ("square4x6", 12, "clt", "fp32", [["passb", 1]], 1),
    ("square4x6", 12, "cr", "fp64", [["passb", 1]], 1),
])
def test_windows_match_oracle(wl, n_up, mode, prec, opts, nwin):
    d = run({"wl": wl, "n_up": n_up, "mode": mode, "prec": prec, "options": opts + [["kernel", 3]],
             "what": (["neighbors"] if wl not in ("ring22j", "square4x6") else []) + ["apply", "lanczos"], "steps": 8})
    assert d["kernel"] == 3 and d["windows"] >= nwin, d


@pytest.mark.parametrize("wl,n_up,mode,prec,opts", [
    ("fring16j", 8, "cr", "fp32", [["passb", 1], ["passb_lo_min", 4], ["tml_split", 5 | (3 << 8)]]),
    ("fring14j", 7, "clt", "fp64", [["passb", 1], ["passb_lo_min", 4], ["tml_split", 5 | (3 << 8)]]),
    ("fring22j", 11, "clt", "fp32", [["passb", 1]]),
    ("fring24j", 12, "cr", "fp32", [["passb", 1]]),
])
@pytest.mark.parametrize("lazy", [0, 1])
def test_tmlr_in_tile_pass_matches_oracle(wl, n_up, mode, prec, opts, lazy):
    d = run({"wl": wl, "n_up": n_up, "mode": mode, "prec": prec,
             "options": opts + [["kernel", 3], ["tmlr", 1], ["lazy_norm", lazy]],
             "what": ["apply", "lanczos"], "steps": 8})
    assert d["kernel"] == 3 and d["tmlr"] == [1, 1], d


@pytest.mark.parametrize("cfg,mode", [(3, "clt"), (3, "cr")])
def test_autotune_config3(cfg, mode):
    d = run({"config": cfg, "mode": mode, "autotune": True, "options": [["allow_unverified", 1]],
             "what": ["sampled"], "blocks": 4})
    assert any(r["name"].startswith("tml+passb") for r in d["autotune"]), d


@pytest.mark.slow
@pytest.mark.parametrize("mode", ["clt", "cr"])
def test_autotune_config4_full_size_sampled_rows(mode):
    """BASELINE config 4 in the configuration bench.py times (ftlm_autotune's choice): every candidate must
    agree with the ROW kernel on the whole vector, and the chosen one with the oracle on sampled row blocks."""
    d = run({"config": 4, "mode": mode, "autotune": True, "options": [["allow_unverified", 1]],
             "what": ["sampled"], "blocks": 6}, timeout=3000)
    assert d["dim"] == 155117520 and d["hv_relerr"] <= 1e-5
