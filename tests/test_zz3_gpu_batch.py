"""-m gpu parity of the batched Lanczos chains (Table 3 footnote L325: B = 4 on the
paper's GPU): ftlm_lanczos with option "batch" = 2, 4 against the same chains run one at a time on the same tiles and windows (bit-identical: the
per-chain arithmetic and the reduction order do not depend on B) and against the FP64 oracle."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import c_oracle as co              # noqa: E402
from oracle import ftlm_oracle as fo           # noqa: E402
from paper_2605_26261_b200 import ftlm         # noqa: E402
from paper_2605_26261_b200 import workloads as W   # noqa: E402
from gpu_util import Ctx                       # noqa: E402


@pytest.mark.parametrize("wl,n_up,mode,prec,opts,R,B,steps", [
    ("ring12j", 6, "cr", "fp64", [["kernel", 1]], 5, 4, 12),
    ("ring16", 15, "clt", "fp32", [["kernel", 1]], 4, 4, 16),                  # D = 16: breakdown inside the batch
    ("ring16j", 8, "clt", "fp32", [["tml_split", 6 | (4 << 8)], ["kernel", 3]], 6, 4, 12),
    ("square4x5", 10, "cr", "fp64", [["tml_split", 7 | (5 << 8)], ["kernel", 3]], 3, 2, 10),
    ("square4x6", 12, "clt", "fp32", [["kernel", 3]], 4, 4, 8),                 # BASELINE config 2's largest sector, auto split
    ("square4x6", 12, "cr", "fp32", [["kernel", 3]], 2, 2, 8),
    # multi-pass step on rows of B chains: TML in-tile pass + PASS-B windows
    ("ring16j", 8, "clt", "fp32", [["passb", 1], ["tml_split", 5 | (3 << 8)], ["kernel", 3]], 5, 4, 12),
    ("rand15_40_5", 7, "cr", "fp64", [["passb", 1], ["passb_lo_min", 3], ["passb_smax", 6], ["tml_split", 5 | (2 << 8)], ["kernel", 3]], 3, 2, 10),
    ("ring20j", 10, "clt", "fp32", [["passb", 1], ["passb_lo_min", 4], ["passb_smax", 7], ["tml_split", 5 | (1 << 8)], ["kernel", 3]], 4, 4, 6),
    ("square4x6", 12, "clt", "fp32", [["passb", 1], ["kernel", 3]], 4, 4, 8),
])
def test_batched_chains_match_single_chains_and_oracle(wl, n_up, mode, prec, opts, R, B, steps):
    from gpu_case import workload
    w = workload({"wl": wl})
    basis = co.enumerate_basis(w.N, n_up)
    with Ctx(w, n_up, mode, prec) as c:
        ftlm.ftlm_set_option(c.ctx, "batch", B)          # first: the split is then one that holds B interleaved tiles
        for k, v in opts:
            ftlm.ftlm_set_option(c.ctx, k, v)
        many = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, R, steps)
        split = (ftlm.ftlm_get_option(c.ctx, "tml_w"), ftlm.ftlm_get_option(c.ctx, "tml_m"))
        if split[0] > 0:
            ftlm.ftlm_set_option(c.ctx, "tml_split", split[0] | (split[1] << 8))
        ftlm.ftlm_set_option(c.ctx, "plan_batch", B)      # the single chains run on the batch's tiles and windows
        ftlm.ftlm_set_option(c.ctx, "batch", 1)
        assert (ftlm.ftlm_get_option(c.ctx, "tml_w"), ftlm.ftlm_get_option(c.ctx, "tml_m")) == split
        one = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, R, steps)
    for key in ("alpha", "beta", "m_eff", "theta", "weight"):
        assert np.array_equal(one[key], many[key]), key
    tol = 1e-9 if prec == "fp64" else 2e-4
    for r in range(R):
        q1 = fo.start_vector(W.SEED_VECTORS, n_up, r, c.dim)
        a, b = co.lanczos(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, q1, min(steps, c.dim))[:2]
        k = min(int(many["m_eff"][r]), len(a), 6)
        assert np.abs(many["alpha"][r][:k] - np.asarray(a)[:k]).max() <= tol
        if k > 1:
            assert np.abs(many["beta"][r][:k - 1] - np.asarray(b)[:k - 1]).max() <= tol
        assert abs(many["weight"][r][: int(many["m_eff"][r])].sum() - 1.0) <= 1e-6
    if wl == "ring16":
        assert many["m_eff"].max() < 16
