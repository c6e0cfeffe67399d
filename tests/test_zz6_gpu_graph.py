"""-m gpu: option "graph" ("capture the step in a CUDA graph"): ftlm_chain_steps replays captured
steps; the kernels and their arithmetic are the same, so alpha, beta must be bit-identical with and without it, the
replays must really happen, and breakdown / chain limits must behave as with direct launches."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2605_26261_b200 import ftlm         # noqa: E402
from paper_2605_26261_b200 import workloads as W   # noqa: E402
from gpu_util import Ctx                       # noqa: E402


@pytest.mark.parametrize("wl,n_up,mode,prec,opts,steps", [
    (W.ring(16), 8, "clt", "fp32", [], 60),                                   # BASELINE config 1, largest sector (ROW)
    (W.ring(16), 8, "cr", "fp64", [["batch", 4]], 60),
    (W.ring(16), 15, "clt", "fp32", [], 16),                                  # D = 16: breakdown at step 9, limit 16
    (W.ring(16), 16, "cr", "fp32", [], 5),                                    # D = 1
    (W.square(4, 6), 12, "clt", "fp32", [["kernel", 3]], 21),                  # BASELINE config 2 (TML), odd step count
    (W.square(4, 6), 12, "cr", "fp32", [["passb", 1], ["kernel", 3], ["tmlr", 1], ["lazy_norm", 1]], 20),
])
def test_graph_replay_is_bit_identical(wl, n_up, mode, prec, opts, steps):
    res = []
    for graph in (0, 1):
        with Ctx(wl, n_up, mode, prec) as c:
            for k, v in opts:
                ftlm.ftlm_set_option(c.ctx, k, v)
            ftlm.ftlm_set_option(c.ctx, "graph", graph)
            out = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, 4, steps)
            launches = ftlm.ftlm_get_option(c.ctx, "graph_launches")
            failed = ftlm.ftlm_get_option(c.ctx, "graph_failed")
        res.append(out)
        if graph:
            assert failed == 0
            if min(steps, c.dim) >= 5:
                assert launches > 0
        else:
            assert launches == 0
    for key in ("alpha", "beta", "m_eff", "theta", "weight"):
        assert np.array_equal(res[0][key], res[1][key]), key


def test_graph_chain_api_in_pieces():
    """ftlm_chain_steps called with 1, 2, 3, 7 steps: replays and direct launches mix; same coefficients."""
    w = W.ring(16)
    outs = []
    for graph in (0, 1):
        with Ctx(w, 8, "clt", "fp32") as c:
            ftlm.ftlm_set_option(c.ctx, "graph", graph)
            ftlm.ftlm_chain_begin(c.ctx, None, W.SEED_VECTORS, 0)
            for n in (1, 2, 3, 7, 1, 6):
                ftlm.ftlm_chain_steps(c.ctx, n)
            outs.append(ftlm.ftlm_chain_end(c.ctx))
    assert outs[0][2] == outs[1][2] == 20
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
