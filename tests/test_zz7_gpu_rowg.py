"""-m gpu parity of kernel ROWG (north_star: "row bit-states by unranking plus Gosper-style successor enumeration";
PAPER.md L136 for the unrank): neighbour indices bit-exact, H.v and the fused chain against the FP64 oracle, in the three
index modes, both precisions, on degenerate sectors, at config 2's size and with 64-bit labels (N = 34)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import c_oracle as co              # noqa: E402
from oracle import ftlm_oracle as fo           # noqa: E402
from paper_2605_26261_b200 import ftlm         # noqa: E402
from paper_2605_26261_b200 import workloads as W   # noqa: E402
from gpu_util import Ctx, HV_TOL, NDT, hv_err  # noqa: E402


@pytest.mark.parametrize("prec", ["fp32", "fp64"])
@pytest.mark.parametrize("mode", ["clt", "cr", "lin"])
@pytest.mark.parametrize("wl,n_up", [("ring16", 8), ("ring16", 15), ("ring16", 16), ("ring16", 0), ("ring13", 5),
                                     ("tri4x5", 9), ("square4x6", 12)])
def test_rowg_apply_H_and_neighbors(wl, n_up, mode, prec):
    from gpu_case import workload
    w = workload({"wl": wl})
    basis = co.enumerate_basis(w.N, n_up)
    rng = np.random.default_rng(23)
    v = rng.standard_normal(basis.shape[0]).astype(NDT[prec])
    ref = co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v.astype(np.float64))
    with Ctx(w, n_up, mode, prec, kernel=ftlm.KERNEL_ROWG) as c:
        assert ftlm.ftlm_get_option(c.ctx, "kernel") == ftlm.KERNEL_ROWG
        assert hv_err(c.apply(v), ref, v, w.J, 0.0, w.N, prec) <= HV_TOL[prec]
        n = min(c.dim, 5003)                                   # not a multiple of 8: ragged last group
        got = c.neighbors(c.dim - n, n)
        exp = co.neighbors_rows(w.N, w.bond_i, w.bond_j, basis, np.arange(c.dim - n, c.dim))
        assert (got == exp).all()


@pytest.mark.parametrize("mode,prec", [("clt", "fp32"), ("cr", "fp64")])
def test_rowg_lanczos_matches_oracle(mode, prec):
    w = W.ring(14, 1.0, 0.5)
    basis = co.enumerate_basis(w.N, 7)
    with Ctx(w, 7, mode, prec, kernel=ftlm.KERNEL_ROWG) as c:
        out = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, 2, 25)
    tol = 1e-9 if prec == "fp64" else 2e-4
    for r in range(2):
        a, b = co.lanczos(w.N, w.bond_i, w.bond_j, w.J, 0.0, 7, basis, fo.start_vector(W.SEED_VECTORS, 7, r, basis.shape[0]), 25)[:2]
        assert np.abs(out["alpha"][r][:6] - np.asarray(a)[:6]).max() <= tol
        assert np.abs(out["beta"][r][:5] - np.asarray(b)[:5]).max() <= tol
        assert abs(out["weight"][r][: int(out["m_eff"][r])].sum() - 1.0) <= 1e-6


def test_rowg_64_bit_labels_sampled_rows():
    N, n_up = 34, 17
    w = W.baseline_config(5)
    _, Dc = fo.cr_tables(N)
    with Ctx(w, n_up, "cr", "fp32", kernel=ftlm.KERNEL_ROWG) as c:
        for r0 in (0, 2 ** 31 - 5, c.dim // 2 + 3, c.dim - 19):
            got = c.neighbors(int(r0), 19)
            lab = fo.alg1_unrank_vec(np.arange(r0, r0 + 19, dtype=np.uint64), N, n_up, Dc)
            for k in range(19):
                for b in range(w.n_bonds):
                    m = (1 << int(w.bond_i[b])) | (1 << int(w.bond_j[b]))
                    x = int(lab[k]) & m
                    assert got[k, b] == (-1 if x in (0, m) else fo.rank_by_counting(int(lab[k]) ^ m, N, n_up))
