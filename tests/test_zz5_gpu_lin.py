"""-m gpu parity of index_mode LIN (Lin's two half-system tables) against the oracle:
state -> index on every label (bit-exact, -1 outside the sector), neighbour lists, H.v in both precisions, the fused
Lanczos chain, and N = 34 with 64-bit labels and indices beyond 2^31."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import c_oracle as co              # noqa: E402
from oracle import ftlm_oracle as fo           # noqa: E402
from paper_2605_26261_b200 import ftlm         # noqa: E402
from paper_2605_26261_b200 import workloads as W   # noqa: E402
from gpu_util import Ctx, HV_TOL, NDT, hv_err  # noqa: E402


@pytest.mark.parametrize("N,n_up", [(14, 5), (14, 7), (9, 0), (9, 9), (3, 1), (1, 0), (1, 1), (20, 10)])
def test_lin_index_of_and_state_of_every_label(N, n_up):
    w = W.ring(max(N, 2)) if N > 1 else W._mk("one", 1, [])
    basis = co.enumerate_basis(N, n_up)
    lab = np.arange(1 << N, dtype=np.uint64)
    with Ctx(w, n_up, "lin", "fp32") as c:
        assert c.dim == math.comb(N, n_up)
        assert (c.index_of(lab) == fo.index_of_sorted(basis, lab)).all()
        assert (c.state_of(np.arange(c.dim)) == basis).all()
        assert ftlm.ftlm_get_option(c.ctx, "kernel") == ftlm.KERNEL_ROW
        h = N // 2
        assert ftlm.lib().ftlm_table_bytes(c.ctx) >= (8 << (N - h)) + (4 << h)


def test_lin_index_beyond_32_bits_sampled():
    N, n_up = 34, 17
    w = W.baseline_config(5)
    rng = np.random.default_rng(3)
    _, Dc = fo.cr_tables(N)
    with Ctx(w, n_up, "lin", "fp32") as c:
        idx = np.concatenate([[0, c.dim - 1, 2 ** 31 - 1, 2 ** 31, c.dim - 2], rng.integers(0, c.dim, 20000)]).astype(np.int64)
        lab = fo.alg1_unrank_vec(idx.astype(np.uint64), N, n_up, Dc)
        assert (c.index_of(lab) == idx).all() and (c.state_of(idx) == lab).all()
        out = rng.integers(0, 2 ** 34, 5000).astype(np.uint64)
        exp = np.where(fo.popcount(out) == n_up, fo.alg1_rank_vec(out, N, n_up, Dc).astype(np.int64), -1)
        assert (c.index_of(out) == exp).all()
        rows = np.array([0, 2 ** 31 - 2, c.dim - 3], dtype=np.int64)
        for r0 in rows:
            got = c.neighbors(int(r0), 3)
            labs = fo.alg1_unrank_vec(np.arange(r0, r0 + 3, dtype=np.uint64), N, n_up, Dc)
            for k in range(3):
                for b in range(w.n_bonds):
                    m = (1 << int(w.bond_i[b])) | (1 << int(w.bond_j[b]))
                    x = int(labs[k]) & m
                    e = -1 if x in (0, m) else fo.rank_by_counting(int(labs[k]) ^ m, N, n_up)
                    assert got[k, b] == e


@pytest.mark.parametrize("prec", ["fp32", "fp64"])
@pytest.mark.parametrize("wl,n_up", [("ring16", 8), ("ring16", 15), ("square4x5", 10), ("tri4x5", 9), ("square4x6", 12)])
def test_lin_apply_H_and_neighbors(wl, n_up, prec):
    from gpu_case import workload
    w = workload({"wl": wl})
    basis = co.enumerate_basis(w.N, n_up)
    rng = np.random.default_rng(17)
    v = rng.standard_normal(basis.shape[0]).astype(NDT[prec])
    ref = co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, v.astype(np.float64))
    with Ctx(w, n_up, "lin", prec) as c:
        assert hv_err(c.apply(v), ref, v, w.J, 0.0, w.N, prec) <= HV_TOL[prec]
        n = min(c.dim, 4000)
        got = c.neighbors(c.dim - n, n)
        exp = co.neighbors_rows(w.N, w.bond_i, w.bond_j, basis, np.arange(c.dim - n, c.dim))
        assert (got == exp).all()


@pytest.mark.parametrize("prec,batch", [("fp64", 1), ("fp32", 4)])
def test_lin_lanczos_matches_oracle(prec, batch):
    w = W.ring(14, 1.0, 0.5)
    n_up = 7
    basis = co.enumerate_basis(w.N, n_up)
    with Ctx(w, n_up, "lin", prec) as c:
        ftlm.ftlm_set_option(c.ctx, "batch", batch)
        out = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, 4, 20)
    tol = 1e-9 if prec == "fp64" else 2e-4
    for r in range(4):
        q1 = fo.start_vector(W.SEED_VECTORS, n_up, r, basis.shape[0])
        a, b = co.lanczos(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, q1, 20)[:2]
        assert np.abs(out["alpha"][r][:6] - np.asarray(a)[:6]).max() <= tol
        assert np.abs(out["beta"][r][:5] - np.asarray(b)[:5]).max() <= tol
        th, _ = fo.ritz(np.asarray(a), np.asarray(b))
        assert abs(out["theta"][r][0] - th[0]) <= (1e-8 if prec == "fp64" else 5e-4)


def test_lin_rejects_tml_kernel_and_large_N():
    w = W.ring(20)
    with Ctx(w, 10, "lin", "fp32") as c:
        with pytest.raises(ftlm.FtlmError) as e:
            ftlm.ftlm_set_option(c.ctx, "kernel", ftlm.KERNEL_TML)
        assert e.value.code == ftlm.EUNSUPPORTED
    with pytest.raises(ftlm.FtlmError) as e:
        ftlm.ftlm_create(50, [0], [1], [1.0], 25, ftlm.INDEX_LIN, ftlm.FP32)
    assert e.value.code == ftlm.EUNSUPPORTED
