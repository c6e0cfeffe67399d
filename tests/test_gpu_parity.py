"""-m gpu parity tests: the CUDA path (through the C ABI) against the FP64 oracle on the same
seeded inputs.  Bars (BASELINE.json): indices bit-exact for CLT and CR; H.v norm-relative error
<= 1e-5 (FP32 mode) / 1e-12 (FP64 mode); C(T), chi(T) <= 1e-4 relative (reading 28)."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import ftlm_oracle as fo           # noqa: E402
from oracle import c_oracle as co              # noqa: E402
from paper_2605_26261_b200 import ftlm         # noqa: E402
from paper_2605_26261_b200 import workloads as W   # noqa: E402
from gpu_util import Ctx, HV_TOL, NDT, hv_err, relerr  # noqa: E402

KERNELS = [ftlm.KERNEL_ROW, ftlm.KERNEL_TML]


def _kernel_ok(c, kernel):
    try:
        ftlm.ftlm_set_option(c.ctx, "kernel", kernel)
    except ftlm.FtlmError as e:
        if e.code == ftlm.EUNSUPPORTED:
            return False
        raise
    return True


# ---------------------------------------------------------------- checked build (csrc/ftlm_access.cuh)

def test_checked_build_suppresses_and_counts_bad_accesses():
    """The range-checked build must catch (and suppress, without a device fault) five deliberately bad accesses:
    global load / store out of range, misaligned global load, shared load out of the window, cp.async from a bad
    source - and leave the violation counter as it found it.  Runs in a child process with FTLM_CHECKED=1."""
    import os
    import subprocess
    import sys
    from paper_2605_26261_b200 import build
    build.build(checked=True)
    code = ("import torch; torch.cuda.init(); from paper_2605_26261_b200 import ftlm; "
            "print(ftlm.ftlm_check_selftest(), ftlm.ftlm_check_info()['check_violations'], ftlm.ftlm_version())")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    p = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, FTLM_CHECKED="1"),
                       capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    caught, left, version = p.stdout.strip().splitlines()[-1].split(None, 2)
    assert int(caught) == 5 and int(left) == 0 and "CHECKED" in version, p.stdout


# ---------------------------------------------------------------- index maps (bit-exact)

@pytest.mark.parametrize("mode", ["clt", "cr"])
@pytest.mark.parametrize("N,n_up", [(14, 5), (14, 7), (9, 0), (9, 9), (3, 1), (1, 0), (1, 1), (20, 10)])
def test_index_of_and_state_of_every_label(mode, N, n_up):
    w = W.ring(N) if N >= 2 else W._mk("one", 1, [])
    with Ctx(w, n_up, mode, "fp32") as c:
        assert c.dim == math.comb(N, n_up)
        labels = np.arange(2 ** N, dtype=np.uint64)
        basis = fo.sector_basis(N, n_up)
        expect = fo.index_of_sorted(basis, labels)
        got = c.index_of(labels)
        assert (got == expect).all()
        st = c.state_of(np.arange(c.dim, dtype=np.int64))
        assert (st == basis).all()
        # labels beyond 2^N and indices outside [0, dim)
        assert (c.index_of(np.array([2 ** N, 2 ** N + 1, 2 ** 40 + 3], dtype=np.uint64)) == -1).all()
        bad = c.state_of(np.array([-1, c.dim], dtype=np.int64))
        assert (bad == np.uint64(2 ** 64 - 1)).all()


def test_clt_table_equals_paper_construction():
    w = W.ring(16)
    for n_up in (8, 3, 16):
        with Ctx(w, n_up, "clt", "fp32") as c:
            M, Cb = fo.clt_build(fo.sector_basis(16, n_up), 16)
            m, cnt = ftlm.ftlm_clt_read(c.ctx, 0, M.shape[0])
            assert (m == M).all() and (cnt.astype(np.int64) == Cb).all()
            assert ftlm.ftlm_table_bytes(c.ctx) >= fo.clt_bytes(16)


@pytest.mark.parametrize("N,n_up", [(34, 17), (36, 18), (40, 3), (33, 16), (62, 2)])
def test_cr_index_maps_beyond_32_bits(N, n_up):
    # sampled labels; expected values from the counting definition (Python ints)
    w = W.ring(N)
    rng = np.random.default_rng(N)
    D = math.comb(N, n_up)
    rows = [0, 1, D - 1, D - 2] + [int(x) for x in rng.integers(0, D, size=300, dtype=np.int64 if D < 2 ** 63 else None)]
    labels = [fo.unrank_by_counting(t, N, n_up) for t in rows]
    with Ctx(w, n_up, "cr", "fp32") as c:
        assert c.dim == D
        got_lab = c.state_of(np.array(rows, dtype=np.int64))
        assert [int(x) for x in got_lab] == labels
        got_idx = c.index_of(np.array(labels, dtype=np.uint64))
        assert [int(x) for x in got_idx] == rows
        off = np.array([labels[0] ^ 1, labels[5] | (1 << (N - 1)) | 1, (1 << N) - 1], dtype=np.uint64)
        exp = [fo.rank_by_counting(int(x), N, n_up) for x in off]
        assert [int(x) for x in c.index_of(off)] == exp


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("mode", ["clt", "cr"])
@pytest.mark.parametrize("wl,n_up", [("ring12j", 6), ("square4x4", 8), ("square4x4", 5), ("tri3x4", 6),
                                     ("icosa", 6), ("ring16", 15), ("ring16", 8), ("ring20j", 10)])
def test_neighbor_indices_bit_exact(kernel, mode, wl, n_up):
    w = {"ring12j": W.ring(12, 1.0, 0.5), "square4x4": W.square(4, 4), "tri3x4": W.triangular(3, 4),
         "icosa": W.icosahedron(), "ring16": W.ring(16), "ring20j": W.ring(20, 1.0, 0.5)}[wl]
    basis = co.enumerate_basis(w.N, n_up)
    with Ctx(w, n_up, mode, "fp32") as c:
        if not _kernel_ok(c, kernel):
            pytest.skip("kernel variant unavailable for this sector")
        D = c.dim
        for row0, nrows in ((0, min(D, 5000)), (max(0, D - 777), min(D, 777)), (D // 3, min(D - D // 3, 1031))):
            got = c.neighbors(row0, nrows)
            exp = co.neighbors_rows(w.N, w.bond_i, w.bond_j, basis, np.arange(row0, row0 + nrows))
            assert (got == exp).all()


def test_neighbors_sampled_rows_N34_cr():
    # config 5 sector (D = 2 333 606 220 > 2^31): sampled rows against the counting definition
    w = W.baseline_config(5)
    N, n_up = 34, 17
    D = math.comb(N, n_up)
    rng = np.random.default_rng(34)
    with Ctx(w, n_up, "cr", "fp32") as c:
        for row0 in [0, D - 64, 2 ** 31 - 32, 2 ** 31 + 5] + [int(x) for x in rng.integers(0, D - 64, size=6)]:
            got = c.neighbors(row0, 64)
            for r in range(0, 64, 7):
                n = fo.unrank_by_counting(row0 + r, N, n_up)
                for b in range(w.n_bonds):
                    i, j = int(w.bond_i[b]), int(w.bond_j[b])
                    anti = ((n >> i) & 1) != ((n >> j) & 1)
                    exp = fo.rank_by_counting(n ^ (1 << i) ^ (1 << j), N, n_up) if anti else -1
                    assert int(got[r, b]) == exp


# ---------------------------------------------------------------- H.v

def _hv_case(w, n_up, mode, prec, kernel, h=0.0, J=None, seed=0):
    J = w.J if J is None else J
    basis = co.enumerate_basis(w.N, n_up)
    rng = np.random.default_rng(seed)
    v = rng.standard_normal(basis.shape[0]).astype(NDT[prec])
    with Ctx(w, n_up, mode, prec, h=h, J=J) as c:
        if not _kernel_ok(c, kernel):
            pytest.skip("kernel variant unavailable for this sector")
        y = c.apply(v)
    ref = co.apply_rows(w.N, w.bond_i, w.bond_j, J, h, n_up, basis, v.astype(np.float64))
    return hv_err(y, ref, v, J, h, w.N, prec)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("prec", ["fp32", "fp64"])
@pytest.mark.parametrize("mode", ["clt", "cr"])
@pytest.mark.parametrize("n_up", [8, 9, 12, 14, 15, 16, 0, 1])
def test_apply_H_config1_sectors(kernel, prec, mode, n_up):
    assert _hv_case(W.baseline_config(1), n_up, mode, prec, kernel) <= HV_TOL[prec]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("prec", ["fp32", "fp64"])
@pytest.mark.parametrize("mode", ["clt", "cr"])
def test_apply_H_random_bonds_zeeman_duplicates(kernel, prec, mode):
    rng = np.random.default_rng(1)
    N = 13
    pairs = [(a, b) for a in range(N) for b in range(a + 1, N) if rng.random() < 0.4] + [(0, 1), (0, 1), (12, 0)]
    w = W._mk("rand13", N, pairs, rng.uniform(-1.0, 1.5, len(pairs)))
    for n_up in (6, 7, 2, 11):
        assert _hv_case(w, n_up, mode, prec, kernel, h=0.37) <= HV_TOL[prec]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("mode", ["clt", "cr"])
@pytest.mark.parametrize("wl,n_up", [("square4x5", 10), ("tri4x5", 9), ("ring22j", 11), ("ring21", 4)])
def test_apply_H_medium_lattices_fp32(kernel, mode, wl, n_up):
    w = {"square4x5": W.square(4, 5), "tri4x5": W.triangular(4, 5), "ring22j": W.ring(22, 1.0, 0.5),
         "ring21": W.ring(21)}[wl]
    assert _hv_case(w, n_up, mode, "fp32", kernel) <= HV_TOL["fp32"]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("mode,prec", [("clt", "fp32"), ("cr", "fp32"), ("cr", "fp64")])
def test_apply_H_config2_full_vector(kernel, mode, prec):
    # 4x6 square lattice, S^z = 0, D = 2 704 156: whole vector against the C oracle
    assert _hv_case(W.baseline_config(2), 12, mode, prec, kernel) <= HV_TOL[prec]


def test_apply_H_no_bonds_and_one_dimensional_sectors():
    w0 = W._mk("nobonds", 5, [])
    with Ctx(w0, 2, "cr", "fp64", h=0.5) as c:
        v = np.arange(1.0, c.dim + 1)
        assert np.allclose(c.apply(v), -0.5 * (2 - 2.5) * v)
    w = W.ring(16)
    for n_up, mode in ((16, "clt"), (0, "cr")):
        with Ctx(w, n_up, mode, "fp32") as c:
            assert c.dim == 1
            assert c.apply(np.array([2.0]))[0] == pytest.approx(8.0)     # N_B J / 4 = 4


def test_apply_H_rejects_aliasing_and_host_variant_matches():
    w = W.ring(12)
    with Ctx(w, 6, "clt", "fp32") as c:
        v = torch.zeros(c.dim, device="cuda")
        with pytest.raises(ftlm.FtlmError):
            ftlm.ftlm_apply_H(c.ctx, v, v)
        hv = np.random.default_rng(0).standard_normal(c.dim).astype(np.float32)
        hy = np.empty_like(hv)
        ftlm.ftlm_apply_H_host(c.ctx, hv, hy)
        assert np.array_equal(hy, c.apply(hv))


# ---------------------------------------------------------------- start vectors

@pytest.mark.parametrize("prec", ["fp32", "fp64"])
def test_fill_random_matches_specified_generator(prec):
    w = W.ring(16)
    for n_up, r in ((8, 0), (8, 7), (11, 2)):
        with Ctx(w, n_up, "cr", prec) as c:
            v = c.fill_random(W.SEED_VECTORS, r).cpu().numpy().astype(np.float64)
            ref = fo.start_vector(W.SEED_VECTORS, n_up, r, c.dim)
            tol = 2e-7 if prec == "fp32" else 1e-14
            assert np.abs(v - ref).max() <= tol * np.abs(ref).max()
            assert abs(np.dot(v, v) - 1.0) < (1e-6 if prec == "fp32" else 1e-13)


# ---------------------------------------------------------------- fused Lanczos

@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("mode", ["clt", "cr"])
def test_lanczos_fp64_coefficients_match_oracle(kernel, mode):
    w = W.ring(14, 1.0, 0.5)
    n_up = 7
    basis = co.enumerate_basis(14, n_up)
    with Ctx(w, n_up, mode, "fp64") as c:
        if not _kernel_ok(c, kernel):
            pytest.skip("kernel variant unavailable")
        out = ftlm.ftlm_lanczos(c.ctx, 77, 2, 40)
    for r in range(2):
        q1 = fo.start_vector(77, n_up, r, basis.shape[0])
        a, b = co.lanczos(14, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, q1, 40)
        assert out["m_eff"][r] == 40
        # early coefficients agree tightly; later ones drift as Ritz values converge (reading 27)
        assert np.abs(out["alpha"][r][:12] - a[:12]).max() < 1e-9
        assert np.abs(out["beta"][r][:11] - b[:11]).max() < 1e-9
        th, wk = fo.ritz(a, b)
        assert abs(out["theta"][r][0] - th[0]) < 1e-9 and abs(out["theta"][r][39] - th[-1]) < 1e-8
        assert abs(out["weight"][r].sum() - 1.0) < 1e-12


def test_lanczos_fp32_extremal_ritz_values_and_sum_rule():
    w = W.ring(16)
    basis = co.enumerate_basis(16, 8)
    with Ctx(w, 8, "clt", "fp32") as c:
        out = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, 2, 60)
    for r in range(2):
        q1 = fo.start_vector(W.SEED_VECTORS, 8, r, basis.shape[0])
        a, b = co.lanczos(16, w.bond_i, w.bond_j, w.J, 0.0, 8, basis, q1, 60)
        th, _ = fo.ritz(a, b)
        assert abs(out["theta"][r][0] - th[0]) < 2e-5            # single-precision round-off (L217)
        assert abs(out["alpha"][r][0] - a[0]) < 1e-5
        assert abs(out["weight"][r].sum() - 1.0) < 1e-12
        assert out["theta"][r][: out["m_eff"][r]].max() <= 4.0 + 1e-4      # sum_b J_b / 4


def test_lanczos_breakdown_small_sectors():
    w = W.ring(16)
    for prec in ("fp32", "fp64"):
        with Ctx(w, 16, "cr", prec) as c:                       # D = 1
            out = ftlm.ftlm_lanczos(c.ctx, 1, 1, 60)
            assert out["m_eff"][0] == 1 and out["alpha"][0][0] == pytest.approx(4.0)
        with Ctx(w, 15, "clt", prec) as c:                      # D = 16, 9 distinct eigenvalues
            out = ftlm.ftlm_lanczos(c.ctx, 1, 3, 60)
            assert (out["m_eff"] <= 16).all() and (out["m_eff"] >= 9).all()
            if prec == "fp64":
                assert (out["m_eff"] == 9).all()
            for r in range(3):
                m = out["m_eff"][r]
                assert abs(out["weight"][r][:m].sum() - 1.0) < 1e-12


def test_lanczos_host_start_vectors_and_chain_api():
    w = W.ring(14)
    n_up = 7
    basis = co.enumerate_basis(14, n_up)
    D = basis.shape[0]
    rng = np.random.default_rng(3)
    q = rng.standard_normal((2, D))
    with Ctx(w, n_up, "cr", "fp64") as c:
        out = ftlm.ftlm_lanczos_host(c.ctx, np.ascontiguousarray(q), 25)
        # same through the chain API with a device start vector, in two batches of steps
        dq = torch.from_numpy(q[1]).cuda()
        ftlm.ftlm_chain_begin(c.ctx, dq, 0, 0)
        ftlm.ftlm_chain_steps(c.ctx, 10)
        ftlm.ftlm_chain_steps(c.ctx, 15)
        a2, b2, m2 = ftlm.ftlm_chain_end(c.ctx)
    assert m2 == 25 and np.array_equal(a2, out["alpha"][1][:25])
    for r in range(2):
        a, b = co.lanczos(14, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, q[r] / np.linalg.norm(q[r]), 25)
        assert np.abs(out["alpha"][r][:10] - a[:10]).max() < 1e-9


# ---------------------------------------------------------------- thermodynamics end to end

def _gpu_ftlm(w, sectors, R, n_steps, seed, T, mode, prec, kernel=None):
    dims, Mz, mult, Rs, m_eff, TH, WW = [], [], [], [], [], [], []
    for n_up in sectors:
        with Ctx(w, n_up, mode, prec, kernel=kernel) as c:
            out = ftlm.ftlm_lanczos(c.ctx, seed, R, n_steps)
            dims.append(c.dim)
        mz = n_up - w.N / 2.0
        Mz.append(mz); mult.append(1 if mz == 0 else 2); Rs.append(R)
        m_eff += list(out["m_eff"]); TH.append(out["theta"]); WW.append(out["weight"])
    return ftlm.ftlm_thermo(dims, Mz, mult, Rs, m_eff, np.vstack(TH), np.vstack(WW), T)


def _max_rel(got, ref):
    scale = np.maximum(np.abs(ref), 1e-3 * np.abs(ref).max())       # reading 28
    return (np.abs(got - ref) / scale).max()


@pytest.mark.parametrize("mode,prec", [("clt", "fp32"), ("cr", "fp32"), ("clt", "fp64"), ("cr", "fp64")])
def test_thermodynamics_ring12_all_sectors_vs_oracle(mode, prec):
    w = W.ring(12)
    T = W.temperature_grid(60)
    R, n_steps, seed = 6, 50, W.SEED_VECTORS
    cast = np.float32 if prec == "fp32" else None
    ref, _, _ = fo.ftlm_run(12, w.bond_i, w.bond_j, w.J, 0.0, w.sectors, R, n_steps, seed, T,
                            tol=1e-12, cast=cast)
    got = _gpu_ftlm(w, w.sectors, R, n_steps, seed, T, mode, prec)
    tol = 1e-4 if prec == "fp32" else 1e-8
    assert _max_rel(got["C"], ref["C"]) <= tol
    assert _max_rel(got["chi"], ref["chi"]) <= tol
    assert _max_rel(got["E"], ref["E"]) <= tol


# ---------------------------------------------------------------- TML kernel: label splits

@pytest.mark.parametrize("prec", ["fp32", "fp64"])
@pytest.mark.parametrize("mode", ["clt", "cr"])
@pytest.mark.parametrize("w_bits,m_bits", [(5, 1), (6, 4), (8, 7), (9, 7), (9, 8), (10, 6), (12, 3), (7, 9), (5, 9)])
def test_tml_kernel_splits(prec, mode, w_bits, m_bits):
    # every LL/MM/ML/TT/TM/TL classification of the same bonds must give the same H.v and indices
    rng = np.random.default_rng(100 * w_bits + m_bits)
    w = W.triangular(4, 5)                       # N = 20, 60 bonds
    J = rng.uniform(0.5, 1.5, w.n_bonds)
    n_up = 9
    basis = co.enumerate_basis(w.N, n_up)
    v = rng.standard_normal(basis.shape[0]).astype(NDT[prec])
    ref = co.apply_rows(w.N, w.bond_i, w.bond_j, J, 0.21, n_up, basis, v.astype(np.float64))
    with Ctx(w, n_up, mode, prec, h=0.21, J=J) as c:
        try:
            ftlm.ftlm_set_option(c.ctx, "tml_low_bits", w_bits)
            ftlm.ftlm_set_option(c.ctx, "tml_mid_bits", m_bits)
        except ftlm.FtlmError as e:
            if e.code == ftlm.EUNSUPPORTED:
                pytest.skip("split does not fit shared memory / class caps")
            raise
        assert ftlm.ftlm_get_option(c.ctx, "tml_w") == w_bits and ftlm.ftlm_get_option(c.ctx, "tml_m") == m_bits
        ftlm.ftlm_set_option(c.ctx, "kernel", ftlm.KERNEL_TML)
        assert ftlm.ftlm_get_option(c.ctx, "kernel") == ftlm.KERNEL_TML
        assert hv_err(c.apply(v), ref, v, J, 0.21, w.N, prec) <= HV_TOL[prec]
        assert hv_err(c.apply(v), ref, v, J, 0.21, w.N, prec) <= HV_TOL[prec]          # second launch: counters were reset
        D = c.dim
        for row0, nrows in ((0, 3000), (D // 2, 3000), (D - 2000, 2000)):
            got = c.neighbors(row0, nrows)
            exp = co.neighbors_rows(w.N, w.bond_i, w.bond_j, basis, np.arange(row0, row0 + nrows))
            assert (got == exp).all()


def test_tml_lanczos_is_bit_reproducible_and_matches_row():
    # dynamic tile scheduling must not change alpha, beta run to run (per-tile partial sums added in
    # fixed order); TML and ROW agree to FP64 round-off in FP64 mode
    w = W.ring(22, 1.0, 0.5)
    n_up = 11
    outs = []
    with Ctx(w, n_up, "cr", "fp64") as c:
        for kern in (ftlm.KERNEL_TML, ftlm.KERNEL_TML, ftlm.KERNEL_ROW):
            ftlm.ftlm_set_option(c.ctx, "kernel", kern)
            outs.append(ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, 1, 40))
    assert (outs[0]["alpha"] == outs[1]["alpha"]).all() and (outs[0]["beta"] == outs[1]["beta"]).all()
    assert np.abs(outs[0]["alpha"][0, :10] - outs[2]["alpha"][0, :10]).max() < 1e-10
    assert abs(outs[0]["theta"][0, 0] - outs[2]["theta"][0, 0]) < 1e-9


def test_tml_and_row_kernels_agree_on_config3_slice_fp32():
    # 4x7 triangular lattice (N = 28, D = 40 116 600): ROW vs TML on the whole vector, and both
    # against the oracle on a slice of rows
    w = W.baseline_config(3)
    n_up = 14
    basis = co.enumerate_basis(w.N, n_up)
    outs = {}
    for mode in ("clt", "cr"):
        with Ctx(w, n_up, mode, "fp32") as c:
            v = c.fill_random(W.SEED_VECTORS, 0)
            for kern in (ftlm.KERNEL_ROW, ftlm.KERNEL_TML):
                ftlm.ftlm_set_option(c.ctx, "kernel", kern)
                y = torch.empty_like(v)
                ftlm.ftlm_apply_H(c.ctx, v, y)
                torch.cuda.synchronize()
                outs[(mode, kern)] = y.cpu().numpy()
            vh = v.cpu().numpy().astype(np.float64)
    D = basis.shape[0]
    for row0 in (0, D // 2 - 50000, D - 100000):
        ref = co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, vh, row0, 100000)
        for key, y in outs.items():
            assert hv_err(y[row0:row0 + 100000], ref, vh, w.J, 0.0, w.N, "fp32") <= HV_TOL["fp32"], key
    base = outs[("clt", ftlm.KERNEL_ROW)].astype(np.float64)
    for key, y in outs.items():
        assert relerr(y, base) <= 1e-6, key


# ---------------------------------------------------------------- full sizes in the checked build (sampled items)

@pytest.mark.parametrize("cfg,mode,tmlr", [(3, "clt", 1), (3, "cr", 0), (4, "clt", 1), (4, "cr", 0), (4, "clt", 0),
                                           (40, "cr", 1), (41, "clt", 0), (5, "cr", 1), (5, "cr", 0)])
def test_checked_full_size_sampled_items(cfg, mode, tmlr):
    """Only in the checked build (FTLM_CHECKED=1; tests/conftest.py runs the -m gpu selection there first): the first,
    last, middle and random tiles / window items of BASELINE configs 3, 4, 4b (40), 4 in lexicographic numbering (41)
    and 5 - real run starts, offsets and vector sizes, rows beyond 2^31 - one at a time through the in-tile pass (TML or
    TMLR) and every PASS-B window, against the oracle's sampled-row form, with zero suppressed accesses
    (tests/gpu_sampled.py).  This is what stands in for the `slow` whole-vector cases in the checked pre-flight."""
    import json
    import os
    import subprocess
    import sys
    if not ftlm.CHECKED:
        pytest.skip("checked build only (debug item hooks are not in the release ABI)")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    p = subprocess.run([sys.executable, os.path.join(root, "tests", "gpu_sampled.py"),
                        json.dumps({"config": cfg, "mode": mode, "tmlr": tmlr, "samples": 2})],
                       capture_output=True, text=True, timeout=1800)
    assert p.returncode == 0, (p.stdout[-1500:], p.stderr[-3000:])
    d = json.loads(p.stdout.strip().splitlines()[-1])
    assert d["ok"], d
    assert d["windows"] >= (1 if cfg != 41 else 0)
