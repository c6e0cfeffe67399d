"""CPU-only tests of the product's host logic and ABI surface: libftlm.so loads and exports
every symbol include/ftlm.h declares, argument validation, the tridiagonal eigensolver and the
trace assembly against the oracle.  No GPU compute calls."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import ftlm_oracle as fo
from paper_2605_26261_b200 import ftlm
from paper_2605_26261_b200 import build as ftlm_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    ftlm_build.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "ftlm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ftlm_[a-z_A-Z0-9]+)\s*\(", hdr))
    assert declared == set(ftlm.EXPORTS)
    L = ftlm.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert "sm_100a" in ftlm.ftlm_version()


def test_checked_library_exports_the_same_symbols():
    """libftlm_checked.so (the range-checked build of the same sources: -m gpu pre-flight, bench.py probe, smoke()) exports
    every declared symbol too and says what it is; it is only inspected here (the binding loads it with FTLM_CHECKED=1)."""
    import ctypes
    so = os.path.join(ROOT, "paper_2605_26261_b200", "libftlm_checked.so")
    if not os.path.exists(so) or ftlm_build.stale(so):
        pytest.skip("libftlm_checked.so not built (python -m paper_2605_26261_b200.build --checked; __graft_entry__.build() builds it)")
    L = ctypes.CDLL(so)
    for name in ftlm.EXPORTS:
        assert hasattr(L, name), name
    L.ftlm_version.restype = ctypes.c_char_p
    assert b"CHECKED" in L.ftlm_version()
    L.ftlm_get_option.restype = ctypes.c_int64
    assert L.ftlm_get_option(None, b"check_build") == 1


def test_create_validates_arguments_before_touching_the_device():
    for kw, code in [
        (dict(N=0, bond_i=[], bond_j=[], J=[], N_up=0), ftlm.EINVAL),
        (dict(N=63, bond_i=[], bond_j=[], J=[], N_up=1), ftlm.EINVAL),
        (dict(N=4, bond_i=[0], bond_j=[0], J=[1.0], N_up=2), ftlm.EINVAL),       # i == j
        (dict(N=4, bond_i=[0], bond_j=[4], J=[1.0], N_up=2), ftlm.EINVAL),       # site out of range
        (dict(N=4, bond_i=[0], bond_j=[1], J=[1.0], N_up=5), ftlm.EINVAL),
        (dict(N=34, bond_i=[0], bond_j=[1], J=[1.0], N_up=17, index_mode=ftlm.INDEX_CLT), ftlm.EUNSUPPORTED),
        (dict(N=4, bond_i=[0], bond_j=[1], J=[1.0], N_up=2, index_mode=7), ftlm.EINVAL),
        (dict(N=4, bond_i=[0], bond_j=[1], J=[1.0], N_up=2, precision=3), ftlm.EINVAL),
    ]:
        with pytest.raises(ftlm.FtlmError) as ei:
            ftlm.ftlm_create(**kw)
        assert ei.value.code == code, kw


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(ftlm.FtlmError) as ei:
        ftlm.ftlm_create(4, [0], [1], [1.0], 2)
    assert ei.value.code == ftlm.ECUDA and "no CPU path" in str(ei.value)


@pytest.mark.parametrize("m", [1, 2, 3, 17, 60, 100, 300])
def test_tridiag_eig_matches_dense_eigh(m):
    rng = np.random.default_rng(m)
    a = rng.standard_normal(m) * 3
    b = np.abs(rng.standard_normal(max(m - 1, 0))) + 0.01
    th, w = ftlm.ftlm_tridiag_eig(a, b)
    th2, w2 = fo.ritz(a, b)
    assert np.abs(th - th2).max() < 1e-12 * max(1.0, np.abs(th2).max())
    assert abs(w.sum() - 1.0) < 1e-12
    # weights of well separated eigenvalues agree; clusters agree in sum (L270)
    assert np.abs(np.cumsum(w) - np.cumsum(w2)).max() < 1e-9


def test_tridiag_eig_on_real_lanczos_coefficients_with_ghosts():
    from paper_2605_26261_b200 import workloads as W
    w_ = W.ring(12)
    basis = fo.sector_basis(12, 6)
    mv = lambda x: fo.apply_H(basis, 12, w_.bond_i, w_.bond_j, w_.J, 0.0, 6, x)
    a, b = fo.lanczos(mv, fo.start_vector(3, 6, 0, basis.shape[0]), 150)    # many ghosts by step 150
    th, w = ftlm.ftlm_tridiag_eig(a, b)
    th2, w2 = fo.ritz(a, b)
    assert np.abs(th - th2).max() < 1e-11
    T = np.array([0.05, 0.5, 5.0])
    for p in (0, 1, 2):   # the thermal sums are what must agree (Eqs. 4-5)
        s1 = (w[None] * th[None] ** p * np.exp(-(th[None] - th2[0]) / T[:, None])).sum(1)
        s2 = (w2[None] * th2[None] ** p * np.exp(-(th2[None] - th2[0]) / T[:, None])).sum(1)
        assert np.abs(s1 - s2).max() < 1e-10 * np.abs(s2).max()


def test_thermo_matches_oracle_assembly():
    rng = np.random.default_rng(8)
    secs, dims, Mzs, mults, Rs, m_eff, TH, WW = [], [], [], [], [], [], [], []
    stride = 12
    for s, (dim, Mz, R) in enumerate([(70, 0.0, 3), (56, 1.0, 2), (28, 2.0, 4), (1, 4.0, 1)]):
        chains = []
        for r in range(R):
            m = int(rng.integers(1, stride + 1)) if dim > 1 else 1
            th = np.sort(rng.uniform(-7.0, 3.0, m))
            w = rng.uniform(0, 1, m)
            w /= w.sum()
            chains.append((th, w))
            row_t, row_w = np.zeros(stride), np.zeros(stride)
            row_t[:m], row_w[:m] = th, w
            TH.append(row_t); WW.append(row_w); m_eff.append(m)
        secs.append(dict(dim=dim, Mz=Mz, mult=1 if Mz == 0 else 2, chains=chains))
        dims.append(dim); Mzs.append(Mz); mults.append(1 if Mz == 0 else 2); Rs.append(R)
    T = np.geomspace(0.05, 10, 40)
    ref = fo.thermo(secs, T)
    got = ftlm.ftlm_thermo(dims, Mzs, mults, Rs, m_eff, np.array(TH), np.array(WW), T)
    assert got["E_ref"] == ref["E_ref"]
    for k in ("Zs", "E", "C", "chi"):
        scale = np.maximum(np.abs(ref[k]), 1e-3 * np.abs(ref[k]).max())
        assert (np.abs(got[k] - ref[k]) / scale).max() < 1e-9, k


def test_thermo_rejects_bad_input():
    with pytest.raises(ftlm.FtlmError):
        ftlm.ftlm_thermo([4], [0.0], [1], [1], [1], np.zeros((1, 3)), np.ones((1, 3)), np.array([0.0]))
