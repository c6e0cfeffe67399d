"""Pins for the oracle's Lanczos (O3/O4), FTLM assembly (O5) and start-vector generator:
sum_k w_k = 1, alpha_1 = <r|H|r>, m = D reproduces the spectrum, FTLM with R = D unit starts
and N_L = D == exact Z, dimer closed forms for C(T) and chi(T), T -> infinity limits.  CPU only."""
import math

import numpy as np
import pytest

from oracle import ftlm_oracle as fo
from oracle import c_oracle as co
from paper_2605_26261_b200 import workloads as W


def _mv(w, basis, n_up, h=0.0):
    return lambda x: fo.apply_H(basis, w.N, w.bond_i, w.bond_j, w.J, h, n_up, x)


def test_weights_sum_to_one_and_alpha1_is_expectation_value():
    w = W.ring(12)
    basis = fo.sector_basis(12, 6)
    q1 = fo.start_vector(42, 6, 3, basis.shape[0])
    assert np.dot(q1, q1) == pytest.approx(1.0, abs=1e-14)
    a, b = fo.lanczos(_mv(w, basis, 6), q1, 60)
    assert len(a) == 60 and len(b) == 59
    th, wk = fo.ritz(a, b)
    assert wk.sum() == pytest.approx(1.0, abs=1e-13)        # L45 sum rule
    Hd = fo.dense_H(12, w.bond_i, w.bond_j, w.J, 0.0, 6)
    assert a[0] == pytest.approx(q1 @ Hd @ q1, abs=1e-13)
    ev = np.linalg.eigvalsh(Hd)
    assert th.min() >= ev[0] - 1e-10 and th.max() <= ev[-1] + 1e-10
    # second moment: <r|H^2|r> = alpha_1^2 + beta_1^2 (first two Lanczos steps, exact)
    assert a[0] ** 2 + b[0] ** 2 == pytest.approx(q1 @ Hd @ Hd @ q1, rel=1e-12)


def test_full_krylov_space_reproduces_spectrum_seen_by_start_vector():
    w = W.ring(6, 1.0, 0.3)
    basis = fo.sector_basis(6, 3)
    Hd = fo.dense_H(6, w.bond_i, w.bond_j, w.J, 0.0, 3)
    ev, U = np.linalg.eigh(Hd)
    q1 = fo.start_vector(7, 3, 0, 20)
    a, b = fo.lanczos(_mv(w, basis, 3), q1, 50)      # m = min(50, D) = 20 (reading 9) or breakdown
    th, wk = fo.ritz(a, b)
    # weight distribution: sum of w over a (possibly degenerate) level = |P_level q1|^2
    for lvl in np.unique(np.round(ev, 9)):
        proj = float(((U[:, np.abs(ev - lvl) < 1e-7].T @ q1) ** 2).sum())
        got = float(wk[np.abs(th - lvl) < 1e-6].sum())
        assert got == pytest.approx(proj, abs=1e-8)


def test_breakdown_rule_and_one_dimensional_sector():
    w = W.ring(16)
    # N_up = 16: D = 1 -> one step, alpha_1 = N_B J / 4
    basis = fo.sector_basis(16, 16)
    a, b = fo.lanczos(_mv(w, basis, 16), np.ones(1), 60)
    assert list(a) == [4.0] and len(b) == 0
    # N_up = 15: D = 16, only 9 distinct eigenvalues -> invariant subspace after 9 steps
    basis = fo.sector_basis(16, 15)
    a, b = fo.lanczos(_mv(w, basis, 15), fo.start_vector(1, 15, 0, 16), 60)
    assert len(a) == 9 and len(b) == 8
    th, wk = fo.ritz(a, b)
    assert wk.sum() == pytest.approx(1.0, abs=1e-13)


@pytest.mark.parametrize("N,n_up", [(8, 4), (10, 7)])
def test_ftlm_with_unit_vector_starts_and_full_krylov_is_exact(N, n_up):
    # R = D orthonormal starts e_1..e_D, N_L = D: Z_FTLM == Tr e^{-beta H} (pins Eq. 7's D/R,
    # the breakdown rule and the weight definition)
    w = W.ring(N)
    basis = fo.sector_basis(N, n_up)
    D = basis.shape[0]
    ev = np.linalg.eigvalsh(fo.dense_H(N, w.bond_i, w.bond_j, w.J, 0.0, n_up))
    chains = []
    for r in range(D):
        e = np.zeros(D)
        e[r] = 1.0
        chains.append(fo.ritz(*fo.lanczos(_mv(w, basis, n_up), e, D)))
    T = np.array([0.1, 1.0, 10.0])
    got = fo.thermo([dict(dim=D, Mz=0.0, mult=1, chains=chains)], T)
    ref = fo.exact_thermo([(0.0, 1, ev)], T)
    assert got["E_ref"] == pytest.approx(ref["E_ref"], abs=1e-10)
    assert got["Zs"] == pytest.approx(ref["Zs"], rel=1e-9)
    assert got["E"] == pytest.approx(ref["E"], rel=1e-9, abs=1e-9)
    assert got["C"] == pytest.approx(ref["C"], rel=1e-6, abs=1e-9)


def test_dimer_thermodynamics_closed_form():
    # C = (bJ)^2 3 e^{-bJ} / (1 + 3 e^{-bJ})^2 ; chi = 8 b / (3 + e^{bJ}) at g = 2
    w = W.dimer()
    J = 1.0
    spectra = []
    for n_up, Mz, mult in ((1, 0.0, 1), (2, 1.0, 2)):
        spectra.append((Mz, mult, np.linalg.eigvalsh(fo.dense_H(2, w.bond_i, w.bond_j, w.J, 0.0, n_up))))
    T = np.array([0.2, 0.7, 3.0])
    out = fo.exact_thermo(spectra, T)
    b = 1.0 / T
    assert out["C"] == pytest.approx((b * J) ** 2 * 3 * np.exp(-b * J) / (1 + 3 * np.exp(-b * J)) ** 2, rel=1e-12)
    assert out["chi"] == pytest.approx(8 * b / (3 + np.exp(b * J)), rel=1e-12)
    assert out["Zs"] * np.exp(-out["E_ref"] / T) == pytest.approx(np.exp(0.75 * b) + 3 * np.exp(-0.25 * b), rel=1e-12)
    # same through the FTLM path (R = D unit vectors) with all M_z >= 0 sectors and mult
    secs = []
    for n_up, Mz, mult in ((1, 0.0, 1), (2, 1.0, 2)):
        basis = fo.sector_basis(2, n_up)
        D = basis.shape[0]
        chains = [fo.ritz(*fo.lanczos(_mv(w, basis, n_up), np.eye(D)[r], D)) for r in range(D)]
        secs.append(dict(dim=D, Mz=Mz, mult=mult, chains=chains))
    got = fo.thermo(secs, T)
    assert got["C"] == pytest.approx(out["C"], rel=1e-10)
    assert got["chi"] == pytest.approx(out["chi"], rel=1e-10)


def test_high_temperature_limits():
    # Z -> 2^N ; C T^2 -> Tr H^2 / 2^N = (3/16) sum_b J_b^2 ; chi T -> g^2 N / 4
    rng = np.random.default_rng(4)
    N = 8
    pairs = [(a, b) for a in range(N) for b in range(a + 1, N) if rng.random() < 0.5]
    J = rng.uniform(0.5, 1.5, len(pairs))
    w = W._mk("rand8", N, pairs, J)
    spectra = []
    for n_up in range(4, 9):
        Mz = n_up - 4.0
        spectra.append((Mz, 1 if Mz == 0 else 2, np.linalg.eigvalsh(fo.dense_H(N, w.bond_i, w.bond_j, w.J, 0.0, n_up))))
    T = np.array([1e4])
    out = fo.exact_thermo(spectra, T)
    assert out["Zs"][0] * math.exp(-out["E_ref"] / T[0]) == pytest.approx(2 ** N, rel=1e-3)
    assert out["C"][0] * T[0] ** 2 == pytest.approx(3.0 / 16.0 * (J ** 2).sum(), rel=1e-3)
    assert out["chi"][0] * T[0] == pytest.approx(4.0 * N / 4.0, rel=1e-3)


def test_ftlm_converges_to_exact_within_stochastic_error():
    # full FTLM (Gaussian starts, all M_z >= 0 sectors) against exact ED on a small ring
    w = W.ring(10)
    T = W.temperature_grid(30, 0.3, 10.0)
    res, secs, _ = fo.ftlm_run(10, w.bond_i, w.bond_j, w.J, 0.0, range(5, 11), 40, 40, 99, T)
    spectra = [(n_up - 5.0, 1 if n_up == 5 else 2,
                np.linalg.eigvalsh(fo.dense_H(10, w.bond_i, w.bond_j, w.J, 0.0, n_up))) for n_up in range(5, 11)]
    ref = fo.exact_thermo(spectra, T)
    # stochastic error ~ 1/sqrt(R Z_eff) (L43): loose at low T, tight at high T
    assert np.abs(res["C"] - ref["C"]).max() < 0.15 * ref["C"].max()
    assert (np.abs(res["chi"] - ref["chi"]) / ref["chi"]).max() < 0.3
    hot = T >= 2.0
    assert (np.abs(res["chi"] - ref["chi"]) / ref["chi"])[hot].max() < 0.02
    assert (np.abs(res["C"] - ref["C"]) / ref["C"])[hot].max() < 0.05
    assert np.abs(res["E"] - ref["E"]).max() < 0.2


def test_c_lanczos_matches_numpy_lanczos():
    w = W.ring(14, 1.0, 0.5)
    basis = co.enumerate_basis(14, 7)
    q1 = fo.start_vector(5, 7, 1, basis.shape[0])
    a1, b1 = fo.lanczos(_mv(w, basis, 7), q1, 30)
    a2, b2 = co.lanczos(14, w.bond_i, w.bond_j, w.J, 0.0, 7, basis, q1, 30)
    assert a2 == pytest.approx(a1, abs=1e-9) and b2 == pytest.approx(b1, abs=1e-9)


def test_start_vector_generator_statistics_and_scalar_reimplementation():
    # the generator's text re-typed with Python ints, element by element
    M = (1 << 64) - 1
    G = 0x9E3779B97F4A7C15

    def mix(x):
        x &= M
        x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & M
        x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & M
        return x ^ (x >> 31)

    seed, n_up, r = 20260526, 8, 3
    key = mix(mix(mix(seed) + G * (n_up + 1)) + G * (r + 1))
    ts = [0, 1, 2, 12869, 2 ** 33 + 5]
    got = fo.gaussian_elements(seed, n_up, r, np.array(ts, dtype=np.uint64))
    for t, g in zip(ts, got):
        a, b = mix(key + G * (2 * t + 1)), mix(key + G * (2 * t + 2))
        u1, u2 = ((a >> 11) + 1) * 2.0 ** -53, (b >> 11) * 2.0 ** -53
        assert g == pytest.approx(math.sqrt(-2 * math.log(u1)) * math.cos(6.283185307179586 * u2), rel=1e-13, abs=1e-15)
    g = fo.gaussian_elements(seed, n_up, r, np.arange(400000, dtype=np.uint64))
    assert abs(g.mean()) < 5e-3 and abs(g.var() - 1) < 1e-2
    assert abs((g ** 4).mean() - 3) < 0.1 and abs((g[1:] * g[:-1]).mean()) < 5e-3
    g2 = fo.gaussian_elements(seed, n_up, r + 1, np.arange(400000, dtype=np.uint64))
    assert abs((g * g2).mean()) < 5e-3          # chains independent (reading 14)
    g3 = fo.gaussian_elements(seed, n_up + 1, r, np.arange(1000, dtype=np.uint64))
    assert not np.allclose(g[:1000], g3)        # sector enters the key
