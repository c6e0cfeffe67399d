"""Host diagnostics (section 3.2 Eqs. 23-25 and Eq. 22): oracle pinned by identities and dense
ED, then the library's host functions against the oracle.  No GPU."""
import numpy as np
import pytest

from oracle import ftlm_oracle as fo
from paper_2605_26261_b200 import ftlm
from paper_2605_26261_b200 import workloads as W


def _random_T(m, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(m), np.abs(rng.standard_normal(m - 1)) + 0.1


def test_oracle_ell_reproduces_the_first_component_identity():
    """For an unreduced symmetric tridiagonal T the squared first components of the eigenvectors are
    w_k = prod_j (theta_k - theta^(1)_j) / prod_{j != k} (theta_k - theta_j) with theta^(1) the eigenvalues of T
    without its first row and column (the fact behind the Cullum-Willoughby test: w_k -> 0 exactly when theta_k meets
    a theta^(1)).  Pins the T^(1) slicing of `ghost_diagnostic` against `ritz`'s weights."""
    for m, seed in ((2, 1), (5, 2), (9, 3)):
        a, b = _random_T(m, seed)
        d = fo.ghost_diagnostic(a, b)
        T1 = np.diag(a[1:]) + np.diag(b[1:], 1) + np.diag(b[1:], -1)
        th1 = np.linalg.eigvalsh(T1)
        for k in range(m):
            num = np.prod(d["theta"][k] - th1)
            den = np.prod(np.delete(d["theta"][k] - d["theta"], k))
            assert num / den == pytest.approx(d["weight"][k], rel=1e-9, abs=1e-14)
            assert d["ell"][k] == pytest.approx(np.abs(d["theta"][k] - th1).min(), abs=1e-12)
        assert not d["ghost"].any()                          # exact arithmetic, separated spectrum: interlacing, no ghosts
        assert d["F"][-1] == pytest.approx(1.0, abs=1e-12)
        assert (np.diff(d["cluster"]) == 1).all()            # every Ritz value its own cluster


def test_oracle_cluster_weights_equal_exact_overlaps_when_fp32_lanczos_makes_ghosts():
    """L264-L270: run FP32 Lanczos far beyond convergence on a small sector (ghosts appear); the total weight of the
    cluster at each converged eigenvalue must equal the exact |<q_1|psi>|^2 summed over that (degenerate) level from
    dense ED - the paper's statement that ghosts only redistribute weight inside converged clusters."""
    w = W.ring(10)
    n_up = 5
    basis = fo.sector_basis(w.N, n_up)
    D = basis.shape[0]
    H = fo.dense_H(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up)
    ev, U = np.linalg.eigh(H)
    q1 = fo.start_vector(7, n_up, 0, D).astype(np.float32)
    mv = lambda x: fo.apply_H(basis, w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, x.astype(np.float64)).astype(np.float32)
    al, be, _ = _lanczos_fp32(mv, q1, 150)
    d = fo.ghost_diagnostic(al, be, C_tau=8.0)
    assert d["ghost"].sum() >= 3                             # far beyond D_Krylov: copies exist
    ov = (U.T @ (q1.astype(np.float64) / np.linalg.norm(q1.astype(np.float64)))) ** 2
    # lowest level (non-degenerate singlet ground state) and the top level: converged first
    for lvl in (ev[0], ev[-1]):
        exact = ov[np.abs(ev - lvl) < 1e-6].sum()
        k = int(np.argmin(np.abs(d["theta"] - lvl)))
        assert abs(d["theta"][k] - lvl) < 1e-4
        assert d["cluster_weight"][k] == pytest.approx(exact, rel=2e-3)
    assert d["cluster_weight"].max() <= 1.0 + 1e-6 and d["F"][-1] == pytest.approx(1.0, abs=1e-5)


def _lanczos_fp32(matvec, q1, m):
    """Textbook recurrence (L45) with FP32 vectors and FP64 scalars, no breakdown stop (ghosts are wanted)."""
    q = q1 / np.float32(np.linalg.norm(q1.astype(np.float64)))
    qp = np.zeros_like(q)
    al, be = [], []
    beta = 0.0
    for _ in range(m):
        y = matvec(q) - np.float32(beta) * qp
        a = float(np.dot(q.astype(np.float64), y.astype(np.float64)))
        y = y - np.float32(a) * q
        beta = float(np.linalg.norm(y.astype(np.float64)))
        al.append(a); be.append(beta)
        qp, q = q, (y / np.float32(beta)).astype(np.float32)
    return np.array(al), np.array(be[:-1]), None


@pytest.mark.parametrize("case", ["random5", "random40", "ghosts", "m1", "m2"])
def test_library_ghost_diagnostic_matches_oracle(case):
    if case == "ghosts":
        w = W.ring(10)
        basis = fo.sector_basis(w.N, 5)
        mv = lambda x: fo.apply_H(basis, w.N, w.bond_i, w.bond_j, w.J, 0.0, 5, x.astype(np.float64)).astype(np.float32)
        a, b, _ = _lanczos_fp32(mv, fo.start_vector(3, 5, 0, basis.shape[0]).astype(np.float32), 120)
    elif case == "m1":
        a, b = np.array([0.7]), np.array([])
    else:
        a, b = _random_T({"random5": 5, "random40": 40, "m2": 2}[case], 11)
    for C_tau in (1.0, 8.0):
        ref = fo.ghost_diagnostic(a, b, C_tau)
        got = ftlm.ftlm_ghost_diagnostic(a, b, C_tau)
        scale = max(1.0, np.abs(ref["theta"]).max())
        assert np.abs(got["theta"] - ref["theta"]).max() <= 1e-12 * scale
        assert got["tau"] == pytest.approx(ref["tau"], rel=1e-9, abs=1e-300)
        assert np.abs(got["F"] - ref["F"]).max() <= 1e-9
        if len(a) > 1:
            # ell of a ghost is itself at rounding level: compare on the scale of the spectrum, flags away from the threshold
            assert np.abs(got["ell"] - ref["ell"]).max() <= 1e-10 * scale
            clear = np.abs(ref["ell"] - ref["tau"]) > 1e-9 * scale
            assert (got["ghost"][clear] == ref["ghost"][clear]).all()
            gaps = np.diff(ref["theta"])
            if (np.abs(gaps - ref["tau"]) > 1e-9 * scale).all():
                assert (got["cluster"] == ref["cluster"]).all()
                assert np.abs(got["cluster_weight"] - ref["cluster_weight"]).max() <= 1e-9
        else:
            assert np.isinf(got["ell"][0]) and not got["ghost"][0] and got["cluster_weight"][0] == pytest.approx(1.0)


def test_sigma_emp_and_sigma_theo():
    mean, sig = ftlm.ftlm_sigma_emp([[1.0, 10.0], [3.0, 10.0]])
    assert mean.tolist() == [2.0, 10.0] and sig.tolist() == [1.0, 0.0]        # Eq. 22 with the 1/N_s it prints
    rng = np.random.default_rng(5)
    s = rng.standard_normal((12, 7))
    m_ref, s_ref = fo.sigma_emp(s)
    m_got, s_got = ftlm.ftlm_sigma_emp(s)
    assert np.allclose(m_got, m_ref, rtol=1e-13) and np.allclose(s_got, s_ref, rtol=1e-12)
    assert np.allclose(s_ref, s.std(axis=0, ddof=0))
    O, Z = rng.standard_normal(7), rng.uniform(1, 100, 7)
    assert np.allclose(ftlm.ftlm_sigma_theo(O, Z), fo.sigma_theo(O, Z), rtol=1e-14)
    assert ftlm.ftlm_sigma_theo([-2.0], [16.0])[0] == 0.5
    with pytest.raises(ftlm.FtlmError):
        ftlm.ftlm_sigma_theo([1.0], [0.0])


def test_sigma_theo_bounds_sigma_emp_in_order_of_magnitude_on_a_small_ring():
    """L230 calls sigma_theo = O / sqrt(Z_eff) an approximate bound for the pooled estimate; on the N = 10 ring with
    R = 4 vectors per sector and 12 seed sets sigma_emp(C) / sqrt(R) stays within a factor ~10 of it at T >= 0.5."""
    w = W.ring(10)
    T = np.array([0.5, 1.0, 3.0])
    runs = [fo.ftlm_run(w.N, w.bond_i, w.bond_j, w.J, 0.0, list(range(5, 11)), 4, 30, 100 + s, T)[0] for s in range(12)]
    mean, sig = fo.sigma_emp([r["C"] for r in runs])
    Zeff = np.mean([r["Zs"] for r in runs], axis=0)
    theo = fo.sigma_theo(mean, Zeff) / np.sqrt(4.0)
    assert (sig < 10 * theo).all() and (sig > theo / 30).all()
