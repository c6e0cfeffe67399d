"""-m gpu: option "persistent" (launch-bound small sectors): all R chains of a sector in ONE launch, one CTA
per chain, the three work vectors resident in shared memory (csrc/ftlm_chain.cu).  Against the oracle chain by chain,
against the ordinary path, and BASELINE config 1's thermodynamics (N = 16 ring, all sectors, R = 20, N_L = 60)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import c_oracle as co              # noqa: E402
from oracle import ftlm_oracle as fo           # noqa: E402
from paper_2605_26261_b200 import ftlm         # noqa: E402
from paper_2605_26261_b200 import workloads as W   # noqa: E402
from gpu_util import Ctx                       # noqa: E402


@pytest.mark.parametrize("wl,n_up,mode,prec,R,steps,fits", [
    (W.ring(12, 1.0, 0.5), 6, "cr", "fp64", 3, 20, 1),
    (W.ring(16), 8, "clt", "fp32", 20, 60, 1),              # config 1's largest sector: 3 x 12 870 floats = 154 KB
    (W.ring(16), 8, "cr", "fp64", 2, 10, 0),                # FP64: does not fit, ordinary path
    (W.ring(16), 15, "lin", "fp32", 4, 16, 1),              # D = 16: breakdown at step 9
    (W.ring(16), 16, "cr", "fp64", 2, 5, 1),                # D = 1
    (W.ring(16), 12, "clt", "fp64", 5, 40, 1),              # D = 1820
])
def test_persistent_chains_match_oracle_and_ordinary_path(wl, n_up, mode, prec, R, steps, fits):
    basis = co.enumerate_basis(wl.N, n_up)
    with Ctx(wl, n_up, mode, prec) as c:
        plain = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, R, steps)
        ftlm.ftlm_set_option(c.ctx, "persistent", 1)
        assert ftlm.ftlm_get_option(c.ctx, "persistent_fits") == fits
        out = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, R, steps)
    tol = 1e-9 if prec == "fp64" else 2e-4
    assert (out["m_eff"] == plain["m_eff"]).all()
    for r in range(R):
        m = int(out["m_eff"][r])
        q1 = fo.start_vector(W.SEED_VECTORS, n_up, r, c.dim)
        a, b = co.lanczos(wl.N, wl.bond_i, wl.bond_j, wl.J, 0.0, n_up, basis, q1, min(steps, c.dim))[:2]
        k = min(m, len(a), 6)
        assert np.abs(out["alpha"][r][:k] - np.asarray(a)[:k]).max() <= tol
        if k > 1:
            assert np.abs(out["beta"][r][:k - 1] - np.asarray(b)[:k - 1]).max() <= tol
        assert abs(out["weight"][r][:m].sum() - 1.0) <= 1e-6
        # the ordinary path does the same arithmetic in another summation order: early coefficients agree closely
        assert np.abs(out["alpha"][r][:k] - plain["alpha"][r][:k]).max() <= tol


@pytest.mark.slow
@pytest.mark.parametrize("mode", ["clt", "cr"])
def test_persistent_config1_thermodynamics(mode):
    w = W.baseline_config(1)
    T = W.temperature_grid(200)
    ref = fo.ftlm_run(w.N, w.bond_i, w.bond_j, w.J, 0.0, w.sectors, w.R, w.n_steps, W.SEED_VECTORS, T, cast=np.float32)[0]
    dims, Mz, mult, Rs, m_eff, TH, WW = [], [], [], [], [], [], []
    for n_up in w.sectors:
        with Ctx(w, n_up, mode, "fp32") as c:
            ftlm.ftlm_set_option(c.ctx, "persistent", 1)
            assert ftlm.ftlm_get_option(c.ctx, "persistent_fits") == 1
            out = ftlm.ftlm_lanczos(c.ctx, W.SEED_VECTORS, w.R, w.n_steps)
            dims.append(c.dim)
        mz = n_up - w.N / 2.0
        Mz.append(mz); mult.append(1 if mz == 0 else 2); Rs.append(w.R)
        m_eff += list(out["m_eff"]); TH.append(out["theta"]); WW.append(out["weight"])
    got = ftlm.ftlm_thermo(dims, Mz, mult, Rs, m_eff, np.vstack(TH), np.vstack(WW), T)
    for key in ("C", "chi", "E"):
        r = ref[key]
        scale = np.maximum(np.abs(r), 1e-3 * np.abs(r).max())
        assert (np.abs(got[key] - r) / scale).max() <= 1e-4, key
