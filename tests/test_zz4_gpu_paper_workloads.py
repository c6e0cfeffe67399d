"""-m gpu: SURVEY 8(f)-2, the paper's second spin-1/2 systems (Fig. 3 c-f; bond lists and their pins:
tests/test_paper_workloads.py) through ftlm_lanczos (batched chains) + ftlm_thermo against the oracle."""
import numpy as np
import pytest

from oracle import ftlm_oracle as fo
from paper_2605_26261_b200 import workloads as W


@pytest.mark.gpu
@pytest.mark.parametrize("name,mode,prec,batch", [("ring20", "clt", "fp32", 4), ("dodecahedron", "cr", "fp32", 4),
                                                  ("dodecahedron", "clt", "fp64", 2), ("ring20", "cr", "fp64", 1)])
def test_all_sectors_thermodynamics_vs_oracle(name, mode, prec, batch):
    """All 11 sectors (D up to C(20,10) = 184 756), R = 4 seeded vectors each in batches, 60 steps (the paper's R = 100,
    N_L = 100 is a matter of run time, not of code): C(T), chi(T), E(T) against the oracle from the same start vectors."""
    import torch  # noqa: F401
    from paper_2605_26261_b200 import ftlm
    from gpu_util import Ctx
    w = W.paper_workload(name)
    T = W.temperature_grid(60)
    R, n_steps, seed = 4, 60, W.SEED_VECTORS
    cast = np.float32 if prec == "fp32" else None
    ref, _, _ = fo.ftlm_run(w.N, w.bond_i, w.bond_j, w.J, 0.0, w.sectors, R, n_steps, seed, T, tol=1e-12, cast=cast)
    dims, Mz, mult, Rs, m_eff, TH, WW = [], [], [], [], [], [], []
    for n_up in w.sectors:
        with Ctx(w, n_up, mode, prec) as c:
            ftlm.ftlm_set_option(c.ctx, "batch", batch)
            out = ftlm.ftlm_lanczos(c.ctx, seed, R, n_steps)
            dims.append(c.dim)
        mz = n_up - w.N / 2.0
        Mz.append(mz); mult.append(1 if mz == 0 else 2); Rs.append(R)
        m_eff += list(out["m_eff"]); TH.append(out["theta"]); WW.append(out["weight"])
    got = ftlm.ftlm_thermo(dims, Mz, mult, Rs, m_eff, np.vstack(TH), np.vstack(WW), T)
    tol = 1e-4 if prec == "fp32" else 1e-8
    for key in ("C", "chi", "E"):
        r = ref[key]
        scale = np.maximum(np.abs(r), 1e-3 * np.abs(r).max())          # reading 28
        assert (np.abs(got[key] - r) / scale).max() <= tol, key
