"""Helpers for the -m gpu parity tests (CUDA path via the C ABI vs the FP64 oracle)."""
import numpy as np
import torch

from paper_2605_26261_b200 import ftlm
from hv_bound import elem_bound  # noqa: F401

MODES = {"clt": ftlm.INDEX_CLT, "cr": ftlm.INDEX_CR, "lin": ftlm.INDEX_LIN}
PRECS = {"fp32": ftlm.FP32, "fp64": ftlm.FP64}
TDT = {"fp32": torch.float32, "fp64": torch.float64}
NDT = {"fp32": np.float32, "fp64": np.float64}
HV_TOL = {"fp32": 1e-5, "fp64": 1e-12}      # BASELINE.json north_star


class Ctx:
    def __init__(self, w, n_up, mode, prec, h=None, J=None, kernel=None):
        self.w, self.n_up, self.mode, self.prec = w, n_up, mode, prec
        self.h = w.h if h is None else h
        self.J = w.J if J is None else J
        self.ctx = ftlm.ftlm_create(w.N, w.bond_i, w.bond_j, self.J, n_up, MODES[mode], PRECS[prec], self.h)
        if kernel is not None:
            ftlm.ftlm_set_option(self.ctx, "kernel", kernel)
        self.dim = ftlm.ftlm_dim(self.ctx)

    def __enter__(self):
        return self

    def __exit__(self, *a):
        ftlm.ftlm_destroy(self.ctx)

    def apply(self, v_np):
        v = torch.from_numpy(np.ascontiguousarray(v_np, dtype=NDT[self.prec])).cuda()
        y = torch.empty_like(v)
        ftlm.ftlm_apply_H(self.ctx, v, y)
        torch.cuda.synchronize()
        return y.cpu().numpy()

    def index_of(self, labels_np):
        lab = torch.from_numpy(np.ascontiguousarray(labels_np, dtype=np.uint64).view(np.int64)).cuda()
        out = torch.empty(lab.numel(), dtype=torch.int64, device="cuda")
        ftlm.ftlm_index_of(self.ctx, lab, out)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    def state_of(self, idx_np):
        idx = torch.from_numpy(np.ascontiguousarray(idx_np, dtype=np.int64)).cuda()
        out = torch.empty(idx.numel(), dtype=torch.int64, device="cuda")
        ftlm.ftlm_state_of(self.ctx, idx, out)
        torch.cuda.synchronize()
        return out.cpu().numpy().view(np.uint64)

    def neighbors(self, row0, nrows):
        out = torch.empty(nrows * max(self.w.n_bonds, 1), dtype=torch.int64, device="cuda")
        ftlm.ftlm_neighbors(self.ctx, row0, nrows, out)
        torch.cuda.synchronize()
        return out.cpu().numpy().reshape(nrows, -1)[:, : self.w.n_bonds]

    def fill_random(self, seed, r):
        v = torch.empty(self.dim, dtype=TDT[self.prec], device="cuda")
        ftlm.ftlm_fill_random(self.ctx, seed, r, v)
        torch.cuda.synchronize()
        return v


def relerr(y, ref):
    y = np.asarray(y, dtype=np.float64)
    den = np.linalg.norm(ref)
    return np.linalg.norm(y - ref) / (den if den > 0 else 1.0)


def hv_err(y, ref, v, J, h, N, prec):
    """Norm-relative error of y against the oracle's ref (north_star's criterion, returned) after asserting the
    element-wise bound on every row."""
    y = np.asarray(y, dtype=np.float64)
    worst = float(np.max(np.abs(y - ref))) if y.size else 0.0
    bound = elem_bound(v, J, h, N, prec)
    assert worst <= bound, f"element-wise: max|y - ref| = {worst:.3e} > {bound:.3e} at row {int(np.argmax(np.abs(y - ref)))}"
    return relerr(y, ref)
