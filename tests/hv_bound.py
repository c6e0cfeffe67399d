"""Element-wise acceptance bound for H.v against the FP64 oracle (used by the -m gpu parity tests and by the
host-emulation cases; no torch, no library import)."""
import numpy as np


EPS = {"fp32": 2.0 ** -24, "fp64": 2.0 ** -53}


def elem_bound(v, J, h, N, prec):
    """Element-wise bound on |y_t - (H v)_t| for a sum of at most N_B + 1 products accumulated sequentially in the
    working precision ("Tolerances"): (N_B + 2) u (sum_b |J_b| + |h| N / 2) max|v|.  A row that
    misses one of its gathers is off by |J_b / 2| |v_j| - three to six orders of magnitude above this - while the
    norm over 10^8 rows would hide it."""
    J = np.asarray(J, dtype=np.float64)
    return (J.shape[0] + 2) * EPS[prec] * (np.abs(J).sum() + abs(h) * N / 2.0) * float(np.max(np.abs(v)))

