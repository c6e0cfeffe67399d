"""ctypes loader for oracle/ftlm_oracle_c.c (large-N FP64 oracle).  TEST INFRASTRUCTURE ONLY:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  Compiles the C file with gcc on first use if the .so is missing or stale."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ftlm_oracle_c.c")
_SO = os.path.join(_HERE, "libftlm_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _SO, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(os.environ.get("FTLM_ORACLE_LIB") or build())   # (a sanitizer build of the same file, for tests)
        _lib.orc_enumerate.restype = C.c_int64
        _lib.orc_index.restype = C.c_int64
        _lib.orc_lanczos.restype = C.c_int
        _lib.orc_threads.restype = C.c_int
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def threads() -> int:
    return int(lib().orc_threads())


def enumerate_basis(N: int, N_up: int) -> np.ndarray:
    D = lib().orc_enumerate(C.c_int(N), C.c_int(N_up), None)
    basis = np.empty(D, dtype=np.uint64)
    lib().orc_enumerate(C.c_int(N), C.c_int(N_up), _p(basis, C.c_uint64))
    return basis


def index_many(basis: np.ndarray, labels: np.ndarray) -> np.ndarray:
    labels = np.ascontiguousarray(labels, dtype=np.uint64)
    out = np.empty(labels.shape[0], dtype=np.int64)
    lib().orc_index_many(_p(basis, C.c_uint64), C.c_int64(basis.shape[0]), _p(labels, C.c_uint64),
                         C.c_int64(labels.shape[0]), _p(out, C.c_int64))
    return out


def _bonds(bond_i, bond_j, J):
    return (np.ascontiguousarray(bond_i, dtype=np.int32), np.ascontiguousarray(bond_j, dtype=np.int32),
            np.ascontiguousarray(J, dtype=np.float64))


def apply_rows(N, bond_i, bond_j, J, h, N_up, basis, v, row0=0, nrows=None) -> np.ndarray:
    bi, bj, Jc = _bonds(bond_i, bond_j, J)
    v = np.ascontiguousarray(v, dtype=np.float64)
    D = basis.shape[0]
    nrows = D - row0 if nrows is None else nrows
    y = np.empty(nrows, dtype=np.float64)
    lib().orc_apply_rows(C.c_int(N), C.c_int(len(Jc)), _p(bi, C.c_int32), _p(bj, C.c_int32),
                         _p(Jc, C.c_double), C.c_double(h), C.c_int(N_up), _p(basis, C.c_uint64),
                         C.c_int64(D), _p(v, C.c_double), C.c_int64(row0), C.c_int64(nrows),
                         _p(y, C.c_double))
    return y


def neighbors_rows(N, bond_i, bond_j, basis, rows) -> np.ndarray:
    bi, bj, _ = _bonds(bond_i, bond_j, np.zeros(len(bond_i)))
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    out = np.empty((rows.shape[0], len(bi)), dtype=np.int64)
    lib().orc_neighbors_rows(C.c_int(N), C.c_int(len(bi)), _p(bi, C.c_int32), _p(bj, C.c_int32),
                             _p(basis, C.c_uint64), C.c_int64(basis.shape[0]), _p(rows, C.c_int64),
                             C.c_int64(rows.shape[0]), _p(out, C.c_int64))
    return out


def lanczos(N, bond_i, bond_j, J, h, N_up, basis, q1, n_steps, tol=1e-12):
    bi, bj, Jc = _bonds(bond_i, bond_j, J)
    q1 = np.ascontiguousarray(q1, dtype=np.float64)
    alpha = np.zeros(n_steps, dtype=np.float64)
    beta = np.zeros(max(n_steps, 1), dtype=np.float64)
    m = lib().orc_lanczos(C.c_int(N), C.c_int(len(Jc)), _p(bi, C.c_int32), _p(bj, C.c_int32),
                          _p(Jc, C.c_double), C.c_double(h), C.c_int(N_up), _p(basis, C.c_uint64),
                          C.c_int64(basis.shape[0]), _p(q1, C.c_double), C.c_int(n_steps),
                          C.c_double(tol), _p(alpha, C.c_double), _p(beta, C.c_double))
    return alpha[:m].copy(), beta[: max(m - 1, 0)].copy()
