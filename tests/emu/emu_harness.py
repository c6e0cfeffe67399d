"""TEST INFRASTRUCTURE: ctypes loader for tests/emu/libftlm_emu.so (the kernel sources compiled for
the host against the SIMT emulation layer).  "Device" buffers are numpy arrays.  Used only by
tests/test_emu_*.py, which run each case in a subprocess (an out-of-bounds access in a kernel hits
a guard page and kills that subprocess, not pytest)."""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

INDEX = {"clt": 0, "cr": 1, "lin": 2}
PREC = {"fp32": 0, "fp64": 1}
NDT = {"fp32": np.float32, "fp64": np.float64}
KERNEL = {"auto": 0, "row": 1, "rowg": 2, "tml": 3}

_lib = None


def lib():
    global _lib
    if _lib is None:
        sys.path.insert(0, HERE)
        import build_emu
        L = C.CDLL(os.environ.get("FTLM_EMU_LIB") or build_emu.build())   # a frozen copy, for long sweeps
        L.ftlm_dim.restype = C.c_int64
        L.ftlm_get_option.restype = C.c_int64
        L.ftlm_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise RuntimeError(f"ftlm(emu) error {rc}: {lib().ftlm_last_error().decode()}")


def _p(a):
    return C.c_void_p(a.ctypes.data)


class EmuCtx:
    def __init__(self, w, n_up, mode="cr", prec="fp64", h=None, J=None, options=()):
        self.w, self.n_up, self.mode, self.prec = w, n_up, mode, prec
        bi = np.ascontiguousarray(w.bond_i, dtype=np.int32)
        bj = np.ascontiguousarray(w.bond_j, dtype=np.int32)
        Jc = np.ascontiguousarray(w.J if J is None else J, dtype=np.float64)
        self.ctx = C.c_void_p()
        _check(lib().ftlm_create(C.byref(self.ctx), C.c_int(w.N), C.c_int(bi.shape[0]), _p(bi), _p(bj), _p(Jc),
                                 C.c_double(w.h if h is None else h), C.c_int(n_up), C.c_int(INDEX[mode]),
                                 C.c_int(PREC[prec]), C.c_int(0)))
        for k, v in options:
            self.set(k, v)
        self.dim = int(lib().ftlm_dim(self.ctx))

    def set(self, key, value):
        _check(lib().ftlm_set_option(self.ctx, key.encode(), C.c_int64(value)))

    def get(self, key):
        return int(lib().ftlm_get_option(self.ctx, key.encode()))

    def close(self):
        _check(lib().ftlm_destroy(self.ctx))

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def apply(self, v, shift=0):
        """shift: the caller's vectors start `shift` elements after a 64-byte boundary (a slice of a larger buffer:
        only element alignment is guaranteed to the library)."""
        buf_v = np.zeros(self.dim + 32, dtype=NDT[self.prec])
        buf_y = np.full(self.dim + 32, np.nan, dtype=NDT[self.prec])
        off = (-buf_v.ctypes.data // buf_v.itemsize) % (64 // buf_v.itemsize) + shift
        offy = (-buf_y.ctypes.data // buf_y.itemsize) % (64 // buf_y.itemsize) + shift
        vv, y = buf_v[off:off + self.dim], buf_y[offy:offy + self.dim]
        vv[:] = v
        _check(lib().ftlm_apply_H(self.ctx, _p(vv), _p(y), C.c_void_p(0)))
        return y.copy()

    def apply_into(self, v, y):
        """y is read-modify-written when only PASS-B windows run (option debug_pass_mask)."""
        assert v.dtype == NDT[self.prec] and y.dtype == NDT[self.prec] and v.flags.c_contiguous and y.flags.c_contiguous
        _check(lib().ftlm_apply_H(self.ctx, _p(v), _p(y), C.c_void_p(0)))

    def bond_classes(self):
        """[(class, entry)] per bond from the TML plan; class 6 = PASS-B window `entry`."""
        out = []
        for b in range(self.w.n_bonds):
            x = self.get(f"tml_bclass:{b}")
            out.append((x & 0xff, x >> 8))
        return out

    def diag0(self):
        return float(np.sum(self.w.J if self.w is not None else 0.0)) / 4.0

    def autotune(self, reps=1):
        import json
        buf = C.create_string_buffer(8192)
        _check(lib().ftlm_autotune(self.ctx, C.c_int(reps), buf, C.c_int(len(buf)), C.c_void_p(0)))
        return json.loads(buf.value.decode())

    def neighbors(self, row0, nrows):
        nb = max(self.w.n_bonds, 1)
        out = np.full(nrows * nb, -7, dtype=np.int64)
        _check(lib().ftlm_neighbors(self.ctx, C.c_int64(row0), C.c_int64(nrows), _p(out), C.c_void_p(0)))
        return out.reshape(nrows, nb)[:, : self.w.n_bonds]

    def index_of(self, labels):
        lab = np.ascontiguousarray(labels, dtype=np.uint64)
        out = np.empty(lab.shape[0], dtype=np.int64)
        _check(lib().ftlm_index_of(self.ctx, _p(lab), C.c_int64(lab.shape[0]), _p(out), C.c_void_p(0)))
        return out

    def state_of(self, idx):
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        out = np.empty(idx.shape[0], dtype=np.uint64)
        _check(lib().ftlm_state_of(self.ctx, _p(idx), C.c_int64(idx.shape[0]), _p(out), C.c_void_p(0)))
        return out

    def lanczos(self, seed, R, n_steps):
        a = np.zeros((R, n_steps)); b = np.zeros((R, n_steps)); m = np.zeros(R, dtype=np.int32)
        th = np.zeros((R, n_steps)); wt = np.zeros((R, n_steps))
        _check(lib().ftlm_lanczos(self.ctx, C.c_uint64(seed), C.c_int(R), C.c_int(n_steps), _p(a), _p(b), _p(m),
                                  _p(th), _p(wt), C.c_void_p(0)))
        return dict(alpha=a, beta=b, m_eff=m, theta=th, weight=wt)
