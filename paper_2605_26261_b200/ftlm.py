"""Thin ctypes binding of libftlm.so: same names as include/ftlm.h, argument marshalling only.

Device buffers are torch CUDA tensors (PyTorch is the allocator / stream provider); host
buffers are numpy arrays.  Every step of the path runs inside the library's CUDA kernels.
There is no fallback: if the shared library is missing or a call fails, FtlmError is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# FTLM_CHECKED=1 selects the range-checked build of the same kernels (csrc/ftlm_access.cuh); it is a test aid,
# several times slower, and reports through ftlm_get_option(ctx, "check_violations").
CHECKED = os.environ.get("FTLM_CHECKED", "0") not in ("", "0")
LIB_PATH = os.path.join(_HERE, "libftlm_checked.so" if CHECKED else "libftlm.so")

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED = 0, 1, 2, 3, 4
INDEX_CLT, INDEX_CR, INDEX_LIN = 0, 1, 2
FP32, FP64 = 0, 1
KERNEL_AUTO, KERNEL_ROW, KERNEL_ROWG, KERNEL_TML = 0, 1, 2, 3
MAX_STEPS = 1024

EXPORTS = [
    "ftlm_create", "ftlm_destroy", "ftlm_dim", "ftlm_set_option", "ftlm_get_option", "ftlm_table_bytes",
    "ftlm_clt_read", "ftlm_index_of", "ftlm_state_of", "ftlm_neighbors", "ftlm_apply_H",
    "ftlm_apply_H_host", "ftlm_fill_random", "ftlm_chain_begin", "ftlm_chain_steps", "ftlm_chain_end",
    "ftlm_chain_begin_batch", "ftlm_chain_end_batch", "ftlm_chain_profile", "ftlm_autotune", "ftlm_lanczos", "ftlm_lanczos_host", "ftlm_tridiag_eig", "ftlm_thermo",
    "ftlm_ghost_diagnostic", "ftlm_sigma_emp", "ftlm_sigma_theo",
    "ftlm_last_error", "ftlm_version",
]


class FtlmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"ftlm error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libftlm.so (built in-tree by `python -m paper_2605_26261_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FtlmError(ECUDA, f"{LIB_PATH} not built; run python -m paper_2605_26261_b200.build "
                                   "(there is no CPU or PyTorch fallback)")
        L = C.CDLL(LIB_PATH)
        L.ftlm_dim.restype = C.c_int64
        L.ftlm_get_option.restype = C.c_int64
        L.ftlm_table_bytes.restype = C.c_int64
        L.ftlm_last_error.restype = C.c_char_p
        L.ftlm_version.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc):
    if rc != OK:
        raise FtlmError(rc, lib().ftlm_last_error().decode())


def _hp(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def _dp(t):
    """Device pointer of a torch CUDA tensor (contiguous)."""
    if t is None:
        return C.c_void_p(0)
    assert t.is_cuda and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def ftlm_version() -> str:
    return lib().ftlm_version().decode()


def ftlm_create(N, bond_i, bond_j, J, N_up, index_mode=INDEX_CLT, precision=FP32, h=0.0, device=0):
    bi = np.ascontiguousarray(bond_i, dtype=np.int32)
    bj = np.ascontiguousarray(bond_j, dtype=np.int32)
    Jc = np.ascontiguousarray(J, dtype=np.float64)
    assert bi.shape == bj.shape == Jc.shape
    h_ = C.c_void_p()
    _check(lib().ftlm_create(C.byref(h_), C.c_int(N), C.c_int(bi.shape[0]), _hp(bi, C.c_int32), _hp(bj, C.c_int32),
                             _hp(Jc, C.c_double), C.c_double(h), C.c_int(N_up), C.c_int(index_mode),
                             C.c_int(precision), C.c_int(device)))
    return h_


def ftlm_destroy(ctx):
    _check(lib().ftlm_destroy(ctx))


def ftlm_dim(ctx) -> int:
    return int(lib().ftlm_dim(ctx))


def ftlm_set_option(ctx, key: str, value: int):
    _check(lib().ftlm_set_option(ctx, key.encode(), C.c_int64(value)))


def ftlm_get_option(ctx, key: str) -> int:
    return int(lib().ftlm_get_option(ctx, key.encode()))


def ftlm_check_info() -> dict:
    """Checked build (FTLM_CHECKED=1): device-side address violations so far in this process and the first one
    (translation unit, source line, kind 0/1 = global range/alignment, 2/3 = shared range/alignment)."""
    keys = ["check_build", "check_violations", "check_first_tu", "check_first_line", "check_first_kind",
            "check_first_block", "check_first_thread", "check_first_addr"]
    return {k: int(lib().ftlm_get_option(C.c_void_p(0), k.encode())) for k in keys}


def ftlm_check_selftest() -> int:
    """Checked build: launch five deliberately bad accesses; returns how many the checker suppressed and counted (5)."""
    return int(lib().ftlm_get_option(C.c_void_p(0), b"check_selftest"))


def ftlm_table_bytes(ctx) -> int:
    return int(lib().ftlm_table_bytes(ctx))


def ftlm_clt_read(ctx, b0: int, nb: int):
    m = np.empty(nb, dtype=np.uint32)
    c = np.empty(nb, dtype=np.uint32)
    _check(lib().ftlm_clt_read(ctx, C.c_int64(b0), C.c_int64(nb), _hp(m, C.c_uint32), _hp(c, C.c_uint32)))
    return m, c


def ftlm_index_of(ctx, d_labels, d_idx, stream=None):
    """d_labels: torch int64/uint64 CUDA tensor holding uint64 labels; d_idx: int64 CUDA tensor."""
    _check(lib().ftlm_index_of(ctx, _dp(d_labels), C.c_int64(d_labels.numel()), _dp(d_idx), _stream(stream)))


def ftlm_state_of(ctx, d_idx, d_labels, stream=None):
    _check(lib().ftlm_state_of(ctx, _dp(d_idx), C.c_int64(d_idx.numel()), _dp(d_labels), _stream(stream)))


def ftlm_neighbors(ctx, row0: int, nrows: int, d_idx, stream=None):
    _check(lib().ftlm_neighbors(ctx, C.c_int64(row0), C.c_int64(nrows), _dp(d_idx), _stream(stream)))


def ftlm_apply_H(ctx, d_v, d_y, stream=None):
    _check(lib().ftlm_apply_H(ctx, _dp(d_v), _dp(d_y), _stream(stream)))


def ftlm_apply_H_host(ctx, h_v: np.ndarray, h_y: np.ndarray):
    assert h_v.flags.c_contiguous and h_y.flags.c_contiguous
    _check(lib().ftlm_apply_H_host(ctx, C.c_void_p(h_v.ctypes.data), C.c_void_p(h_y.ctypes.data)))


def ftlm_fill_random(ctx, seed: int, r: int, d_v, stream=None):
    _check(lib().ftlm_fill_random(ctx, C.c_uint64(seed), C.c_int(r), _dp(d_v), _stream(stream)))


def ftlm_chain_begin(ctx, d_q1, seed: int, r: int, stream=None):
    _check(lib().ftlm_chain_begin(ctx, _dp(d_q1), C.c_uint64(seed), C.c_int(r), _stream(stream)))


def ftlm_chain_steps(ctx, nsteps: int, stream=None):
    _check(lib().ftlm_chain_steps(ctx, C.c_int(nsteps), _stream(stream)))


def ftlm_chain_end(ctx, cap: int = MAX_STEPS, stream=None):
    a = np.zeros(cap, dtype=np.float64)
    b = np.zeros(cap, dtype=np.float64)
    m = C.c_int(0)
    _check(lib().ftlm_chain_end(ctx, _hp(a, C.c_double), _hp(b, C.c_double), C.c_int(cap), C.byref(m), _stream(stream)))
    k = min(m.value, cap)
    return a[:k].copy(), b[: max(k - 1, 0)].copy(), m.value


def ftlm_chain_begin_batch(ctx, seed: int, r0: int, batch: int, stream=None):
    _check(lib().ftlm_chain_begin_batch(ctx, C.c_uint64(seed), C.c_int(r0), C.c_int(batch), _stream(stream)))


def ftlm_chain_end_batch(ctx, batch: int, cap: int = MAX_STEPS, stream=None):
    """Returns (alpha[batch, cap], beta[batch, cap], m_eff[batch]) of the batch in progress."""
    a = np.zeros((batch, cap), dtype=np.float64)
    b = np.zeros((batch, cap), dtype=np.float64)
    m = np.zeros(batch, dtype=np.int32)
    _check(lib().ftlm_chain_end_batch(ctx, _hp(a, C.c_double), _hp(b, C.c_double), C.c_int(cap), _hp(m, C.c_int), _stream(stream)))
    return a, b, m


def ftlm_chain_profile(ctx, nsteps: int, stream=None):
    x, y = C.c_double(0), C.c_double(0)
    _check(lib().ftlm_chain_profile(ctx, C.c_int(nsteps), _stream(stream), C.byref(x), C.byref(y)))
    return x.value, y.value


def ftlm_autotune(ctx, reps: int = 3, stream=None):
    """Measure the kernel candidates on the device, keep the fastest valid one; returns the report list."""
    import json
    buf = C.create_string_buffer(8192)
    _check(lib().ftlm_autotune(ctx, C.c_int(reps), buf, C.c_int(len(buf)), _stream(stream)))
    return json.loads(buf.value.decode())


def _lanczos_out(R, n_steps):
    return (np.zeros((R, n_steps)), np.zeros((R, n_steps)), np.zeros(R, dtype=np.int32),
            np.zeros((R, n_steps)), np.zeros((R, n_steps)))


def ftlm_lanczos(ctx, seed: int, R: int, n_steps: int, stream=None):
    """Returns dict(alpha[R,n], beta[R,n], m_eff[R], theta[R,n], weight[R,n])."""
    a, b, m, th, w = _lanczos_out(R, n_steps)
    _check(lib().ftlm_lanczos(ctx, C.c_uint64(seed), C.c_int(R), C.c_int(n_steps), _hp(a, C.c_double),
                              _hp(b, C.c_double), _hp(m, C.c_int), _hp(th, C.c_double), _hp(w, C.c_double),
                              _stream(stream)))
    return dict(alpha=a, beta=b, m_eff=m, theta=th, weight=w)


def ftlm_lanczos_host(ctx, h_q1: np.ndarray, n_steps: int, stream=None):
    """h_q1: host array [R, dim] in the handle's precision (pinned memory recommended)."""
    assert h_q1.ndim == 2 and h_q1.flags.c_contiguous
    R = h_q1.shape[0]
    a, b, m, th, w = _lanczos_out(R, n_steps)
    _check(lib().ftlm_lanczos_host(ctx, C.c_void_p(h_q1.ctypes.data), C.c_int(R), C.c_int(n_steps),
                                   _hp(a, C.c_double), _hp(b, C.c_double), _hp(m, C.c_int), _hp(th, C.c_double),
                                   _hp(w, C.c_double), _stream(stream)))
    return dict(alpha=a, beta=b, m_eff=m, theta=th, weight=w)


def ftlm_tridiag_eig(alpha, beta):
    alpha = np.ascontiguousarray(alpha, dtype=np.float64)
    beta = np.ascontiguousarray(beta, dtype=np.float64)
    m = alpha.shape[0]
    assert beta.shape[0] >= m - 1
    th, w = np.zeros(m), np.zeros(m)
    bb = beta if beta.shape[0] > 0 else np.zeros(1)
    _check(lib().ftlm_tridiag_eig(C.c_int(m), _hp(alpha, C.c_double), _hp(bb, C.c_double), _hp(th, C.c_double),
                                  _hp(w, C.c_double)))
    return th, w


def ftlm_thermo(dim, Mz, mult, R, m_eff, theta, weight, T, g=2.0):
    """Sectors s: dim[s], Mz[s], mult[s], R[s]; chains stacked in sector order: m_eff[sum R],
    theta/weight [sum R, stride].  Returns dict(E_ref, Zs, E, C, chi)."""
    dim = np.ascontiguousarray(dim, dtype=np.int64)
    Mz = np.ascontiguousarray(Mz, dtype=np.float64)
    mult = np.ascontiguousarray(mult, dtype=np.float64)
    R = np.ascontiguousarray(R, dtype=np.int32)
    m_eff = np.ascontiguousarray(m_eff, dtype=np.int32)
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    weight = np.ascontiguousarray(weight, dtype=np.float64)
    T = np.ascontiguousarray(T, dtype=np.float64)
    assert theta.ndim == 2 and theta.shape == weight.shape and theta.shape[0] == int(R.sum()) == m_eff.shape[0]
    nT = T.shape[0]
    eref = C.c_double(0)
    Zs, E, Cv, chi = (np.zeros(nT) for _ in range(4))
    _check(lib().ftlm_thermo(C.c_int(dim.shape[0]), _hp(dim, C.c_int64), _hp(Mz, C.c_double), _hp(mult, C.c_double),
                             _hp(R, C.c_int), C.c_int(theta.shape[1]), _hp(m_eff, C.c_int), _hp(theta, C.c_double),
                             _hp(weight, C.c_double), C.c_int(nT), _hp(T, C.c_double), C.c_double(g), C.byref(eref),
                             _hp(Zs, C.c_double), _hp(E, C.c_double), _hp(Cv, C.c_double), _hp(chi, C.c_double)))
    return dict(E_ref=eref.value, Zs=Zs, E=E, C=Cv, chi=chi)


def ftlm_ghost_diagnostic(alpha, beta, C_tau: float = 1.0) -> dict:
    """Host: Cullum-Willoughby ghost flags, clusters and cluster weights of one chain (include/ftlm.h)."""
    a = np.ascontiguousarray(alpha, dtype=np.float64)
    m = a.shape[0]
    b = np.zeros(max(m, 1), dtype=np.float64)
    b[: max(m - 1, 0)] = np.asarray(beta, dtype=np.float64)[: max(m - 1, 0)]
    th, w, ell, cw, F = (np.zeros(m) for _ in range(5))
    gh, cl = np.zeros(m, dtype=np.int32), np.zeros(m, dtype=np.int32)
    tau = C.c_double(0)
    _check(lib().ftlm_ghost_diagnostic(C.c_int(m), _hp(a, C.c_double), _hp(b, C.c_double), C.c_double(C_tau),
                                       _hp(th, C.c_double), _hp(w, C.c_double), _hp(ell, C.c_double), _hp(gh, C.c_int),
                                       _hp(cl, C.c_int), _hp(cw, C.c_double), _hp(F, C.c_double), C.byref(tau)))
    return dict(theta=th, weight=w, ell=ell, ghost=gh.astype(bool), cluster=cl, cluster_weight=cw, F=F, tau=tau.value)


def ftlm_sigma_emp(samples):
    a = np.ascontiguousarray(samples, dtype=np.float64)
    mean, sig = np.zeros(a.shape[1]), np.zeros(a.shape[1])
    _check(lib().ftlm_sigma_emp(C.c_int(a.shape[0]), C.c_int(a.shape[1]), _hp(a, C.c_double), _hp(mean, C.c_double), _hp(sig, C.c_double)))
    return mean, sig


def ftlm_sigma_theo(O, Z_eff):
    o = np.ascontiguousarray(O, dtype=np.float64)
    z = np.ascontiguousarray(Z_eff, dtype=np.float64)
    sig = np.zeros_like(o)
    _check(lib().ftlm_sigma_theo(C.c_int(o.shape[0]), _hp(o, C.c_double), _hp(z, C.c_double), _hp(sig, C.c_double)))
    return sig
