"""ctypes front-end of the C oracle (oracle/tg_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

All floating-point inputs are widened to float64 here (bf16 / fp32 values are exactly
representable), all outputs are float64 and are never rounded.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tg_oracle.c")
_SO = os.path.join(_HERE, "libtg_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O3 -march=native -fopenmp.  Building the checker is not using it."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def num_threads() -> int:
    return int(_load().ora_num_threads())


def set_num_threads(n: int) -> None:
    """OpenMP thread count of the following calls (timing legs only; results do not depend on it)."""
    _load().ora_set_num_threads(C.c_int(int(n)))


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


@dataclass
class OracleBlock:
    R: int
    E: int
    U: int
    indptr: np.ndarray
    perm: np.ndarray
    kv_row: np.ndarray
    uniq_node: np.ndarray
    t_indptr: np.ndarray
    t_edge: np.ndarray
    t_dst: np.ndarray
    eid_csr: np.ndarray | None
    ts_csr: np.ndarray | None


def block_build(R, root_idx, nbr_node, edge_id=None, ts=None, dedup_mode=1) -> OracleBlock:
    lib = _load()
    root_idx = _i32(root_idx)
    nbr_node = np.ascontiguousarray(nbr_node, dtype=np.int64)
    E = int(root_idx.shape[0])
    edge_id = None if edge_id is None else np.ascontiguousarray(edge_id, dtype=np.int64)
    ts = None if ts is None else np.ascontiguousarray(ts, dtype=np.float32)
    indptr = np.zeros(R + 1, np.int32)
    perm = np.zeros(E, np.int32)
    kv_row = np.zeros(E, np.int32)
    uniq = np.zeros(max(E, 1), np.int64)
    t_indptr = np.zeros(E + 1, np.int32)
    t_edge = np.zeros(E, np.int32)
    t_dst = np.zeros(E, np.int32)
    eid_csr = None if edge_id is None else np.zeros(E, np.int64)
    ts_csr = None if ts is None else np.zeros(E, np.float32)
    U = C.c_int64(0)
    lib.ora_block_build.restype = C.c_int
    rc = lib.ora_block_build(C.c_int64(R), C.c_int64(E), _p(root_idx, C.c_int32), _p(nbr_node, C.c_int64),
                             _p(edge_id, C.c_int64), _p(ts, C.c_float), C.c_int(dedup_mode),
                             _p(indptr, C.c_int32), _p(perm, C.c_int32), _p(kv_row, C.c_int32), _p(uniq, C.c_int64),
                             _p(t_indptr, C.c_int32), _p(t_edge, C.c_int32), _p(t_dst, C.c_int32),
                             _p(eid_csr, C.c_int64), _p(ts_csr, C.c_float), C.byref(U))
    if rc != 0:
        raise ValueError(f"ora_block_build failed with code {rc}")
    U = int(U.value)
    return OracleBlock(R, E, U, indptr, perm, kv_row, uniq[:U].copy(), t_indptr[:U + 1].copy(), t_edge, t_dst, eid_csr, ts_csr)


def _dims(x):
    assert x.ndim == 3
    return int(x.shape[1]), int(x.shape[2])


def sddmm(indptr, kv_row, A, B, scale=1.0):
    lib = _load()
    A, B = _f64(A), _f64(B)
    H, D = _dims(A)
    indptr, kv_row = _i32(indptr), _i32(kv_row)
    R, E = len(indptr) - 1, len(kv_row)
    s = np.zeros((E, H), np.float64)
    lib.ora_sddmm(C.c_int64(R), C.c_int64(H), C.c_int64(D), _p(indptr, C.c_int32), _p(kv_row, C.c_int32),
                  _p(A, C.c_double), _p(B, C.c_double), C.c_double(scale), _p(s, C.c_double))
    return s


def edge_softmax_fwd(indptr, s):
    lib = _load()
    s = _f64(s)
    indptr = _i32(indptr)
    R, H = len(indptr) - 1, int(s.shape[1])
    alpha = np.zeros_like(s)
    lib.ora_edge_softmax_fwd(C.c_int64(R), C.c_int64(H), _p(indptr, C.c_int32), _p(s, C.c_double), _p(alpha, C.c_double))
    return alpha


def edge_softmax_bwd(indptr, alpha, dalpha):
    lib = _load()
    alpha, dalpha = _f64(alpha), _f64(dalpha)
    indptr = _i32(indptr)
    R, H = len(indptr) - 1, int(alpha.shape[1])
    ds = np.zeros_like(alpha)
    lib.ora_edge_softmax_bwd(C.c_int64(R), C.c_int64(H), _p(indptr, C.c_int32), _p(alpha, C.c_double),
                             _p(dalpha, C.c_double), _p(ds, C.c_double))
    return ds


def aggregate_fwd(indptr, kv_row, w, X):
    lib = _load()
    X, w = _f64(X), _f64(w)
    H, D = _dims(X)
    indptr, kv_row = _i32(indptr), _i32(kv_row)
    R = len(indptr) - 1
    Y = np.zeros((R, H, D), np.float64)
    lib.ora_aggregate_fwd(C.c_int64(R), C.c_int64(H), C.c_int64(D), _p(indptr, C.c_int32), _p(kv_row, C.c_int32),
                          _p(w, C.c_double), _p(X, C.c_double), _p(Y, C.c_double))
    return Y


def aggregate_bwd(indptr, kv_row, U, w, X, dY, want_dw=True):
    lib = _load()
    X, w, dY = _f64(X), _f64(w), _f64(dY)
    H, D = _dims(dY)
    indptr, kv_row = _i32(indptr), _i32(kv_row)
    R, E = len(indptr) - 1, len(kv_row)
    dX = np.zeros((U, H, D), np.float64)
    dw = np.zeros((E, H), np.float64) if (want_dw and X is not None) else None
    lib.ora_aggregate_bwd(C.c_int64(R), C.c_int64(U), C.c_int64(H), C.c_int64(D), _p(indptr, C.c_int32),
                          _p(kv_row, C.c_int32), _p(w, C.c_double), _p(X, C.c_double), _p(dY, C.c_double),
                          _p(dX, C.c_double), _p(dw, C.c_double))
    return dX, dw


def attn_fwd(indptr, kv_row, Q, K, V, scale=1.0, want_alpha=False):
    lib = _load()
    Q, K, V = _f64(Q), _f64(K), _f64(V)
    H, D = _dims(Q)
    indptr, kv_row = _i32(indptr), _i32(kv_row)
    R, E = len(indptr) - 1, len(kv_row)
    O = np.zeros((R, H, D), np.float64)
    LSE = np.zeros((R, H), np.float64)
    alpha = np.zeros((E, H), np.float64) if want_alpha else None
    lib.ora_attn_fwd(C.c_int64(R), C.c_int64(H), C.c_int64(D), _p(indptr, C.c_int32), _p(kv_row, C.c_int32),
                     _p(Q, C.c_double), _p(K, C.c_double), _p(V, C.c_double), C.c_double(scale),
                     _p(O, C.c_double), _p(LSE, C.c_double), _p(alpha, C.c_double))
    return (O, LSE, alpha) if want_alpha else (O, LSE)


def attn_bwd(indptr, kv_row, Q, K, V, dO, scale=1.0):
    lib = _load()
    Q, K, V, dO = _f64(Q), _f64(K), _f64(V), _f64(dO)
    H, D = _dims(Q)
    U = int(K.shape[0])
    indptr, kv_row = _i32(indptr), _i32(kv_row)
    R = len(indptr) - 1
    dQ = np.zeros((R, H, D), np.float64)
    dK = np.zeros((U, H, D), np.float64)
    dV = np.zeros((U, H, D), np.float64)
    lib.ora_attn_bwd.restype = C.c_int
    rc = lib.ora_attn_bwd(C.c_int64(R), C.c_int64(U), C.c_int64(H), C.c_int64(D), _p(indptr, C.c_int32),
                          _p(kv_row, C.c_int32), _p(Q, C.c_double), _p(K, C.c_double), _p(V, C.c_double),
                          _p(dO, C.c_double), C.c_double(scale), _p(dQ, C.c_double), _p(dK, C.c_double), _p(dV, C.c_double))
    if rc != 0:
        raise MemoryError("ora_attn_bwd allocation failed")
    return dQ, dK, dV


def attn_edge_fwd(indptr, kv_row, Q, K, V, Ke=None, Ve=None, scale=1.0, slope=1.0):
    """NEXT-1: per-edge additive key/value rows + LeakyReLU on the logits; see tg_oracle.c."""
    lib = _load()
    Q, K, V = _f64(Q), _f64(K), _f64(V)
    Ke = None if Ke is None else _f64(Ke)
    Ve = None if Ve is None else _f64(Ve)
    H, D = _dims(Q)
    indptr, kv_row = _i32(indptr), _i32(kv_row)
    R = len(indptr) - 1
    O = np.zeros((R, H, D), np.float64)
    LSE = np.zeros((R, H), np.float64)
    lib.ora_attn_edge_fwd(C.c_int64(R), C.c_int64(H), C.c_int64(D), _p(indptr, C.c_int32), _p(kv_row, C.c_int32),
                          _p(Q, C.c_double), _p(K, C.c_double), _p(V, C.c_double), _p(Ke, C.c_double), _p(Ve, C.c_double),
                          C.c_double(scale), C.c_double(slope), _p(O, C.c_double), _p(LSE, C.c_double))
    return O, LSE


def attn_edge_bwd(indptr, kv_row, Q, K, V, Ke, Ve, dO, scale=1.0, slope=1.0):
    lib = _load()
    Q, K, V, dO = _f64(Q), _f64(K), _f64(V), _f64(dO)
    Ke = None if Ke is None else _f64(Ke)
    Ve = None if Ve is None else _f64(Ve)
    H, D = _dims(Q)
    U = int(K.shape[0])
    indptr, kv_row = _i32(indptr), _i32(kv_row)
    R, E = len(indptr) - 1, len(kv_row)
    dQ = np.zeros((R, H, D), np.float64)
    dK = np.zeros((U, H, D), np.float64)
    dV = np.zeros((U, H, D), np.float64)
    dKe = np.zeros((E, H, D), np.float64)
    dVe = np.zeros((E, H, D), np.float64)
    lib.ora_attn_edge_bwd(C.c_int64(R), C.c_int64(U), C.c_int64(H), C.c_int64(D), _p(indptr, C.c_int32), _p(kv_row, C.c_int32),
                          _p(Q, C.c_double), _p(K, C.c_double), _p(V, C.c_double), _p(Ke, C.c_double), _p(Ve, C.c_double),
                          _p(dO, C.c_double), C.c_double(scale), C.c_double(slope),
                          _p(dQ, C.c_double), _p(dK, C.c_double), _p(dV, C.c_double), _p(dKe, C.c_double), _p(dVe, C.c_double))
    return dQ, dK, dV, dKe, dVe
