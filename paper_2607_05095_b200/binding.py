"""Thin ctypes binding over ``libfasttg.so`` (include/fasttg.h).  Argument marshalling only.

Every step of the path runs in the library's CUDA kernels; this module turns torch tensors into
device pointers, allocates outputs / workspaces through torch (the library never allocates), and
raises ``FastTGError`` on a non-zero status.  There is no CPU fallback: if the shared library is
missing or no CUDA device is present, calls fail loudly.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libfasttg.so")
_lib = None

TG_F32, TG_BF16 = 0, 1
_DTYPES = {torch.float32: TG_F32, torch.bfloat16: TG_BF16}

# Signature of every export of include/fasttg.h and include/fasttg_diag.h: name -> (result, arguments), one letter per C type:
#   I int / enum   L int64_t   Q uint64_t / unsigned long long   Z size_t   F float   D double   P any pointer (incl. tg_stream_t)
#   S const char*.  lib() turns this into ctypes argtypes / restype, so a call with the wrong number or kind of arguments raises
# instead of shifting every later argument by one slot; tests/test_host_abi.py re-derives the table from the header.
SIGNATURES = {
    "tg_status_string": ("S", "I"),
    "tg_last_error": ("S", ""),
    "tg_version": ("I", ""),
    "tg_launch_count": ("Q", ""),
    "tg_probe_gather": ("I", "PIIIPPPP"),
    "tg_probe_gather_bulk": ("I", "PIIIIPPPPP"),
    "tg_supported": ("I", "III"),
    "tg_block_workspace_bytes": ("I", "LLIP"),
    "tg_block_build": ("I", "LLPPPPIPPPPPPPPPPPZPP"),
    "tg_sched_workspace_bytes": ("I", "LLLP"),
    "tg_block_from_csr": ("I", "LLLPPPPPPZPP"),
    "tg_block_destroy": ("I", "P"),
    "tg_block_info": ("I", "PPPPP"),
    "tg_block_sched_info": ("I", "PP"),
    "tg_block_build_retries": ("Q", ""),
    "tg_tcsr_workspace_bytes": ("I", "LLP"),
    "tg_tcsr_build": ("I", "LLPPPPPPPPZP"),
    "tg_sample_workspace_bytes": ("I", "LP"),
    "tg_sample_neighbors": ("I", "IIQLPPLPPPPPPPPPPZP"),
    "tg_sddmm": ("I", "PIIIPPFPP"),
    "tg_edge_softmax_fwd": ("I", "PIPPP"),
    "tg_edge_softmax_bwd": ("I", "PIPPPP"),
    "tg_aggregate_fwd": ("I", "PIIIPPPPZP"),
    "tg_aggregate_bwd": ("I", "PIIIPPPPPPZP"),
    "tg_block_coo_dst": ("I", "PPP"),
    "tg_aggregate_coo": ("I", "PIIIIPPPP"),
    "tg_attn_workspace_bytes": ("I", "PIIIPP"),
    "tg_attn_fused_fwd": ("I", "PIIIPPPFPPPPZP"),
    "tg_attn_fused_bwd": ("I", "PIIIPPPPPPPFPPPPZP"),
    "tg_attn_fused_bwd_dst": ("I", "PIIIPPPPPPPFPPZP"),
    "tg_attn_fused_bwd_src": ("I", "PIIIPPPPFPPPZP"),
    "tg_attn_edge_fused_fwd": ("I", "PIIIPPPPPFFPPPZP"),
    "tg_attn_edge_fused_bwd": ("I", "PIIIPPPPPPPPFFPPPPPPZP"),
    "tg_cache_greedy_select": ("I", "DLPPPPLLPPPP"),
    "tg_cache_lookup_workspace_bytes": ("I", "LP"),
    "tg_cache_lookup": ("I", "LPPPPPPZP"),
    "tg_cache_lookup_static": ("I", "LPPPPPP"),
    "tg_feature_reconstruct": ("I", "LLPPPPPP"),
}
EXPORTS = list(SIGNATURES)
_CTYPE = {"I": C.c_int, "L": C.c_int64, "Q": C.c_uint64, "Z": C.c_size_t, "F": C.c_float, "D": C.c_double, "P": C.c_void_p, "S": C.c_char_p}


class FastTGError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str):
        super().__init__(f"{where}: status {status} ({detail})")
        self.status = status


def lib() -> C.CDLL:
    """Loads libfasttg.so (built by ``paper_2607_05095_b200.build``); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise FileNotFoundError(f"{_LIB_PATH} not found: run `python -m paper_2607_05095_b200.build` (no CPU fallback exists)")
        L = C.CDLL(_LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)  # fail loudly on a missing symbol
            fn.restype = _CTYPE[res]
            fn.argtypes = [_CTYPE[a] for a in args]
        _lib = L
    return _lib


def launch_count() -> int:
    """tg_launch_count: kernels launched by the library in this process so far."""
    return int(lib().tg_launch_count())


def block_build_retries() -> int:
    """tg_block_build_retries: builds repeated in this process because the speculation was too optimistic."""
    return int(lib().tg_block_build_retries())


def probe_gather(table_rows: int, gathers_per_group: int = 4096, iters: int = 5) -> float:
    """tg_probe_gather: GB/s of 256-byte row gathers from a table of `table_rows` rows (small: all L1 hits)."""
    table = torch.randint(0, 2 ** 31 - 1, (table_rows, 64), dtype=torch.int32, device="cuda")
    sink = torch.zeros(1, dtype=torch.int32, device="cuda")
    ms, nbytes = C.c_float(0), C.c_double(0)
    _check(lib().tg_probe_gather(_ptr(table), C.c_int(table_rows), C.c_int(gathers_per_group), C.c_int(iters), _ptr(sink),
                                 _stream(), C.byref(ms), C.byref(nbytes)), "tg_probe_gather")
    return nbytes.value / (ms.value * 1e-3) / 1e9


def probe_gather_bulk(table_rows: int, stages: int = 4, gathers_per_group: int = 4096, iters: int = 5):
    """tg_probe_gather_bulk: (GB/s, resident CTAs per SM) of the same gathers issued as cp.async.bulk into a shared-memory ring."""
    table = torch.randint(0, 2 ** 31 - 1, (table_rows, 64), dtype=torch.int32, device="cuda")
    sink = torch.zeros(2, dtype=torch.int32, device="cuda")
    ms, nbytes, occ = C.c_float(0), C.c_double(0), C.c_int(0)
    _check(lib().tg_probe_gather_bulk(_ptr(table), C.c_int(table_rows), C.c_int(gathers_per_group), C.c_int(stages), C.c_int(iters),
                                      _ptr(sink), _stream(), C.byref(ms), C.byref(nbytes), C.byref(occ)), "tg_probe_gather_bulk")
    return nbytes.value / (ms.value * 1e-3) / 1e9, occ.value


def _check(st: int, where: str):
    if st != 0:
        L = lib()
        raise FastTGError(st, where, f"{L.tg_status_string(st).decode()}: {L.tg_last_error().decode()}")


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dt(t: torch.Tensor) -> int:
    try:
        return _DTYPES[t.dtype]
    except KeyError:
        raise TypeError(f"unsupported storage dtype {t.dtype}") from None


def _rows(t: torch.Tensor, name: str) -> torch.Tensor:
    if t.dim() != 3 or not t.is_contiguous() or not t.is_cuda:
        raise ValueError(f"{name} must be a contiguous CUDA tensor [rows, H, D]")
    return t


def _check_rows(t: torch.Tensor, name: str, rows: int, like: torch.Tensor, exact: bool = True) -> torch.Tensor:
    """Shape / dtype / device / contiguity of one row tensor against the block and the reference tensor `like` ([*, H, D]):
    the C ABI only sees raw pointers, a wrong-sized or non-contiguous tensor would be read or written out of bounds."""
    _rows(t, name)
    if t.dtype != like.dtype or t.device != like.device or tuple(t.shape[1:]) != tuple(like.shape[1:]):
        raise ValueError(f"{name}: expected [*, {like.shape[1]}, {like.shape[2]}] {like.dtype} on {like.device}, got {tuple(t.shape)} {t.dtype} on {t.device}")
    if (exact and t.shape[0] != rows) or t.shape[0] < rows:
        raise ValueError(f"{name}: {t.shape[0]} rows, the block needs {'exactly' if exact else 'at least'} {rows}")
    return t


def _check_scalars(t: torch.Tensor, name: str, rows: int, H: int, like: torch.Tensor) -> torch.Tensor:
    if t.dtype != torch.float32 or tuple(t.shape) != (rows, H) or not t.is_contiguous() or t.device != like.device:
        raise ValueError(f"{name} must be a contiguous float32 [{rows}, {H}] tensor on {like.device}")
    return t


def supported(H: int, D: int, dtype: torch.dtype) -> bool:
    return bool(lib().tg_supported(C.c_int(H), C.c_int(D), C.c_int(_DTYPES[dtype])))


class Block:
    """Destination-grouped CSR block + unique-row remap + transposed CSR (tg_block_build)."""

    def __init__(self):
        self.handle = C.c_void_p(0)
        self.R = self.E = self.U = 0
        self.indptr = self.perm = self.kv_row = self.uniq_node = None
        self.t_indptr = self.t_edge = self.t_dst = self.eid_csr = self.ts_csr = None
        self._ws = None
        self._full = None      # block_build: the full-capacity output arrays and the workspace (block_build(reuse=...))
        self._attn_ws = {}

    def destroy(self):
        """tg_block_destroy; the Block must not be used afterwards (its arrays may be handed to another build)."""
        if self.handle and _lib is not None:
            _lib.tg_block_destroy(self.handle)
        self.handle = C.c_void_p(0)
        self._full = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def info(self):
        R, E, U = C.c_int64(), C.c_int64(), C.c_int64()
        stats = (C.c_int64 * 8)()
        _check(lib().tg_block_info(self.handle, C.byref(R), C.byref(E), C.byref(U), stats), "tg_block_info")
        keys = ["dst_group_small", "dst_group_big", "dst_warp_items", "dst_slots", "src_group_small", "src_group_big", "src_warp_items", "src_slots"]
        return {"R": R.value, "E": E.value, "U": U.value, **{k: int(v) for k, v in zip(keys, stats)}}

    def sched_info(self):
        """tg_block_sched_info: group-tier limit, warp-item chunk, hub count and largest degree of both sides."""
        out = (C.c_int64 * 8)()
        _check(lib().tg_block_sched_info(self.handle, out), "tg_block_sched_info")
        keys = ["group_max", "chunk", "hubs", "max_deg"]
        return {side + "_" + k: int(out[4 * i + j]) for i, side in enumerate(("dst", "src")) for j, k in enumerate(keys)}

    def attn_workspace(self, H: int, D: int, dtype: torch.dtype):
        """(forward, backward) workspaces of this block, cached per (H, D, dtype).  They are shared by every call on the
        block: calls that use the same block concurrently must be ordered on one stream (or use separate Block objects)."""
        key = (H, D, dtype)
        if key not in self._attn_ws:
            fb, bb = C.c_size_t(), C.c_size_t()
            _check(lib().tg_attn_workspace_bytes(self.handle, C.c_int(H), C.c_int(D), C.c_int(_DTYPES[dtype]),
                                                 C.byref(fb), C.byref(bb)), "tg_attn_workspace_bytes")
            dev = self.indptr.device
            self._attn_ws[key] = (torch.empty(fb.value, dtype=torch.uint8, device=dev),
                                  torch.empty(bb.value, dtype=torch.uint8, device=dev))
        return self._attn_ws[key]


def block_build(R: int, root_idx: torch.Tensor, nbr_node: torch.Tensor, edge_id: torch.Tensor | None = None,
                ts: torch.Tensor | None = None, dedup_mode: int = 1, reuse: Block | None = None) -> Block:
    """tg_block_build.  root_idx int32 [E], nbr_node int64 [E], edge_id int64 [E] | None, ts float32 [E] | None (CUDA).
    reuse: a Block of the same (R, E, dedup_mode, pass-through arrays) whose output arrays and workspace are taken over
    instead of allocating new ones (a training loop with a fixed batch shape); that Block is destroyed by the call."""
    L = lib()
    dev = root_idx.device
    if not root_idx.is_cuda:
        raise ValueError("block_build needs CUDA tensors (no CPU fallback)")
    E = int(root_idx.shape[0])
    assert root_idx.dtype == torch.int32 and nbr_node.dtype == torch.int64
    root_idx, nbr_node = root_idx.contiguous(), nbr_node.contiguous()
    if edge_id is not None:
        assert edge_id.dtype == torch.int64
        edge_id = edge_id.contiguous()
    if ts is not None:
        assert ts.dtype == torch.float32
        ts = ts.contiguous()
    b = Block()
    i32 = dict(dtype=torch.int32, device=dev)
    nbytes = C.c_size_t()
    _check(L.tg_block_workspace_bytes(C.c_int64(R), C.c_int64(E), C.c_int(dedup_mode), C.byref(nbytes)), "tg_block_workspace_bytes")
    key = (R, E, dedup_mode, edge_id is not None, ts is not None, dev, nbytes.value)
    if reuse is not None:
        if reuse._full is None or reuse._full["key"] != key:
            raise ValueError("block_build(reuse=...): the Block to reuse was built for another shape")
        full = reuse._full
        reuse.destroy()
    else:
        full = dict(key=key, indptr=torch.empty(R + 1, **i32), perm=torch.empty(E, **i32), kv_row=torch.empty(E, **i32),
                    uniq_node=torch.empty(max(E, 1), dtype=torch.int64, device=dev), t_indptr=torch.empty(E + 1, **i32),
                    t_edge=torch.empty(E, **i32), t_dst=torch.empty(E, **i32),
                    eid_csr=None if edge_id is None else torch.empty(E, dtype=torch.int64, device=dev),
                    ts_csr=None if ts is None else torch.empty(E, dtype=torch.float32, device=dev),
                    ws=torch.empty(nbytes.value, dtype=torch.uint8, device=dev))
    b._full = full
    b.indptr, b.perm, b.kv_row, b.uniq_node, b.t_indptr = full["indptr"], full["perm"], full["kv_row"], full["uniq_node"], full["t_indptr"]
    b.t_edge, b.t_dst, b.eid_csr, b.ts_csr, b._ws = full["t_edge"], full["t_dst"], full["eid_csr"], full["ts_csr"], full["ws"]
    U = C.c_int64()
    _check(L.tg_block_build(C.c_int64(R), C.c_int64(E), _ptr(root_idx), _ptr(nbr_node), _ptr(edge_id), _ptr(ts),
                            C.c_int(dedup_mode), _ptr(b.indptr), _ptr(b.perm), _ptr(b.kv_row), _ptr(b.uniq_node),
                            _ptr(b.t_indptr), _ptr(b.t_edge), _ptr(b.t_dst), _ptr(b.eid_csr), _ptr(b.ts_csr),
                            C.byref(U), _ptr(b._ws), C.c_size_t(nbytes.value), _stream(), C.byref(b.handle)), "tg_block_build")
    b.R, b.E, b.U = R, E, int(U.value)
    b.uniq_node = b.uniq_node[:b.U]
    b.t_indptr = b.t_indptr[:b.U + 1]
    return b


def block_from_csr(indptr, kv_row, U, t_indptr, t_edge, t_dst) -> Block:
    """tg_block_from_csr: wrap existing device index arrays, build only the schedules."""
    L = lib()
    b = Block()
    b.indptr, b.kv_row, b.t_indptr, b.t_edge, b.t_dst = (x.contiguous() for x in (indptr, kv_row, t_indptr, t_edge, t_dst))
    R, E = int(indptr.shape[0]) - 1, int(kv_row.shape[0])
    nbytes = C.c_size_t()
    _check(L.tg_sched_workspace_bytes(C.c_int64(R), C.c_int64(E), C.c_int64(U), C.byref(nbytes)), "tg_sched_workspace_bytes")
    b._ws = torch.empty(nbytes.value, dtype=torch.uint8, device=indptr.device)
    _check(L.tg_block_from_csr(C.c_int64(R), C.c_int64(E), C.c_int64(U), _ptr(b.indptr), _ptr(b.kv_row), _ptr(b.t_indptr),
                               _ptr(b.t_edge), _ptr(b.t_dst), _ptr(b._ws), C.c_size_t(nbytes.value), _stream(),
                               C.byref(b.handle)), "tg_block_from_csr")
    b.R, b.E, b.U = R, E, int(U)
    return b


def sddmm(b: Block, A: torch.Tensor, B: torch.Tensor, scale: float = 1.0, out: torch.Tensor | None = None) -> torch.Tensor:
    _rows(A, "A"); _rows(B, "B")
    H, D = A.shape[1], A.shape[2]
    s = out if out is not None else torch.empty(b.E, H, dtype=torch.float32, device=A.device)
    _check(lib().tg_sddmm(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(A)), _ptr(A), _ptr(B), C.c_float(scale), _ptr(s), _stream()), "tg_sddmm")
    return s


def edge_softmax_fwd(b: Block, s: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
    H = s.shape[1]
    alpha = out if out is not None else torch.empty_like(s)
    _check(lib().tg_edge_softmax_fwd(b.handle, C.c_int(H), _ptr(s), _ptr(alpha), _stream()), "tg_edge_softmax_fwd")
    return alpha


def edge_softmax_bwd(b: Block, alpha: torch.Tensor, dalpha: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
    H = alpha.shape[1]
    ds = out if out is not None else torch.empty_like(alpha)
    _check(lib().tg_edge_softmax_bwd(b.handle, C.c_int(H), _ptr(alpha), _ptr(dalpha), _ptr(ds), _stream()), "tg_edge_softmax_bwd")
    return ds


def aggregate_fwd(b: Block, w: torch.Tensor | None, X: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
    _rows(X, "X")
    H, D = X.shape[1], X.shape[2]
    Y = out if out is not None else torch.empty(b.R, H, D, dtype=X.dtype, device=X.device)
    ws, _ = b.attn_workspace(H, D, X.dtype)
    _check(lib().tg_aggregate_fwd(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(X)), _ptr(w), _ptr(X), _ptr(Y), _ptr(ws),
                                  C.c_size_t(ws.numel()), _stream()), "tg_aggregate_fwd")
    return Y


def aggregate_bwd(b: Block, w: torch.Tensor | None, X: torch.Tensor | None, dY: torch.Tensor, want_dw: bool = True):
    _rows(dY, "dY")
    H, D = dY.shape[1], dY.shape[2]
    dX = torch.empty(b.U, H, D, dtype=dY.dtype, device=dY.device)
    dw = torch.empty(b.E, H, dtype=torch.float32, device=dY.device) if (want_dw and X is not None) else None
    _, ws = b.attn_workspace(H, D, dY.dtype)
    _check(lib().tg_aggregate_bwd(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(dY)), _ptr(w), _ptr(X), _ptr(dY), _ptr(dX),
                                  _ptr(dw), _ptr(ws), C.c_size_t(ws.numel()), _stream()), "tg_aggregate_bwd")
    return dX, dw


def _check_o32(o32, b: Block, Q: torch.Tensor):
    if o32 is not None and (o32.dtype != torch.float32 or tuple(o32.shape) != (b.R,) + tuple(Q.shape[1:]) or not o32.is_contiguous() or o32.device != Q.device):
        raise ValueError(f"o32 must be a contiguous float32 [{b.R}, {Q.shape[1]}, {Q.shape[2]}] tensor on {Q.device}")
    return o32


def attn_fused_fwd(b: Block, Q: torch.Tensor, K: torch.Tensor, V: torch.Tensor, scale: float = 1.0, out=None, o32: torch.Tensor | None = None):
    """tg_attn_fused_fwd.  o32 (optional, float32 [R,H,D]): receives the unrounded copy of O for attn_fused_bwd (bf16 storage)."""
    _check_rows(Q, "Q", b.R, Q); _check_rows(K, "K", b.U, Q, exact=False); _check_rows(V, "V", b.U, Q, exact=False)
    H, D = Q.shape[1], Q.shape[2]
    if out is None:
        O = torch.empty_like(Q)
        lse = torch.empty(b.R, H, dtype=torch.float32, device=Q.device)
    else:
        O, lse = out
        _check_rows(O, "O", b.R, Q); _check_scalars(lse, "lse", b.R, H, Q)
    ws, _ = b.attn_workspace(H, D, Q.dtype)
    _check(lib().tg_attn_fused_fwd(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(Q)), _ptr(Q), _ptr(K), _ptr(V), C.c_float(scale),
                                   _ptr(O), _ptr(lse), _ptr(_check_o32(o32, b, Q)), _ptr(ws), C.c_size_t(ws.numel()), _stream()), "tg_attn_fused_fwd")
    return O, lse


def attn_fused_bwd(b: Block, Q, K, V, O, lse, dO, scale: float = 1.0, out=None, o32=None):
    for t, n in ((Q, "Q"), (O, "O"), (dO, "dO")):
        _check_rows(t, n, b.R, Q)
    _check_rows(K, "K", b.U, Q, exact=False); _check_rows(V, "V", b.U, Q, exact=False)
    H, D = Q.shape[1], Q.shape[2]
    _check_scalars(lse, "lse", b.R, H, Q)
    if out is None:
        dQ, dK, dV = torch.empty_like(Q), torch.empty_like(K), torch.empty_like(V)
    else:
        dQ, dK, dV = out
        _check_rows(dQ, "dQ", b.R, Q); _check_rows(dK, "dK", b.U, Q, exact=False); _check_rows(dV, "dV", b.U, Q, exact=False)
    _, ws = b.attn_workspace(H, D, Q.dtype)
    _check(lib().tg_attn_fused_bwd(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(Q)), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(_check_o32(o32, b, Q)), _ptr(lse),
                                   _ptr(dO), C.c_float(scale), _ptr(dQ), _ptr(dK), _ptr(dV), _ptr(ws), C.c_size_t(ws.numel()),
                                   _stream()), "tg_attn_fused_bwd")
    return dQ, dK, dV


def attn_fused_bwd_dst(b: Block, Q, K, V, O, lse, dO, scale: float, dQ, o32=None):
    """First half of attn_fused_bwd (destination-major): dQ and the internal {LSE, delta} table."""
    for t, n in ((Q, "Q"), (O, "O"), (dO, "dO"), (dQ, "dQ")):
        _check_rows(t, n, b.R, Q)
    _check_rows(K, "K", b.U, Q, exact=False); _check_rows(V, "V", b.U, Q, exact=False)
    H, D = Q.shape[1], Q.shape[2]
    _check_scalars(lse, "lse", b.R, H, Q)
    _, ws = b.attn_workspace(H, D, Q.dtype)
    _check(lib().tg_attn_fused_bwd_dst(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(Q)), _ptr(Q), _ptr(K), _ptr(V), _ptr(O),
                                       _ptr(_check_o32(o32, b, Q)), _ptr(lse), _ptr(dO), C.c_float(scale), _ptr(dQ), _ptr(ws), C.c_size_t(ws.numel()),
                                       _stream()), "tg_attn_fused_bwd_dst")
    return dQ


def attn_fused_bwd_src(b: Block, Q, K, V, dO, scale: float, dK, dV):
    """Second half of attn_fused_bwd (source-major over the transposed CSR): dK, dV.  The block's cached workspace carries
    the {LSE, delta} table from attn_fused_bwd_dst: both halves must run on the same stream, in this order."""
    _check_rows(Q, "Q", b.R, Q); _check_rows(dO, "dO", b.R, Q)
    for t, n in ((K, "K"), (V, "V"), (dK, "dK"), (dV, "dV")):
        _check_rows(t, n, b.U, Q, exact=False)
    H, D = Q.shape[1], Q.shape[2]
    _, ws = b.attn_workspace(H, D, Q.dtype)
    _check(lib().tg_attn_fused_bwd_src(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(Q)), _ptr(Q), _ptr(K), _ptr(V), _ptr(dO),
                                       C.c_float(scale), _ptr(dK), _ptr(dV), _ptr(ws), C.c_size_t(ws.numel()), _stream()),
           "tg_attn_fused_bwd_src")
    return dK, dV


def attn_edge_fused_fwd(b: Block, Q, K, V, Ke, Ve, scale: float = 1.0, slope: float = 1.0, out=None):
    """tg_attn_edge_fused_fwd: per-edge additive key/value rows Ke, Ve [E,H,D] (CSR order) + LeakyReLU(slope) on the logits."""
    Q, K, V, Ke, Ve = (_rows(t, n) for t, n in ((Q, "Q"), (K, "K"), (V, "V"), (Ke, "Ke"), (Ve, "Ve")))
    R, H, D = Q.shape
    O, lse = out if out is not None else (torch.empty_like(Q), torch.empty(R, H, dtype=torch.float32, device=Q.device))
    fws, _ = b.attn_workspace(H, D, Q.dtype)
    _check(lib().tg_attn_edge_fused_fwd(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(Q)), _ptr(Q), _ptr(K), _ptr(V), _ptr(Ke), _ptr(Ve),
                                        C.c_float(scale), C.c_float(slope), _ptr(O), _ptr(lse), _ptr(fws), C.c_size_t(fws.numel()),
                                        _stream()), "tg_attn_edge_fused_fwd")
    return O, lse


def attn_edge_fused_bwd(b: Block, Q, K, V, Ke, Ve, O, lse, dO, scale: float = 1.0, slope: float = 1.0):
    """tg_attn_edge_fused_bwd: returns dQ, dK, dV, dKe, dVe."""
    Q, K, V, Ke, Ve, O, dO = (_rows(t, n) for t, n in ((Q, "Q"), (K, "K"), (V, "V"), (Ke, "Ke"), (Ve, "Ve"), (O, "O"), (dO, "dO")))
    R, H, D = Q.shape
    dQ, dK, dV, dKe, dVe = torch.empty_like(Q), torch.empty_like(K), torch.empty_like(V), torch.empty_like(Ke), torch.empty_like(Ve)
    _, bws = b.attn_workspace(H, D, Q.dtype)
    _check(lib().tg_attn_edge_fused_bwd(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(Q)), _ptr(Q), _ptr(K), _ptr(V), _ptr(Ke), _ptr(Ve),
                                        _ptr(O), _ptr(lse), _ptr(dO), C.c_float(scale), C.c_float(slope), _ptr(dQ), _ptr(dK), _ptr(dV),
                                        _ptr(dKe), _ptr(dVe), _ptr(bws), C.c_size_t(bws.numel()), _stream()), "tg_attn_edge_fused_bwd")
    return dQ, dK, dV, dKe, dVe


def cache_greedy_select(alpha: float, batches, n_nodes: int, n_edges: int):
    """tg_cache_greedy_select (host): batches = list of (node_id_array, edge_id_array); returns (hot_nodes, hot_edges) int64."""
    import numpy as np
    nptr, eptr = [0], [0]
    for nk, ek in batches:
        nptr.append(nptr[-1] + len(nk)); eptr.append(eptr[-1] + len(ek))
    cat = lambda xs: np.ascontiguousarray(np.concatenate([np.asarray(x, np.int64) for x in xs]) if xs else np.zeros(0, np.int64))
    nid, eid = cat([b[0] for b in batches]), cat([b[1] for b in batches])
    nptr, eptr = np.array(nptr, np.int64), np.array(eptr, np.int64)
    hn, he = np.zeros(max(n_nodes, 1), np.int64), np.zeros(max(n_edges, 1), np.int64)
    cn, ce = C.c_int64(0), C.c_int64(0)
    P = lambda a: a.ctypes.data_as(C.POINTER(C.c_int64))
    _check(lib().tg_cache_greedy_select(C.c_double(alpha), C.c_int64(len(batches)), P(nptr), P(nid), P(eptr), P(eid),
                                        C.c_int64(n_nodes), C.c_int64(n_edges), P(hn), C.byref(cn), P(he), C.byref(ce)),
           "tg_cache_greedy_select")
    return hn[:cn.value].copy(), he[:ce.value].copy()


def cache_lookup(uniq_ids: torch.Tensor, slot_of_id: torch.Tensor):
    """tg_cache_lookup: returns (map int32 [U], fresh_ids int64 [n_fresh])."""
    U = int(uniq_ids.shape[0])
    m = torch.empty(U, dtype=torch.int32, device=uniq_ids.device)
    fresh = torch.empty(U, dtype=torch.int64, device=uniq_ids.device)
    nb = C.c_size_t()
    _check(lib().tg_cache_lookup_workspace_bytes(C.c_int64(U), C.byref(nb)), "tg_cache_lookup_workspace_bytes")
    ws = torch.empty(nb.value, dtype=torch.uint8, device=uniq_ids.device)
    n = C.c_int64(0)
    _check(lib().tg_cache_lookup(C.c_int64(U), _ptr(uniq_ids.contiguous()), _ptr(slot_of_id.contiguous()), _ptr(m), _ptr(fresh), C.byref(n),
                                 _ptr(ws), C.c_size_t(nb.value), _stream()), "tg_cache_lookup")
    return m, fresh[:n.value]


CACHE_STATIC_MAX_IDS = 1 << 22   # TG_CACHE_STATIC_MAX_IDS of include/fasttg.h


def cache_lookup_static(uniq_ids: torch.Tensor, slot_of_id: torch.Tensor, map_out: torch.Tensor, fresh_out: torch.Tensor):
    """tg_cache_lookup_static: tg_cache_lookup without a workspace, for callers that must not allocate device memory
    (fixed memory pool, no allocator of their own, no cudaMalloc on the serving thread).  The caller passes both outputs
    (map_out int32 [>= U], fresh_out int64 [>= U]); nothing is allocated here or in the library.  Returns n_fresh; the
    valid results are map_out[:U] and fresh_out[:n_fresh].  U <= CACHE_STATIC_MAX_IDS, else FastTGError (TG_ERR_WORKSPACE).
    Calls on one device share the library's built-in scratch and must not overlap on the GPU."""
    U = int(uniq_ids.shape[0])
    if not (uniq_ids.is_contiguous() and slot_of_id.is_contiguous() and map_out.is_contiguous() and fresh_out.is_contiguous()):
        raise ValueError("cache_lookup_static: tensors must be contiguous (a copy would allocate)")
    if map_out.dtype != torch.int32 or fresh_out.dtype != torch.int64 or map_out.numel() < U or fresh_out.numel() < U:
        raise ValueError("cache_lookup_static: map_out int32 [>= U] and fresh_out int64 [>= U] are required")
    n = C.c_int64(0)
    _check(lib().tg_cache_lookup_static(C.c_int64(U), _ptr(uniq_ids), _ptr(slot_of_id), _ptr(map_out), _ptr(fresh_out), C.byref(n),
                                        _stream()), "tg_cache_lookup_static")
    return int(n.value)


def feature_reconstruct(inv_idx, map_: torch.Tensor, fresh_rows: torch.Tensor, cache_rows: torch.Tensor, out: torch.Tensor | None = None):
    """tg_feature_reconstruct: rows [n, ...] of the occurrences listed by inv_idx (None: one per map entry)."""
    n = int(inv_idx.shape[0]) if inv_idx is not None else int(map_.shape[0])
    fresh_rows, cache_rows = fresh_rows.contiguous(), cache_rows.contiguous()
    tail = tuple(fresh_rows.shape[1:])
    row_bytes = int(fresh_rows[0].numel() * fresh_rows.element_size()) if fresh_rows.shape[0] else int(cache_rows[0].numel() * cache_rows.element_size())
    if out is None:
        out = torch.empty((n,) + tail, dtype=fresh_rows.dtype, device=map_.device)
    _check(lib().tg_feature_reconstruct(C.c_int64(n), C.c_int64(row_bytes), _ptr(inv_idx), _ptr(map_), _ptr(fresh_rows), _ptr(cache_rows),
                                        _ptr(out), _stream()), "tg_feature_reconstruct")
    return out


class TCSR:
    """Per-node, time-ordered incidence lists on the device (tg_tcsr_build)."""

    def __init__(self, n_nodes, indptr, nbr, eid, ts):
        self.n_nodes, self.indptr, self.nbr, self.eid, self.ts = n_nodes, indptr, nbr, eid, ts


def tcsr_build(n_nodes: int, u: torch.Tensor, v: torch.Tensor, t: torch.Tensor) -> TCSR:
    """tg_tcsr_build.  u, v int64 [M], t float32 [M] (CUDA, stream order = time order)."""
    assert u.is_cuda and u.dtype == torch.int64 and v.dtype == torch.int64 and t.dtype == torch.float32
    u, v, t = u.contiguous(), v.contiguous(), t.contiguous()
    M = int(u.shape[0])
    dev = u.device
    indptr = torch.empty(n_nodes + 1, dtype=torch.int64, device=dev)
    nbr = torch.empty(2 * M, dtype=torch.int64, device=dev)
    eid = torch.empty(2 * M, dtype=torch.int64, device=dev)
    ts = torch.empty(2 * M, dtype=torch.float32, device=dev)
    nb = C.c_size_t()
    _check(lib().tg_tcsr_workspace_bytes(C.c_int64(n_nodes), C.c_int64(M), C.byref(nb)), "tg_tcsr_workspace_bytes")
    ws = torch.empty(nb.value, dtype=torch.uint8, device=dev)
    _check(lib().tg_tcsr_build(C.c_int64(n_nodes), C.c_int64(M), _ptr(u), _ptr(v), _ptr(t), _ptr(indptr), _ptr(nbr), _ptr(eid), _ptr(ts),
                               _ptr(ws), C.c_size_t(nb.value), _stream()), "tg_tcsr_build")
    return TCSR(n_nodes, indptr, nbr, eid, ts)


def sample_neighbors(g: TCSR, root_node: torch.Tensor, root_cutoff: torch.Tensor, k: int, mode: str = "recent", seed: int = 0):
    """tg_sample_neighbors: returns tg_block_build's inputs (root_idx int32, nbr_node int64, edge_id int64, ts float32), E entries."""
    assert root_node.is_cuda and root_node.dtype == torch.int64 and root_cutoff.dtype == torch.int64
    root_node, root_cutoff = root_node.contiguous(), root_cutoff.contiguous()
    n = int(root_node.shape[0])
    dev = root_node.device
    cap = max(n * k, 1)
    root_idx = torch.empty(cap, dtype=torch.int32, device=dev)
    nbr = torch.empty(cap, dtype=torch.int64, device=dev)
    eid = torch.empty(cap, dtype=torch.int64, device=dev)
    ts = torch.empty(cap, dtype=torch.float32, device=dev)
    nb = C.c_size_t()
    _check(lib().tg_sample_workspace_bytes(C.c_int64(n), C.byref(nb)), "tg_sample_workspace_bytes")
    ws = torch.empty(nb.value, dtype=torch.uint8, device=dev)
    E = C.c_int64(0)
    _check(lib().tg_sample_neighbors(C.c_int({"recent": 0, "uniform": 1}[mode]), C.c_int(k), C.c_uint64(seed), C.c_int64(n), _ptr(root_node),
                                     _ptr(root_cutoff), C.c_int64(g.n_nodes), _ptr(g.indptr), _ptr(g.nbr), _ptr(g.eid), _ptr(g.ts),
                                     _ptr(root_idx), _ptr(nbr), _ptr(eid), _ptr(ts), C.byref(E), _ptr(ws), C.c_size_t(nb.value), _stream()),
           "tg_sample_neighbors")
    e = int(E.value)
    return root_idx[:e], nbr[:e], eid[:e], ts[:e]


def block_coo_dst(b: Block) -> torch.Tensor:
    """tg_block_coo_dst: the COO row array (destination of every CSR edge), int32 [E]."""
    out = torch.empty(b.E, dtype=torch.int32, device=b.indptr.device)
    _check(lib().tg_block_coo_dst(b.handle, _ptr(out), _stream()), "tg_block_coo_dst")
    return out


def aggregate_coo(b: Block, X: torch.Tensor, coo_dst: torch.Tensor, backward: bool = False, out: torch.Tensor | None = None) -> torch.Tensor:
    """tg_aggregate_coo: the paper's COO / atomic plain sum; returns float32 [R or U, H, D]."""
    _rows(X, "X")
    H, D = X.shape[1], X.shape[2]
    rows = b.U if backward else b.R
    Y = out if out is not None else torch.empty(rows, H, D, dtype=torch.float32, device=X.device)
    _check(lib().tg_aggregate_coo(b.handle, C.c_int(H), C.c_int(D), C.c_int(_dt(X)), C.c_int(1 if backward else 0), _ptr(coo_dst),
                                  _ptr(X), _ptr(Y), _stream()), "tg_aggregate_coo")
    return Y
