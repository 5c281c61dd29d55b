"""Helpers shared by the `-m gpu` parity tests: move a seeded Workload to the device, run the C-ABI
path through the binding, run the oracle on the same arrays, compare with BASELINE.json's tolerances.

Tolerances (BASELINE.json north_star): fp32 storage |gpu - ref| <= 1e-5 + 1e-4*|ref|;
bf16 storage with fp32 accumulation |gpu - ref| <= 1e-3 + 2e-2*|ref|.  In addition the max error
relative to the tensor's largest magnitude is bounded (SURVEY.md §8(c) "tolerance hazard"), so an
all-zero small-magnitude gradient cannot pass.
"""
import numpy as np
import torch

TOL = {"f32": (1e-5, 1e-4, 5e-5), "bf16": (1e-3, 2e-2, 1.5e-2)}   # atol, rtol, max-normalised error
TDT = {"f32": torch.float32, "bf16": torch.bfloat16}


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.to(dtype)


def host(t):
    return t.detach().float().cpu().numpy() if t.is_floating_point() else t.detach().cpu().numpy()


def gpu_block(B, w, dedup=None):
    return B.block_build(w.R, dev(w.root_idx), dev(w.nbr_node), dev(w.edge_id), dev(w.ts),
                         w.dedup_mode if dedup is None else dedup)


def assert_close(name, got, ref, dtype, extra_atol=0.0):
    """extra_atol (scalar or array): an additional absolute term a test derives from the arithmetic
    (condition number of a long fp32 sum, logit-scale amplification); 0 for the BASELINE.json bound."""
    atol, rtol, nmax = TOL[dtype]
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape, (name, got.shape, ref.shape)
    if got.size == 0:
        return
    inf = np.isneginf(ref)
    assert np.array_equal(np.isneginf(got), inf), f"{name}: -inf pattern differs"
    g, r = got[~inf], ref[~inf]
    extra = np.broadcast_to(np.asarray(extra_atol, dtype=np.float64), ref.shape)[~inf]
    assert np.all(np.isfinite(g)), f"{name}: non-finite values"
    err = np.abs(g - r)
    bad = err > atol + rtol * np.abs(r) + extra
    assert not bad.any(), f"{name}: {bad.sum()} of {bad.size} outside |d| <= {atol} + {rtol}|ref|; worst {err.max():.3e} at ref {r[np.argmax(err)]:.3e}"
    if r.size and np.abs(r).max() > 100 * atol:      # a tensor that is ~0 everywhere is judged by atol alone
        n = np.max(np.maximum(err - extra, 0.0)) / np.abs(r).max()
        assert n <= nmax, f"{name}: max error / max |ref| = {n:.3e} > {nmax}"


def run_fused(B, blk, w, feats, scale):
    """GPU fused forward + backward through the C ABI; returns host float arrays."""
    q, k, v, do = (dev(x, TDT[w.dtype]) for x in feats)
    O, lse = B.attn_fused_fwd(blk, q, k, v, scale)
    dQ, dK, dV = B.attn_fused_bwd(blk, q, k, v, O, lse, do, scale)
    torch.cuda.synchronize()
    return tuple(host(x) for x in (O, lse, dQ, dK, dV))


def oracle_fused(oracle, ob, feats, scale):
    q, k, v, do = feats
    O, LSE = oracle.attn_fwd(ob.indptr, ob.kv_row, q, k, v, scale)
    dQ, dK, dV = oracle.attn_bwd(ob.indptr, ob.kv_row, q, k, v, do, scale)
    return O, LSE, dQ, dK, dV
