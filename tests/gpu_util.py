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

# (name, used fraction of the bound = max err / (atol + rtol*|ref| + extra), max err / max |ref|) of every comparison;
# tests/conftest.py prints the table in the terminal summary so that the margin of each tensor is visible.
MARGINS = []


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
    bound = atol + rtol * np.abs(r) + extra
    used = float(np.max(err / bound)) if r.size else 0.0
    rmax = float(np.abs(r).max()) if r.size else 0.0
    nerr = float(np.max(np.maximum(err - extra, 0.0)) / rmax) if rmax > 0 else 0.0
    MARGINS.append((name, dtype, used, nerr, int(r.size)))
    bad = err > bound
    assert not bad.any(), f"{name}: {bad.sum()} of {bad.size} outside |d| <= {atol} + {rtol}|ref|; worst {err.max():.3e} at ref {r[np.argmax(err)]:.3e}"
    # Second gate (SURVEY.md §8(c) "tolerance hazard"): the absolute term must not hide an all-wrong small tensor.
    # Applied whenever the tensor has any element that the relative term can see (max |ref| > atol).
    if rmax > atol:
        assert nerr <= nmax, f"{name}: max error / max |ref| = {nerr:.3e} > {nmax}"
    return used


def run_fused(B, blk, w, feats, scale, side_copy=False):
    """GPU fused forward + backward through the C ABI; returns host float arrays.
    side_copy: the forward also writes its float32 copy of O and the backward takes delta from it (bf16 storage)."""
    q, k, v, do = (dev(x, TDT[w.dtype]) for x in feats)
    o32 = torch.empty(q.shape, dtype=torch.float32, device=q.device) if side_copy else None
    O, lse = B.attn_fused_fwd(blk, q, k, v, scale, o32=o32)
    dQ, dK, dV = B.attn_fused_bwd(blk, q, k, v, O, lse, do, scale, o32=o32)
    torch.cuda.synchronize()
    return tuple(host(x) for x in (O, lse, dQ, dK, dV))


def oracle_fused(oracle, ob, feats, scale):
    q, k, v, do = feats
    O, LSE = oracle.attn_fwd(ob.indptr, ob.kv_row, q, k, v, scale)
    dQ, dK, dV = oracle.attn_bwd(ob.indptr, ob.kv_row, q, k, v, do, scale)
    return O, LSE, dQ, dK, dV


def slab_source_rows(oracle_mod, indptr, kv_row, feats, scale, src_rows, slab_edges):
    """dK, dV of the listed source rows as float64 sums of the oracle's results on destination slabs
    (each slab = a contiguous range of complete destinations with K/V compressed to the rows it references)."""
    q, k, v, do = feats
    R = len(indptr) - 1
    src_rows = np.asarray(src_rows, dtype=np.int64)
    dK = np.zeros((len(src_rows),) + k.shape[1:], np.float64)
    dV = np.zeros_like(dK)
    lo = 0
    while lo < R:
        hi = int(np.searchsorted(indptr, indptr[lo] + slab_edges, side="right")) - 1
        hi = min(max(hi, lo + 1), R)
        e0, e1 = int(indptr[lo]), int(indptr[hi])
        used, sub_kv = np.unique(kv_row[e0:e1], return_inverse=True)
        sub_indptr = (indptr[lo:hi + 1] - e0).astype(np.int32)
        _, sdK, sdV = oracle_mod.attn_bwd(sub_indptr, sub_kv.astype(np.int32), q[lo:hi], k[used], v[used], do[lo:hi], scale)
        loc = np.searchsorted(used, src_rows)
        ok = (loc < len(used))
        ok[ok] &= used[loc[ok]] == src_rows[ok]
        dK[ok] += sdK[loc[ok]]
        dV[ok] += sdV[loc[ok]]
        lo = hi
    return dK, dV


# ------------------------------------------------------------------------------------------------------------
# fp32 rounding budget.  BASELINE.json's fp32 bound 1e-5 + 1e-4*|ref| is relative to the RESULT;
# an element whose terms cancel (a gradient on a hot source row, a dQ element under logits of magnitude 30-40)
# carries the rounding of its TERMS.  The budget below is the first-order error model of evaluating the §2
# formulas in fp32, computed by the oracle on absolute values (no value comes from the CUDA path):
#   alpha_e has relative error  eta_e = u*(K_DOT*A_e + |LSE_v|),  A_e = sum_d |scale*q_d*k_d|   (fp32 logit and stored fp32 LSE)
#   delta_v = <dO_v, O_v> is taken from the forward's fp32 O, which carries the forward's own alpha errors:
#       |d delta_v| <= D_v = sum_{e in N(v)} alpha_e*(eta_e + u*sqrt(h))*B_e + u*K_DOT*C_v,
#       B_e = sum_d |dO_d v_d|, C_v = sum_d |dO_d O_d|
#   ds_e = alpha_e*(dalpha_e - delta_v) has absolute error  eta_e*|ds_e| + alpha_e*(u*K_DOT*B_e + D_v)
#   a sum over n terms evaluated as chains + merge tree of depth h adds  u*sqrt(h)*sum |terms|   (h <= H_SUM)
# u = 2^-24.  K_DOT = 2 bounds the measured fp32 logit error (tg_sddmm against the oracle on config 5: max 1.6 u*A_e, rms 0.22).
# C_BUDGET stays 1: the terminal summary prints the largest (error beyond the stated bound) / budget of every test that
# uses it, so the budget cannot hide an error that is not rounding.
# ------------------------------------------------------------------------------------------------------------
U32 = 2.0 ** -24
K_DOT = 2.0        # sqrt-type constant of a D-term fp32 dot product evaluated as two FMA chains + a shuffle tree
H_SUM = 288        # longest chain (1024-edge chunk over 4 groups = 256) + group / hub merge levels
C_BUDGET = 1.0


def fp32_budget(oracle, indptr, kv_row, U, feats, scale):
    """Per-element absolute rounding budgets {'dQ', 'dK', 'dV'} of the fused backward in fp32 (see above)."""
    q, k, v, do = (np.asarray(x, dtype=np.float64) for x in feats)
    indptr = np.asarray(indptr)
    R = len(indptr) - 1
    dst = np.repeat(np.arange(R), np.diff(indptr))
    s = oracle.sddmm(indptr, kv_row, q, k, scale)
    alpha = oracle.edge_softmax_fwd(indptr, s)
    O, LSE = oracle.attn_fwd(indptr, kv_row, q, k, v, scale)
    _, dalpha = oracle.aggregate_bwd(indptr, kv_row, U, alpha, v, do)
    ds = oracle.edge_softmax_bwd(indptr, alpha, dalpha)
    del s, dalpha
    A = oracle.sddmm(indptr, kv_row, np.abs(q), np.abs(k), abs(scale))
    Bd = oracle.sddmm(indptr, kv_row, np.abs(do), np.abs(v), 1.0)
    Cv = (np.abs(do) * np.abs(O)).sum(-1)
    lse_abs = np.where(np.isfinite(LSE), np.abs(LSE), 0.0)
    eta = U32 * (K_DOT * A + lse_abs[dst])
    del A
    hs = U32 * np.sqrt(H_SUM)
    Dv = U32 * K_DOT * Cv
    term = alpha * (eta + hs) * Bd
    for h in range(term.shape[1]):
        Dv[:, h] += np.bincount(dst, weights=term[:, h], minlength=R)
    del term
    w_ds = (eta + hs) * np.abs(ds) + alpha * (U32 * K_DOT * Bd + Dv[dst])
    w_dv = (eta + hs) * alpha
    del Bd, eta, ds, alpha
    out = {
        "dQ": abs(scale) * oracle.aggregate_fwd(indptr, kv_row, w_ds, np.abs(k)),
        "dK": abs(scale) * oracle.aggregate_bwd(indptr, kv_row, U, w_ds, None, np.abs(q), want_dw=False)[0],
        "dV": oracle.aggregate_bwd(indptr, kv_row, U, w_dv, None, np.abs(do), want_dw=False)[0],
    }
    return {n: C_BUDGET * x for n, x in out.items()}


BUDGET_USE = []   # (name, max (err - stated bound)+ / budget) of every comparison that was given a budget


def assert_close_budget(name, got, ref, dtype, budget):
    """assert_close with the derived fp32 rounding budget as the extra absolute term; records how much of the
    budget the elements that exceed the stated bound actually use."""
    atol, rtol, _ = TOL[dtype]
    g = np.asarray(got, dtype=np.float64)
    r = np.asarray(ref, dtype=np.float64)
    over = np.maximum(np.abs(g - r) - (atol + rtol * np.abs(r)), 0.0)
    n_over = int((over > 0).sum())
    use = float(np.max(over / np.maximum(budget, 1e-300))) if over.size else 0.0
    BUDGET_USE.append((name, use, n_over, int(over.size)))
    return assert_close(name, got, ref, dtype, extra_atol=budget)
