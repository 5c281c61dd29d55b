"""Pins for the oracle's floating-point functions (CPU only, `-m "not gpu"`).

Nothing here re-types the oracle's own loops: each test is a closed form, an invariant, a brute-force
enumeration in pure Python, a torch float64 library routine (scaled_dot_product_attention, softmax,
autograd on a padded-dense formulation) or a central finite difference.  Chosen so that a dropped
term, a wrong sign / index or a transposed operand in tg_oracle.c fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
import torch

import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
RTOL, ATOL = 1e-10, 1e-12


def _block(oracle_mod, w, dedup=None):
    return oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, w.dedup_mode if dedup is None else dedup)


def _rand_feats(seed, R, U, H, D):
    r = np.random.default_rng(seed)
    return (r.standard_normal((R, H, D)), r.standard_normal((U, H, D)), r.standard_normal((U, H, D)), r.standard_normal((R, H, D)))


def _dense_torch(indptr, kv_row, Q, K, V, scale):
    """Padded-dense masked-softmax formulation in torch float64 (library ops only)."""
    R = len(indptr) - 1
    deg = np.diff(indptr)
    n = max(int(deg.max()) if R else 0, 1)
    idx = np.zeros((R, n), np.int64)
    mask = np.zeros((R, n), bool)
    for v in range(R):
        idx[v, :deg[v]] = kv_row[indptr[v]:indptr[v + 1]]
        mask[v, :deg[v]] = True
    idx_t, mask_t = torch.from_numpy(idx), torch.from_numpy(mask)
    Kg, Vg = K[idx_t], V[idx_t]                                   # [R,n,H,D]
    s = scale * torch.einsum("rhd,rnhd->rnh", Q, Kg)
    s = s.masked_fill(~mask_t[:, :, None], float("-inf"))
    lse = torch.logsumexp(s, dim=1)
    a = torch.softmax(s, dim=1)
    a = torch.where(mask_t[:, :, None], a, torch.zeros_like(a))  # zero-degree rows: nan -> 0
    O = torch.einsum("rnh,rnhd->rhd", a, Vg)
    return O, lse, a, mask


# ------------------------------------------------------------------------------------------------
# closed forms and golden fixture
# ------------------------------------------------------------------------------------------------

def _golden():
    sym = {"ln3": math.log(3.0), "ln4": math.log(4.0)}
    out = {}
    for ln in open(os.path.join(GOLDEN, "two_neighbour_closed_form.txt")):
        if not ln.strip() or ln.startswith("#"):
            continue
        name, *vals = ln.split()
        out[name] = np.array([eval(x, {"__builtins__": {}}, sym) for x in vals], dtype=np.float64)
    return out


def test_golden_two_neighbour(oracle_mod):
    g = _golden()
    indptr = np.array([0, 2], np.int32)
    kv = np.array([0, 1], np.int32)
    Q = g["q"].reshape(1, 1, 1); K = g["k"].reshape(2, 1, 1); V = g["v"].reshape(2, 1, 1); dO = g["dO"].reshape(1, 1, 1)
    O, LSE, alpha = oracle_mod.attn_fwd(indptr, kv, Q, K, V, 1.0, want_alpha=True)
    np.testing.assert_allclose(alpha.ravel(), g["alpha"], rtol=1e-14)
    np.testing.assert_allclose(O.ravel(), g["O"], rtol=1e-14)
    np.testing.assert_allclose(LSE.ravel(), g["LSE"], rtol=1e-14)
    dQ, dK, dV = oracle_mod.attn_bwd(indptr, kv, Q, K, V, dO, 1.0)
    np.testing.assert_allclose(dQ.ravel(), g["dQ"], rtol=1e-13)
    np.testing.assert_allclose(dK.ravel(), g["dK"], rtol=1e-13)
    np.testing.assert_allclose(dV.ravel(), g["dV"], rtol=1e-13)
    # the same numbers through the unfused chain
    s = oracle_mod.sddmm(indptr, kv, Q, K, 1.0)
    np.testing.assert_allclose(s.ravel(), g["k"], rtol=1e-14)
    a = oracle_mod.edge_softmax_fwd(indptr, s)
    np.testing.assert_allclose(a.ravel(), g["alpha"], rtol=1e-14)
    ds = oracle_mod.edge_softmax_bwd(indptr, a, g["v"].reshape(2, 1))
    np.testing.assert_allclose(ds.ravel(), g["ds"], rtol=1e-13)


def test_single_neighbour_alpha_is_one(oracle_mod):
    R, H, D = 7, 2, 5
    indptr = np.arange(R + 1, dtype=np.int32)
    kv = np.arange(R, dtype=np.int32)[::-1].copy()
    Q, K, V, dO = _rand_feats(0, R, R, H, D)
    O, LSE, alpha = oracle_mod.attn_fwd(indptr, kv, Q, K, V, 0.7, want_alpha=True)
    assert np.all(alpha == 1.0)
    np.testing.assert_allclose(O, V[kv], rtol=1e-15)
    np.testing.assert_allclose(LSE, 0.7 * np.einsum("rhd,rhd->rh", Q, K[kv]), rtol=1e-13)
    dQ, dK, dV = oracle_mod.attn_bwd(indptr, kv, Q, K, V, dO, 0.7)
    assert np.all(dQ == 0) and np.all(dK == 0)            # alpha is constant => no gradient through logits
    np.testing.assert_allclose(dV[kv], dO, rtol=1e-15)


def test_equal_logits_give_mean(oracle_mod):
    H, D, n = 2, 4, 6
    indptr = np.array([0, n], np.int32)
    kv = np.arange(n, dtype=np.int32)
    r = np.random.default_rng(1)
    Q = r.standard_normal((1, H, D))
    K = np.broadcast_to(r.standard_normal((1, H, D)), (n, H, D)).copy()     # identical keys -> equal logits
    V = r.standard_normal((n, H, D))
    O, LSE, alpha = oracle_mod.attn_fwd(indptr, kv, Q, K, V, 1.3, want_alpha=True)
    np.testing.assert_allclose(alpha, 1.0 / n, rtol=1e-14)
    np.testing.assert_allclose(O[0], V.mean(axis=0), rtol=1e-13)
    s0 = 1.3 * np.einsum("hd,hd->h", Q[0], K[0])
    np.testing.assert_allclose(LSE[0], s0 + math.log(n), rtol=1e-13)


def test_two_neighbour_sigmoid(oracle_mod):
    r = np.random.default_rng(2)
    for _ in range(20):
        s = r.standard_normal((2, 3)) * 5
        a = oracle_mod.edge_softmax_fwd(np.array([0, 2], np.int32), s)
        np.testing.assert_allclose(a[0], 1.0 / (1.0 + np.exp(s[1] - s[0])), rtol=1e-13)
        np.testing.assert_allclose(a[1], 1.0 / (1.0 + np.exp(s[0] - s[1])), rtol=1e-13)


# ------------------------------------------------------------------------------------------------
# invariants (north_star list)
# ------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("seed", [0, 1])
def test_alpha_sums_shift_and_permutation_invariance(oracle_mod, seed):
    w = W.small_random(seed, 60, 12, 25, 2, 6)
    b = _block(oracle_mod, w)
    Q, K, V, dO = _rand_feats(seed, w.R, b.U, w.H, w.D)
    O, LSE, alpha = oracle_mod.attn_fwd(b.indptr, b.kv_row, Q, K, V, 2.0, want_alpha=True)
    deg = np.diff(b.indptr)
    sums = np.add.reduceat(alpha, b.indptr[:-1][deg > 0], axis=0) if b.E else np.zeros((0, w.H))
    np.testing.assert_allclose(sums, 1.0, rtol=1e-13)
    assert np.all(O[deg == 0] == 0) and np.all(np.isneginf(LSE[deg == 0]))
    # shift invariance: s + c_v leaves alpha unchanged, LSE moves by c_v
    s = oracle_mod.sddmm(b.indptr, b.kv_row, Q, K, 2.0)
    c = np.random.default_rng(seed + 10).standard_normal((w.R, w.H)) * 30
    dst = np.repeat(np.arange(w.R), deg)
    a0 = oracle_mod.edge_softmax_fwd(b.indptr, s)
    a1 = oracle_mod.edge_softmax_fwd(b.indptr, s + c[dst])
    np.testing.assert_allclose(a1, a0, rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(a0, alpha, rtol=1e-13)
    # permuting a destination's edges permutes alpha and leaves O, LSE unchanged
    rng = np.random.default_rng(seed + 20)
    kv2 = b.kv_row.copy()
    for v in range(w.R):
        seg = slice(b.indptr[v], b.indptr[v + 1])
        kv2[seg] = rng.permutation(kv2[seg])
    O2, LSE2 = oracle_mod.attn_fwd(b.indptr, kv2, Q, K, V, 2.0)
    np.testing.assert_allclose(O2, O, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(LSE2[deg > 0], LSE[deg > 0], rtol=1e-12)


def test_large_logits_stable(oracle_mod):
    """max-subtraction (PAPER.md:225 'numerically stable'): logits x 1e4 must not overflow."""
    w = W.small_random(3, 30, 9, 10, 2, 4)
    b = _block(oracle_mod, w)
    Q, K, V, dO = _rand_feats(3, w.R, b.U, w.H, w.D)
    O, LSE, alpha = oracle_mod.attn_fwd(b.indptr, b.kv_row, Q, K, V, 1e4, want_alpha=True)
    assert np.all(np.isfinite(O)) and np.all(np.isfinite(alpha))
    dQ, dK, dV = oracle_mod.attn_bwd(b.indptr, b.kv_row, Q, K, V, dO, 1e4)
    assert all(np.all(np.isfinite(x)) for x in (dQ, dK, dV))


# ------------------------------------------------------------------------------------------------
# brute force in pure Python on tiny graphs
# ------------------------------------------------------------------------------------------------

def test_brute_force_tiny(oracle_mod):
    w = W.small_random(5, 6, 4, 5, 2, 3)
    b = _block(oracle_mod, w)
    Q, K, V, dO = _rand_feats(5, w.R, b.U, w.H, w.D)
    scale = 0.9
    O, LSE, alpha = oracle_mod.attn_fwd(b.indptr, b.kv_row, Q, K, V, scale, want_alpha=True)
    H, D = w.H, w.D
    for v in range(w.R):
        edges = list(range(b.indptr[v], b.indptr[v + 1]))
        for h in range(H):
            s = [scale * sum(Q[v, h, d] * K[b.kv_row[e], h, d] for d in range(D)) for e in edges]
            if not edges:
                assert LSE[v, h] == -math.inf and all(O[v, h, d] == 0 for d in range(D))
                continue
            z = sum(math.exp(x) for x in s)                      # naive (unshifted) softmax is fine at this scale
            for i, e in enumerate(edges):
                assert abs(alpha[e, h] - math.exp(s[i]) / z) < 1e-13
            assert abs(LSE[v, h] - math.log(z)) < 1e-12
            for d in range(D):
                ref = sum(math.exp(s[i]) / z * V[b.kv_row[e], h, d] for i, e in enumerate(edges))
                assert abs(O[v, h, d] - ref) < 1e-12
    # unfused pieces
    s = oracle_mod.sddmm(b.indptr, b.kv_row, Q, K, scale)
    Y = oracle_mod.aggregate_fwd(b.indptr, b.kv_row, alpha, V)
    np.testing.assert_allclose(Y, O, rtol=1e-12, atol=1e-14)
    Ys = oracle_mod.aggregate_fwd(b.indptr, b.kv_row, None, V)   # the paper's plain AGG
    ref = np.zeros_like(Ys)
    dst = np.repeat(np.arange(w.R), np.diff(b.indptr))
    np.add.at(ref, dst, V[b.kv_row])
    np.testing.assert_allclose(Ys, ref, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(oracle_mod.edge_softmax_fwd(b.indptr, s), alpha, rtol=1e-12)


# ------------------------------------------------------------------------------------------------
# library special cases: SDPA on a regular block, padded-dense masked softmax in general
# ------------------------------------------------------------------------------------------------

def test_regular_block_is_sdpa(oracle_mod):
    R, n, H, D = 9, 7, 2, 8
    indptr = (np.arange(R + 1) * n).astype(np.int32)
    kv = np.arange(R * n, dtype=np.int32)                      # private rows per destination
    Q, K, V, dO = _rand_feats(7, R, R * n, H, D)
    scale = 1.0 / math.sqrt(D)
    O, LSE = oracle_mod.attn_fwd(indptr, kv, Q, K, V, scale)
    q = torch.from_numpy(Q).permute(1, 0, 2).reshape(H, R, 1, D).permute(1, 0, 2, 3)     # [R,H,1,D]
    k = torch.from_numpy(K).reshape(R, n, H, D).permute(0, 2, 1, 3)                      # [R,H,n,D]
    v = torch.from_numpy(V).reshape(R, n, H, D).permute(0, 2, 1, 3)
    ref = torch.nn.functional.scaled_dot_product_attention(q, k, v)                      # default scale 1/sqrt(D)
    np.testing.assert_allclose(O, ref[:, :, 0, :].numpy(), rtol=1e-11, atol=1e-13)


@pytest.mark.parametrize("cfg", ["small", "hub", "config1", "config1_dedup"])
def test_fwd_bwd_vs_torch_autograd(oracle_mod, cfg):
    if cfg == "small":
        w = W.small_random(8, 50, 10, 20, 2, 5); scale = 1.7
    elif cfg == "hub":
        w = W.small_random(9, 4, 300, 40, 3, 4, zero_frac=0.0); scale = 3.0
    elif cfg == "config1":
        w = W.config1(seed=0); scale = w.scale
    else:
        w = W.config1(seed=0, dedup_mode=1); scale = math.sqrt(50.0)
    b = _block(oracle_mod, w)
    Qn, Kn, Vn, dOn = (x.astype(np.float64) for x in w.features(b.U))
    Q, K, V = (torch.from_numpy(x).requires_grad_(True) for x in (Qn, Kn, Vn))
    O, lse, a, mask = _dense_torch(b.indptr, b.kv_row, Q, K, V, scale)
    O.backward(torch.from_numpy(dOn))
    Oo, LSEo, alpha = oracle_mod.attn_fwd(b.indptr, b.kv_row, Qn, Kn, Vn, scale, want_alpha=True)
    np.testing.assert_allclose(Oo, O.detach().numpy(), rtol=1e-10, atol=1e-13)
    deg = np.diff(b.indptr)
    np.testing.assert_allclose(LSEo[deg > 0], lse.detach().numpy()[deg > 0], rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(alpha, a.detach().numpy()[mask], rtol=1e-10, atol=1e-15)
    dQ, dK, dV = oracle_mod.attn_bwd(b.indptr, b.kv_row, Qn, Kn, Vn, dOn, scale)
    np.testing.assert_allclose(dQ, Q.grad.numpy(), rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(dK, K.grad.numpy(), rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(dV, V.grad.numpy(), rtol=1e-9, atol=1e-12)


def test_unfused_backward_vs_torch_autograd(oracle_mod):
    w = W.small_random(12, 40, 9, 15, 2, 4)
    b = _block(oracle_mod, w)
    r = np.random.default_rng(12)
    E, H, D = b.E, w.H, w.D
    dst = torch.from_numpy(np.repeat(np.arange(w.R), np.diff(b.indptr)))
    row = torch.from_numpy(b.kv_row.astype(np.int64))
    # aggregate: Y = index_add(w * X[row])
    wt = torch.from_numpy(r.standard_normal((E, H))).requires_grad_(True)
    X = torch.from_numpy(r.standard_normal((b.U, H, D))).requires_grad_(True)
    dY = r.standard_normal((w.R, H, D))
    Y = torch.zeros(w.R, H, D, dtype=torch.float64).index_add(0, dst, wt[:, :, None] * X[row])
    Y.backward(torch.from_numpy(dY))
    Yo = oracle_mod.aggregate_fwd(b.indptr, b.kv_row, wt.detach().numpy(), X.detach().numpy())
    np.testing.assert_allclose(Yo, Y.detach().numpy(), rtol=1e-11, atol=1e-13)
    dX, dw = oracle_mod.aggregate_bwd(b.indptr, b.kv_row, b.U, wt.detach().numpy(), X.detach().numpy(), dY)
    np.testing.assert_allclose(dX, X.grad.numpy(), rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(dw, wt.grad.numpy(), rtol=1e-10, atol=1e-13)
    # plain AGG backward (w = NULL): dX = index_add of dY rows
    dX0, _ = oracle_mod.aggregate_bwd(b.indptr, b.kv_row, b.U, None, None, dY, want_dw=False)
    ref = torch.zeros(b.U, H, D, dtype=torch.float64).index_add(0, row, torch.from_numpy(dY)[dst])
    np.testing.assert_allclose(dX0, ref.numpy(), rtol=1e-12, atol=1e-13)
    # edge softmax backward through torch softmax per destination
    s = torch.from_numpy(r.standard_normal((E, H)) * 3).requires_grad_(True)
    da = r.standard_normal((E, H))
    outs = []
    for v in range(w.R):
        seg = s[b.indptr[v]:b.indptr[v + 1]]
        if len(seg):
            outs.append(torch.softmax(seg, dim=0))
    a = torch.cat(outs, dim=0)
    a.backward(torch.from_numpy(da))
    ao = oracle_mod.edge_softmax_fwd(b.indptr, s.detach().numpy())
    np.testing.assert_allclose(ao, a.detach().numpy(), rtol=1e-12)
    dso = oracle_mod.edge_softmax_bwd(b.indptr, ao, da)
    np.testing.assert_allclose(dso, s.grad.numpy(), rtol=1e-9, atol=1e-13)
    # sddmm vs einsum
    A = r.standard_normal((w.R, H, D))
    so = oracle_mod.sddmm(b.indptr, b.kv_row, A, X.detach().numpy(), 0.37)
    ref = 0.37 * np.einsum("ehd,ehd->eh", A[dst.numpy()], X.detach().numpy()[b.kv_row])
    np.testing.assert_allclose(so, ref, rtol=1e-12, atol=1e-14)


# ------------------------------------------------------------------------------------------------
# central finite differences + gradient identities
# ------------------------------------------------------------------------------------------------

def test_backward_central_finite_differences(oracle_mod):
    w = W.small_random(13, 7, 5, 6, 2, 3)
    b = _block(oracle_mod, w)
    Q, K, V, dO = _rand_feats(13, w.R, b.U, w.H, w.D)
    scale = 1.1

    def loss(Q_, K_, V_):
        O, _ = oracle_mod.attn_fwd(b.indptr, b.kv_row, Q_, K_, V_, scale)
        return float(np.sum(dO * O))

    dQ, dK, dV = oracle_mod.attn_bwd(b.indptr, b.kv_row, Q, K, V, dO, scale)
    h = 1e-6
    rng = np.random.default_rng(0)
    for name, X, G in (("Q", Q, dQ), ("K", K, dK), ("V", V, dV)):
        flat = X.reshape(-1)
        for i in rng.choice(flat.size, size=min(40, flat.size), replace=False):
            old = flat[i]
            flat[i] = old + h; lp = loss(Q, K, V)
            flat[i] = old - h; lm = loss(Q, K, V)
            flat[i] = old
            fd = (lp - lm) / (2 * h)
            assert abs(fd - G.reshape(-1)[i]) < 1e-7 * (1 + abs(fd)), (name, i, fd, G.reshape(-1)[i])


@pytest.mark.parametrize("seed", [0, 1])
def test_gradient_identities(oracle_mod, seed):
    w = W.small_random(20 + seed, 80, 15, 30, 2, 6)
    b = _block(oracle_mod, w)
    Q, K, V, dO = _rand_feats(seed, w.R, b.U, w.H, w.D)
    scale = 1.9
    deg = np.diff(b.indptr)
    dQ, dK, dV = oracle_mod.attn_bwd(b.indptr, b.kv_row, Q, K, V, dO, scale)
    # sum_u dV[u] = sum_{v: deg>0} dO[v]   (alphas sum to one)
    np.testing.assert_allclose(dV.sum(axis=0), dO[deg > 0].sum(axis=0), rtol=1e-11, atol=1e-12)
    # sum <Q,dQ> = sum <K,dK>  (both equal sum_e ds*s)
    np.testing.assert_allclose(np.sum(Q * dQ), np.sum(K * dK), rtol=1e-10, atol=1e-12)
    # sum_{N(v)} ds = 0
    _, _, alpha = oracle_mod.attn_fwd(b.indptr, b.kv_row, Q, K, V, scale, want_alpha=True)
    dst = np.repeat(np.arange(w.R), deg)
    dalpha = np.einsum("ehd,ehd->eh", dO[dst], V[b.kv_row])
    ds = oracle_mod.edge_softmax_bwd(b.indptr, alpha, dalpha)
    seg = np.add.reduceat(ds, b.indptr[:-1][deg > 0], axis=0)
    np.testing.assert_allclose(seg, 0.0, atol=1e-12)
    # fused backward == unfused chain
    dQ2 = scale * oracle_mod.aggregate_fwd(b.indptr, b.kv_row, ds, K)
    dK2, _ = oracle_mod.aggregate_bwd(b.indptr, b.kv_row, b.U, ds, None, Q, want_dw=False)
    dV2, dal2 = oracle_mod.aggregate_bwd(b.indptr, b.kv_row, b.U, alpha, V, dO)
    np.testing.assert_allclose(dQ2, dQ, rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(scale * dK2, dK, rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(dV2, dV, rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(dal2, dalpha, rtol=1e-11, atol=1e-13)
    # all V rows equal => ds = 0 => dQ = dK = 0 exactly
    Vc = np.broadcast_to(V[:1], V.shape).copy()
    dQc, dKc, _ = oracle_mod.attn_bwd(b.indptr, b.kv_row, Q, K, Vc, dO, scale)
    assert np.max(np.abs(dQc)) < 1e-13 and np.max(np.abs(dKc)) < 1e-13
    # backward is linear in dO
    dQa, dKa, dVa = oracle_mod.attn_bwd(b.indptr, b.kv_row, Q, K, V, 2.5 * dO, scale)
    np.testing.assert_allclose(dQa, 2.5 * dQ, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(dKa, 2.5 * dK, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(dVa, 2.5 * dV, rtol=1e-11, atol=1e-13)


def test_online_merge_associativity():
    """(m,l,acc) split-and-merge (online normalizer, ref [16] at PAPER.md:225, 437) reproduces the 3-pass
    softmax: checked in numpy float64 on random split points; no oracle call (pins the algebra the CUDA path uses)."""
    r = np.random.default_rng(4)
    for _ in range(50):
        n = int(r.integers(1, 60))
        s = r.standard_normal(n) * 10
        x = r.standard_normal((n, 3))
        m = s.max(); p = np.exp(s - m); ref = (p[:, None] * x).sum(0) / p.sum(); ref_lse = m + math.log(p.sum())
        cuts = np.sort(r.integers(0, n + 1, size=int(r.integers(0, 5))))
        parts = []
        for a, bnd in zip(np.concatenate([[0], cuts]), np.concatenate([cuts, [n]])):
            if bnd > a:
                mm = s[a:bnd].max(); pp = np.exp(s[a:bnd] - mm)
                parts.append((mm, pp.sum(), (pp[:, None] * x[a:bnd]).sum(0)))
        r.shuffle(parts)
        M = max(q[0] for q in parts)
        L = sum(q[1] * math.exp(q[0] - M) for q in parts)
        A = sum(q[2] * math.exp(q[0] - M) for q in parts)
        np.testing.assert_allclose(A / L, ref, rtol=1e-12, atol=1e-14)
        assert abs(M + math.log(L) - ref_lse) < 1e-12


def test_slab_decomposition_of_source_gradients(oracle_mod):
    """dK / dV are sums over edges and a slab of complete destinations carries the block's softmax statistics:
    adding the oracle's per-slab results in float64 reproduces the oracle on the whole block (the host-memory
    fallback of tests/test_gpu_configs.py for config 5 rests on this)."""
    from gpu_util import slab_source_rows
    w = W.small_random(77, 400, 60, 150, 2, 8, shuffle=False)
    ob = oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, 1)
    feats = w.features(ob.U)
    q, k, v, do = feats
    _, dK, dV = oracle_mod.attn_bwd(ob.indptr, ob.kv_row, q, k, v, do, 1.7)
    rows = np.arange(0, ob.U, 3)
    sK, sV = slab_source_rows(oracle_mod, ob.indptr, ob.kv_row, feats, 1.7, rows, slab_edges=700)
    np.testing.assert_allclose(sK, dK[rows], rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(sV, dV[rows], rtol=1e-12, atol=1e-14)
