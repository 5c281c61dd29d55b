"""Pins of the NEXT-1 oracle (oracle.attn_edge_fwd / attn_edge_bwd: per-edge additive key/value rows + LeakyReLU).

None of these re-types the oracle's loops: they tie it to (a) the already pinned base oracle on the cases where the
edge term reduces to it, (b) a dense NumPy evaluation written from the formulas with explicit per-destination
matrices, (c) a hand-derived one-neighbour closed form, (d) central finite differences of L = sum dO*O for all five
gradients, on both sides of the LeakyReLU kink, (e) identities that hold for any input.
"""
import numpy as np
import pytest


def _block(rng, R, max_deg, U):
    deg = rng.integers(0, max_deg + 1, size=R)
    indptr = np.zeros(R + 1, np.int32)
    np.cumsum(deg, out=indptr[1:])
    kv = rng.integers(0, U, size=int(indptr[-1])).astype(np.int32)
    return indptr, kv


def _rand(rng, *shape):
    return rng.standard_normal(shape)


def test_reduces_to_base_attention(oracle_mod):
    """Ke = Ve = 0 (or None) and slope = 1 is the base fused attention; adding Ke to K rows that are private to one
    edge is the same as the edge term."""
    rng = np.random.default_rng(0)
    R, U, H, D = 40, 25, 2, 6
    indptr, kv = _block(rng, R, 9, U)
    E = len(kv)
    Q, K, V, dO = _rand(rng, R, H, D), _rand(rng, U, H, D), _rand(rng, U, H, D), _rand(rng, R, H, D)
    O0, L0 = oracle_mod.attn_fwd(indptr, kv, Q, K, V, 0.7)
    for Ke, Ve in ((None, None), (np.zeros((E, H, D)), np.zeros((E, H, D)))):
        O1, L1 = oracle_mod.attn_edge_fwd(indptr, kv, Q, K, V, Ke, Ve, 0.7, 1.0)
        assert np.allclose(O0, O1, rtol=0, atol=1e-14) and np.array_equal(np.isneginf(L0), np.isneginf(L1))
        assert np.allclose(L0[~np.isneginf(L0)], L1[~np.isneginf(L1)], rtol=0, atol=1e-14)
        dQ0, dK0, dV0 = oracle_mod.attn_bwd(indptr, kv, Q, K, V, dO, 0.7)
        dQ1, dK1, dV1, dKe, dVe = oracle_mod.attn_edge_bwd(indptr, kv, Q, K, V, Ke, Ve, dO, 0.7, 1.0)
        assert np.allclose(dQ0, dQ1, atol=1e-13) and np.allclose(dK0, dK1, atol=1e-13) and np.allclose(dV0, dV1, atol=1e-13)
    # per-edge rows folded into private K/V rows: identity-mode base attention on K2 = K[kv] + Ke, V2 = V[kv] + Ve
    Ke, Ve = _rand(rng, E, H, D), _rand(rng, E, H, D)
    ident = np.arange(E, dtype=np.int32)
    O2, L2 = oracle_mod.attn_fwd(indptr, ident, Q, K[kv] + Ke, V[kv] + Ve, 0.7)
    O3, L3 = oracle_mod.attn_edge_fwd(indptr, kv, Q, K, V, Ke, Ve, 0.7, 1.0)
    assert np.allclose(O2, O3, atol=1e-13)
    dQ2, dK2, dV2 = oracle_mod.attn_bwd(indptr, ident, Q, K[kv] + Ke, V[kv] + Ve, dO, 0.7)
    dQ3, dK3, dV3, dKe3, dVe3 = oracle_mod.attn_edge_bwd(indptr, kv, Q, K, V, Ke, Ve, dO, 0.7, 1.0)
    assert np.allclose(dQ2, dQ3, atol=1e-13) and np.allclose(dK2, dKe3, atol=1e-13) and np.allclose(dV2, dVe3, atol=1e-13)


def _dense_forward(indptr, kv, Q, K, V, Ke, Ve, scale, slope):
    """explicit per-destination matrices, NumPy only"""
    R, H, D = Q.shape
    O = np.zeros_like(Q)
    for v in range(R):
        e = np.arange(indptr[v], indptr[v + 1])
        if len(e) == 0:
            continue
        Kd = K[kv[e]] + Ke[e]                      # [n, H, D]
        Vd = V[kv[e]] + Ve[e]
        z = scale * np.einsum("hd,nhd->nh", Q[v], Kd)
        s = np.where(z > 0, z, slope * z)
        a = np.exp(s - s.max(0))
        a /= a.sum(0)
        O[v] = np.einsum("nh,nhd->hd", a, Vd)
    return O


@pytest.mark.parametrize("slope", [1.0, 0.2, 0.0])
def test_dense_numpy_and_one_neighbour(oracle_mod, slope):
    rng = np.random.default_rng(1)
    R, U, H, D = 30, 12, 3, 5
    indptr, kv = _block(rng, R, 7, U)
    E = len(kv)
    Q, K, V, Ke, Ve = _rand(rng, R, H, D), _rand(rng, U, H, D), _rand(rng, U, H, D), _rand(rng, E, H, D), _rand(rng, E, H, D)
    O, L = oracle_mod.attn_edge_fwd(indptr, kv, Q, K, V, Ke, Ve, 1.3, slope)
    assert np.allclose(O, _dense_forward(indptr, kv, Q, K, V, Ke, Ve, 1.3, slope), atol=1e-12)
    # one neighbour: alpha = 1, O = V + Ve, LSE = lrelu(z); dQ = 0, dKe = 0 (softmax of one logit is constant), dVe = dO
    ip1 = np.array([0, 1], np.int32); kv1 = np.array([4], np.int32)
    O1, L1 = oracle_mod.attn_edge_fwd(ip1, kv1, Q[:1], K, V, Ke[:1], Ve[:1], 1.3, slope)
    z = 1.3 * np.einsum("hd,hd->h", Q[0], K[4] + Ke[0])
    assert np.allclose(O1[0], V[4] + Ve[0], atol=1e-14) and np.allclose(L1[0], np.where(z > 0, z, slope * z), atol=1e-14)
    dO = _rand(rng, 1, H, D)
    dQ, dK, dV, dKe, dVe = oracle_mod.attn_edge_bwd(ip1, kv1, Q[:1], K, V, Ke[:1], Ve[:1], dO, 1.3, slope)
    assert np.abs(dQ).max() < 1e-14 and np.abs(dKe).max() < 1e-14 and np.allclose(dVe[0], dO[0]) and np.allclose(dV[4], dO[0])


@pytest.mark.parametrize("slope", [1.0, 0.3])
def test_finite_differences_all_gradients(oracle_mod, slope):
    rng = np.random.default_rng(2)
    R, U, H, D = 6, 5, 2, 3
    indptr, kv = _block(rng, R, 4, U)
    E = len(kv)
    T = dict(Q=_rand(rng, R, H, D), K=_rand(rng, U, H, D), V=_rand(rng, U, H, D), Ke=_rand(rng, E, H, D), Ve=_rand(rng, E, H, D))
    dO = _rand(rng, R, H, D)
    scale = 0.9

    def loss(t):
        O, _ = oracle_mod.attn_edge_fwd(indptr, kv, t["Q"], t["K"], t["V"], t["Ke"], t["Ve"], scale, slope)
        return float((O * dO).sum())

    # keep every pre-activation away from the kink so that central differences are valid
    z = scale * np.einsum("ehd,ehd->eh", T["Q"][np.repeat(np.arange(R), np.diff(indptr))], T["K"][kv] + T["Ke"])
    assert np.abs(z).min() > 1e-3
    g = dict(zip(("Q", "K", "V", "Ke", "Ve"), oracle_mod.attn_edge_bwd(indptr, kv, T["Q"], T["K"], T["V"], T["Ke"], T["Ve"], dO, scale, slope)))
    h = 1e-6
    for name in ("Q", "K", "V", "Ke", "Ve"):
        num = np.zeros_like(T[name])
        it = np.nditer(T[name], flags=["multi_index"])
        for _ in it:
            i = it.multi_index
            tp = {k: v.copy() for k, v in T.items()}; tm = {k: v.copy() for k, v in T.items()}
            tp[name][i] += h; tm[name][i] -= h
            num[i] = (loss(tp) - loss(tm)) / (2 * h)
        assert np.allclose(g[name], num, rtol=1e-6, atol=1e-7), name


def test_identities(oracle_mod):
    rng = np.random.default_rng(3)
    R, U, H, D = 50, 20, 2, 4
    indptr, kv = _block(rng, R, 12, U)
    E = len(kv)
    Q, K, V, Ke, Ve, dO = (_rand(rng, *s) for s in ((R, H, D), (U, H, D), (U, H, D), (E, H, D), (E, H, D), (R, H, D)))
    dQ, dK, dV, dKe, dVe = oracle_mod.attn_edge_bwd(indptr, kv, Q, K, V, Ke, Ve, dO, 0.8, 0.2)
    deg = np.diff(indptr)
    dst = np.repeat(np.arange(R), deg)
    # dK / dV are the sums of the per-edge terms over the edges that reference the row
    ref_dK = np.zeros_like(dK); np.add.at(ref_dK, kv, dKe)
    ref_dV = np.zeros_like(dV); np.add.at(ref_dV, kv, dVe)
    assert np.allclose(dK, ref_dK, atol=1e-13) and np.allclose(dV, ref_dV, atol=1e-13)
    # sum of dVe over a destination's edges = dO of that destination (alphas sum to 1)
    s = np.zeros_like(dO); np.add.at(s, dst, dVe)
    assert np.allclose(s[deg > 0], dO[deg > 0], atol=1e-13)
    # sum over a destination's edges of dz = 0 when slope = 1; <Q,dQ> = sum_e <K[r]+Ke, dKe>
    assert np.isclose((Q * dQ).sum(), ((K[kv] + Ke) * dKe).sum(), rtol=1e-12)
    # shifting every key of a destination along q changes all its logits by the same amount when slope = 1: O unchanged
    O1, _ = oracle_mod.attn_edge_fwd(indptr, kv, Q, K, V, Ke, Ve, 0.8, 1.0)
    shift = 0.37 * Q[dst] / (Q[dst] ** 2).sum(-1, keepdims=True)
    O2, _ = oracle_mod.attn_edge_fwd(indptr, kv, Q, K, V, Ke + shift, Ve, 0.8, 1.0)
    assert np.allclose(O1, O2, atol=1e-12)
