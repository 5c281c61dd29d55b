"""`-m gpu` tests of SURVEY.md §8(f) next-4: block chaining and the plain-AGG workload.

* Config 2, CHAINED (SURVEY.md §4 names it as the integration test of forward / backward composition): hop 2's output rows
  are hop 1's K = V rows -- hop 2 has one root per hop-1 edge, so hop 1 runs with per-edge rows (dedup_mode 0) -- and the
  gradient flows back through both blocks: dO of hop 2 = dK + dV of hop 1.  The oracle is composed the same way in
  float64; every tensor of both hops is compared within BASELINE.json's fp32 tolerance.
* Plain AGG (PAPER.md:215 h_v = sum v_u) through both partitionings: the CSR gather (tg_aggregate_fwd / _bwd with w = NULL)
  and the paper's COO / atomic scheme (tg_aggregate_coo) against oracle.aggregate_fwd / _bwd.
"""
import numpy as np
import pytest
import torch

import workloads as W
from gpu_util import H_SUM, TDT, U32, assert_close, dev, gpu_block, host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2607_05095_b200 import binding
    binding.lib()
    return binding


def test_config2_chained(B, oracle_mod):
    w1, w2 = W.config2(0)
    assert w2.R == w1.E                                     # one hop-2 root per hop-1 edge (reading R21)
    b1 = gpu_block(B, w1, dedup=0)
    b2 = gpu_block(B, w2)
    o1 = oracle_mod.block_build(w1.R, w1.root_idx, w1.nbr_node, w1.edge_id, w1.ts, 0)
    o2 = oracle_mod.block_build(w2.R, w2.root_idx, w2.nbr_node, w2.edge_id, w2.ts, 1)
    assert np.array_equal(o1.perm, np.arange(w1.E))         # hop-1 CSR order = sampler order = hop-2 root order
    q1, _, _, do1 = w1.features(1)
    q2, k2, v2, _ = w2.features(o2.U)
    # ---- GPU: hop 2 forward, hop 1 forward on its rows, hop 1 backward, hop 2 backward ----
    tq1, tdo1, tq2, tk2, tv2 = (dev(x) for x in (q1, do1, q2, k2, v2))
    O2, L2 = B.attn_fused_fwd(b2, tq2, tk2, tv2, 1.0)
    O1, L1 = B.attn_fused_fwd(b1, tq1, O2, O2, 1.0)
    dQ1, dK1, dV1 = B.attn_fused_bwd(b1, tq1, O2, O2, O1, L1, tdo1, 1.0)
    dO2 = dK1 + dV1                                         # K = V = O2: both gradients land on the same rows
    dQ2, dK2, dV2 = B.attn_fused_bwd(b2, tq2, tk2, tv2, O2, L2, dO2, 1.0)
    torch.cuda.synchronize()
    # ---- oracle, composed the same way in float64 ----
    rO2, rL2 = oracle_mod.attn_fwd(o2.indptr, o2.kv_row, q2, k2, v2, 1.0)
    rO1, rL1 = oracle_mod.attn_fwd(o1.indptr, o1.kv_row, q1, rO2, rO2, 1.0)
    rdQ1, rdK1, rdV1 = oracle_mod.attn_bwd(o1.indptr, o1.kv_row, q1, rO2, rO2, do1, 1.0)
    rdO2 = rdK1 + rdV1
    rdQ2, rdK2, rdV2 = oracle_mod.attn_bwd(o2.indptr, o2.kv_row, q2, k2, v2, rdO2, 1.0)
    for n, g, r in (("O2", O2, rO2), ("LSE2", L2, rL2), ("O1", O1, rO1), ("LSE1", L1, rL1), ("dQ1", dQ1, rdQ1), ("dK1", dK1, rdK1),
                    ("dV1", dV1, rdV1), ("dO2", dO2, rdO2), ("dQ2", dQ2, rdQ2), ("dK2", dK2, rdK2), ("dV2", dV2, rdV2)):
        assert_close(f"config2_chained.{n}", host(g), r, "f32")


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("case", ["small", "hub"])
def test_plain_agg_csr_and_coo(B, oracle_mod, dtype, case):
    if case == "small":
        w = W.small_random(5, 700, 40, 300, 8, 16, dtype=dtype, shuffle=True)
    else:
        w = W.config4(0, R=3000)
        w.dtype = dtype
    ob = oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, 1)
    blk = gpu_block(B, w, dedup=1)
    _, _, v, do = w.features(ob.U)
    if dtype == "bf16":
        v, do = W.round_to_bf16(v), W.round_to_bf16(do)
    tv, tdo = dev(v, TDT[dtype]), dev(do, TDT[dtype])
    rY = oracle_mod.aggregate_fwd(ob.indptr, ob.kv_row, None, v)
    rdX, _ = oracle_mod.aggregate_bwd(ob.indptr, ob.kv_row, ob.U, None, None, do, want_dw=False)
    # CSR gather (w = NULL).  fp32 storage: a hot source row sums ~1e5 N(0,1) terms; an element whose terms cancel carries
    # their rounding, u*sqrt(h)*sum|terms| for chains + merge tree of depth h <= H_SUM
    hs = (U32 * np.sqrt(H_SUM)) if dtype == "f32" else 0.0
    assert_close(f"plain_agg_{case}.Y[csr]", host(B.aggregate_fwd(blk, None, tv)), rY, dtype, extra_atol=hs * _abs_sum(ob, v, False))
    assert_close(f"plain_agg_{case}.dX[csr]", host(B.aggregate_bwd(blk, None, None, tdo, want_dw=False)[0]), rdX, dtype, extra_atol=hs * _abs_sum(ob, do, True))
    # the paper's COO / atomic scheme: float32 output whatever the storage of X
    coo = B.block_coo_dst(blk)
    assert np.array_equal(host(coo), np.repeat(np.arange(w.R, dtype=np.int32), np.diff(ob.indptr)))
    assert_close(f"plain_agg_{case}.Y[coo]", host(B.aggregate_coo(blk, tv, coo)), rY, "f32", extra_atol=_sum_budget(ob, v, False))
    assert_close(f"plain_agg_{case}.dX[coo]", host(B.aggregate_coo(blk, tdo, coo, backward=True)), rdX, "f32", extra_atol=_sum_budget(ob, do, True))


def _abs_sum(ob, x, backward):
    return _sum_budget(ob, x, backward, counts=False)


def _sum_budget(ob, x, backward, counts=True):
    """fp32 atomics add the terms in arrival order: a plain recursive sum of n terms has the first-order bound
    (n - 1) * 2^-24 * sum |terms| (Higham, Accuracy and Stability of Numerical Algorithms, §4.2); computed on absolute values.
    counts=False: just sum |terms| per output element."""
    ax = np.abs(x).astype(np.float64)
    if backward:
        s = np.zeros((ob.U,) + x.shape[1:])
        dst = np.repeat(np.arange(ob.R), np.diff(ob.indptr))
        np.add.at(s, ob.kv_row, ax[dst])
        n = np.bincount(ob.kv_row, minlength=ob.U)
    else:
        s = np.zeros((ob.R,) + x.shape[1:])
        dst = np.repeat(np.arange(ob.R), np.diff(ob.indptr))
        np.add.at(s, dst, ax[ob.kv_row])
        n = np.diff(ob.indptr)
    if not counts:
        return s
    return np.maximum(n - 1, 0).reshape(-1, 1, 1) * 2.0 ** -24 * s
