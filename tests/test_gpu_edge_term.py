"""`-m gpu` parity of NEXT-1 (tg_attn_edge_fused_fwd / _bwd: per-edge additive key/value rows + LeakyReLU) against
oracle.attn_edge_fwd / attn_edge_bwd on the same seeded inputs: small ragged blocks (all degree classes, zero-degree
rows), blocks with multi-chunk destination hubs and a hot source row, both sides of the LeakyReLU, both storage types."""
import math

import numpy as np
import pytest
import torch

import workloads as W
from gpu_util import TDT, assert_close, dev, gpu_block, host
from test_gpu_parity import _hub_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2607_05095_b200 import binding
    binding.lib()
    return binding


def _edge_rows(w, E):
    rng = np.random.default_rng([w.seed, 777, E])
    ke = (rng.standard_normal((E, w.H, w.D)) / math.sqrt(w.D)).astype(np.float32)
    ve = (rng.standard_normal((E, w.H, w.D)) / math.sqrt(w.D)).astype(np.float32)
    if w.dtype == "bf16":
        ke, ve = W.round_to_bf16(ke), W.round_to_bf16(ve)
    return ke, ve


def _compare(B, oracle_mod, w, scale, slope):
    ob = oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, w.dedup_mode)
    gb = gpu_block(B, w)
    q, k, v, do = w.features(ob.U)
    ke, ve = _edge_rows(w, w.E)
    dt = TDT[w.dtype]
    tq, tk, tv, tke, tve, tdo = (dev(x, dt) for x in (q, k, v, ke, ve, do))
    O, lse = B.attn_edge_fused_fwd(gb, tq, tk, tv, tke, tve, scale, slope)
    got_b = B.attn_edge_fused_bwd(gb, tq, tk, tv, tke, tve, O, lse, tdo, scale, slope)
    torch.cuda.synchronize()
    rO, rL = oracle_mod.attn_edge_fwd(ob.indptr, ob.kv_row, q, k, v, ke, ve, scale, slope)
    ref_b = oracle_mod.attn_edge_bwd(ob.indptr, ob.kv_row, q, k, v, ke, ve, do, scale, slope)
    assert_close("O", host(O), rO, w.dtype)
    assert_close("LSE", host(lse), rL, w.dtype)
    for n, g, r in zip(("dQ", "dK", "dV", "dKe", "dVe"), got_b, ref_b):
        assert_close(n, host(g), r, w.dtype)
    deg = np.diff(ob.indptr)
    assert np.all(host(O)[deg == 0] == 0) and np.all(np.isneginf(host(lse)[deg == 0]))


@pytest.mark.parametrize("slope", [1.0, 0.2])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("H,D", [(2, 50), (4, 32), (8, 16), (2, 64)])
def test_edge_term_small_blocks(B, oracle_mod, H, D, dtype, slope):
    w = W.small_random(300 + H * D, 400, 40, 90, H, D, dtype=dtype, shuffle=True, zero_frac=0.15)
    _compare(B, oracle_mod, w, 2.0, slope)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("H,D", [(2, 50), (4, 32), (8, 16), (2, 64)])
def test_edge_term_with_hubs(B, oracle_mod, H, D, dtype):
    w = _hub_workload(17 + H, H, D, dtype, hub_deg=6000)
    _compare(B, oracle_mod, w, float(math.sqrt(D)), 0.2)


def test_edge_term_reduces_to_base_on_gpu(B):
    """Ke = Ve = 0 and slope = 1: the edge-term kernels give the base fused kernels' result (independent code paths)."""
    w = W.small_random(5, 600, 70, 150, 8, 16, dtype="bf16", shuffle=True)
    gb = gpu_block(B, w)
    q, k, v, do = (dev(x, torch.bfloat16) for x in w.features(gb.U))
    z = torch.zeros(w.E, 8, 16, device="cuda", dtype=torch.bfloat16)
    O0, l0 = B.attn_fused_fwd(gb, q, k, v, 1.5)
    O1, l1 = B.attn_edge_fused_fwd(gb, q, k, v, z, z, 1.5, 1.0)
    torch.cuda.synchronize()
    assert torch.allclose(O0.float(), O1.float(), atol=2e-3, rtol=2e-2) and torch.allclose(l0[~torch.isinf(l0)], l1[~torch.isinf(l1)], atol=1e-4)
