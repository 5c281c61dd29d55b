"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Index structures bit-exact; floating point within BASELINE.json's tolerances.
Sizes are chosen so that every degree tier (group tier up to 8 / up to the side's group_max edges, warp-tier chunks of
64..1024 edges, hub rows merged from several chunks) and a ragged tail are exercised while the oracle still finishes in seconds."""
import math

import numpy as np
import pytest
import torch

import workloads as W

from gpu_util import C_BUDGET, H_SUM, TDT, U32, assert_close, assert_close_budget, dev, fp32_budget, gpu_block, host, oracle_fused, run_fused

pytestmark = pytest.mark.gpu

SHAPES = [(2, 50), (4, 32), (8, 16), (2, 64)]


@pytest.fixture(scope="module")
def B():
    from paper_2607_05095_b200 import binding
    binding.lib()
    assert torch.cuda.is_available(), "no CUDA device: the product path has no CPU fallback"
    return binding


def _oblock(oracle_mod, w, dedup=None):
    return oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, w.dedup_mode if dedup is None else dedup)


def _hub_workload(seed, H, D, dtype, n_hub_dst=2, hub_deg=20000, n_src=300, src_hub_frac=0.6, R=700, max_deg=300):
    """Mixed block: random small/warp/cta rows + a few destination hubs (several cta chunks) + one hot source row
    referenced by a large share of all edges (source-side hub with partial merge)."""
    w = W.small_random(seed, R, max_deg, n_src, H, D, dtype=dtype, zero_frac=0.1)
    r = np.random.default_rng(seed + 1000)
    deg = np.bincount(w.root_idx, minlength=R)
    hub_rows = r.choice(R, size=n_hub_dst, replace=False)
    extra_root = np.repeat(hub_rows.astype(np.int32), hub_deg)
    extra_nbr = r.integers(0, n_src, size=len(extra_root)).astype(np.int64) * 7 + 3
    hot = r.random(len(extra_root)) < src_hub_frac
    extra_nbr[hot] = 3                                      # node id 3 = source rank 0: the hot row
    w.root_idx = np.concatenate([w.root_idx, extra_root]).astype(np.int32)
    w.nbr_node = np.concatenate([w.nbr_node, extra_nbr])
    p = r.permutation(len(w.root_idx))                      # unsorted sampler order
    w.root_idx, w.nbr_node = w.root_idx[p], w.nbr_node[p]
    w.edge_id = np.arange(len(p), dtype=np.int64)
    w.ts = r.random(len(p), dtype=np.float32)
    return w


# ------------------------------------------------------------------------------------------------
# index structures: bit-exact
# ------------------------------------------------------------------------------------------------

def _block_cases():
    yield W.small_random(1, 40, 6, 12, 2, 4, shuffle=True)
    yield W.small_random(2, 3000, 20, 500, 2, 4, shuffle=True)
    yield W.small_random(3, 3000, 20, 500, 2, 4, shuffle=False)
    yield W.small_random(4, 5, 3000, 3, 2, 4, shuffle=True)
    yield W.small_random(5, 100, 3, 1, 2, 4, shuffle=True)
    yield W.small_random(6, 2500, 700, 4000, 2, 4, shuffle=True, zero_frac=0.3)
    yield W.config1(seed=0)


@pytest.mark.parametrize("w", list(_block_cases()), ids=lambda w: w.name)
@pytest.mark.parametrize("dedup", [0, 1])
def test_block_build_bit_exact(B, oracle_mod, w, dedup):
    ob = _oblock(oracle_mod, w, dedup)
    gb = gpu_block(B, w, dedup)
    assert gb.U == ob.U
    for name in ("indptr", "perm", "kv_row", "uniq_node", "t_indptr", "t_edge", "t_dst", "eid_csr", "ts_csr"):
        got, ref = host(getattr(gb, name)), getattr(ob, name)
        assert got.dtype == ref.dtype and np.array_equal(got, ref), name
    info = gb.info()
    assert info["R"] == w.R and info["E"] == w.E and info["U"] == ob.U
    # Schedule statistics against the block's own parameters (tg_block_sched_info), exactly, on both sides.  A side with
    # >= 2^20 edges keeps rows of up to 64 edges in the group tier; a launch-bound side uses the build's smaller limit.
    sched = gb.sched_info()
    for side, ptr in (("dst", ob.indptr), ("src", ob.t_indptr[:ob.U + 1])):
        deg = np.diff(ptr)
        lim, chunk = sched[side + "_group_max"], sched[side + "_chunk"]
        assert lim == 64 if w.E >= (1 << 20) else lim in (16, 32), (side, sched)
        want_chunk = 64
        while want_chunk < 1024 and w.E // want_chunk > 148 * 16 * 4:
            want_chunk *= 2
        assert chunk == want_chunk, (side, sched)
        big = deg[deg > lim]
        assert info[side + "_group_small"] == int((deg <= 8).sum()), side
        assert info[side + "_group_big"] == int(((deg > 8) & (deg <= lim)).sum()), side
        assert info[side + "_warp_items"] == int(np.ceil(big / chunk).sum()), side
        assert sched[side + "_hubs"] == int((big > chunk).sum()), side
        assert info[side + "_slots"] == int(np.ceil(big[big > chunk] / chunk).sum()), side
        assert sched[side + "_max_deg"] == (int(deg.max()) if deg.size and deg.max() > 8 else 0), side


def test_block_build_speculation_is_sticky(B, oracle_mod):
    """A thread that alternates between blocks with different needs (sorted / shuffled lists, 16- / 17-bit neighbour ids)
    repeats a build only when the need grows: the hint follows the largest recent need (tg_block_build_retries)."""
    narrow = W.small_random(21, 300, 9, 200, 2, 4, shuffle=False)           # sorted roots, ids < 2^16
    wide = W.small_random(22, 300, 9, 200, 2, 4, shuffle=True)
    wide.nbr_node = wide.nbr_node + (1 << 16)                                # shuffled roots, 17-bit ids: one more radix pass
    ref = {id(w): _oblock(oracle_mod, w, 1) for w in (narrow, wide)}
    gpu_block(B, wide, 1)                                                     # whatever the hint was, it now covers `wide`
    before = B.block_build_retries()
    for w in (narrow, wide) * 6:
        gb = gpu_block(B, w, 1)
        for name in ("indptr", "perm", "kv_row", "uniq_node", "t_indptr", "t_edge", "t_dst"):
            assert np.array_equal(host(getattr(gb, name)), getattr(ref[id(w)], name)), (w.name, name)
    assert B.block_build_retries() == before, "alternating builds must not re-run once the hint covers the larger one"
    for _ in range(10):                                                       # a long run of small builds relaxes the hint ...
        gpu_block(B, narrow, 1)
    gpu_block(B, wide, 1)                                                     # ... and the next large one pays one retry
    assert B.block_build_retries() == before + 1


@pytest.mark.parametrize("where", ["tail", "middle", "head", "short_gaps_only"])
def test_block_build_long_runs_of_empty_rows(B, oracle_mod, where):
    """Sorted lists with R >> E: a run of empty destinations longer than the in-kernel fill handles (>= 32 rows) is
    filled by the search kernel; runs just below the limit stay on the single-pass path.  Bit-exact either way."""
    rng = np.random.default_rng(5)
    R = 2_000_003
    if where == "short_gaps_only":
        R = 40_000
        roots = np.arange(0, R, 31)                                           # gaps of 30 empty rows, none at the tail beyond 31
    else:
        lo = {"tail": 0, "middle": 0, "head": R - 700}[where]
        roots = np.sort(rng.integers(lo, lo + 700, size=1500))
        if where == "middle":
            roots = np.concatenate([roots, [R - 1, R - 1]])
    E = len(roots)
    nbr = rng.integers(0, 300, size=E).astype(np.int64)
    ob = oracle_mod.block_build(R, roots.astype(np.int32), nbr, None, None, 1)
    gb = B.block_build(R, dev(roots.astype(np.int32)), dev(nbr), None, None, 1)
    for name in ("indptr", "perm", "kv_row", "uniq_node", "t_indptr", "t_edge", "t_dst"):
        assert np.array_equal(host(getattr(gb, name)), getattr(ob, name)), (where, name)
    assert gb.info()["dst_group_small"] == int((np.diff(ob.indptr) <= 8).sum())


def test_block_build_reuses_preallocated_outputs(B, oracle_mod):
    """block_build(reuse=...): a second build into the first one's arrays and workspace (no allocation) gives the oracle's
    block for the NEW lists; a Block of another shape is refused."""
    w1 = W.small_random(31, 900, 14, 300, 2, 4, shuffle=True)
    w2 = W.small_random(31, 900, 14, 300, 2, 4, shuffle=True)
    w2.nbr_node = (w2.nbr_node * 5 + 1) % 977                             # same shape, other neighbours
    g = gpu_block(B, w1, 1)
    ptrs = (g.indptr.data_ptr(), g.kv_row.data_ptr(), g.t_edge.data_ptr())
    g2 = B.block_build(w2.R, dev(w2.root_idx), dev(w2.nbr_node), dev(w2.edge_id), dev(w2.ts), 1, reuse=g)
    assert ptrs == (g2.indptr.data_ptr(), g2.kv_row.data_ptr(), g2.t_edge.data_ptr()) and not g.handle
    ob = _oblock(oracle_mod, w2, 1)
    assert g2.U == ob.U
    for name in ("indptr", "perm", "kv_row", "uniq_node", "t_indptr", "t_edge", "t_dst", "eid_csr", "ts_csr"):
        assert np.array_equal(host(getattr(g2, name)), getattr(ob, name)), name
    w3 = W.small_random(32, 901, 14, 300, 2, 4, shuffle=True)
    with pytest.raises(ValueError):
        B.block_build(w3.R, dev(w3.root_idx), dev(w3.nbr_node), dev(w3.edge_id), dev(w3.ts), 1, reuse=g2)


def test_block_build_negative_ids_and_empty(B, oracle_mod):
    w = W.small_random(7, 50, 9, 30, 2, 4, shuffle=True)
    w.nbr_node = w.nbr_node - 100                           # negative node ids: full 64-bit key sort
    ob = _oblock(oracle_mod, w, 1)
    gb = gpu_block(B, w, 1)
    for name in ("kv_row", "uniq_node", "t_indptr", "t_edge", "t_dst"):
        assert np.array_equal(host(getattr(gb, name)), getattr(ob, name)), name
    e = B.block_build(3, dev(np.zeros(0, np.int32)), dev(np.zeros(0, np.int64)), None, None, 1)
    assert e.U == 0 and host(e.indptr).tolist() == [0, 0, 0, 0] and host(e.t_indptr).tolist() == [0]
    e0 = B.block_build(0, dev(np.zeros(0, np.int32)), dev(np.zeros(0, np.int64)), None, None, 0)
    assert e0.U == 0 and host(e0.indptr).tolist() == [0]
    with pytest.raises(B.FastTGError) as ei:
        B.block_build(2, dev(np.array([0, 2], np.int32)), dev(np.array([1, 1], np.int64)), None, None, 1)
    assert ei.value.status == 1


# ------------------------------------------------------------------------------------------------
# fused forward + backward
# ------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("dtype", ["f32", "bf16", "bf16+o32"])
@pytest.mark.parametrize("H,D", SHAPES + [(1, 128), (2, 32), (4, 16), (2, 128)])
def test_fused_small_blocks(B, oracle_mod, H, D, dtype):
    """degrees 0..40: small + warp tiers, zero-degree rows, ragged group tails.  'bf16+o32': the forward also writes its
    float32 copy of O and the backward takes delta = <dO, O> from it instead of accumulating it from the edges."""
    side_copy = dtype.endswith("+o32")
    dtype = dtype.split("+")[0]
    w = W.small_random(100 + H * D, 500, 40, 120, H, D, dtype=dtype, shuffle=True, zero_frac=0.15)
    ob = _oblock(oracle_mod, w)
    gb = gpu_block(B, w)
    feats = w.features(ob.U)
    scale = 2.0
    got = run_fused(B, gb, w, feats, scale, side_copy=side_copy)
    ref = oracle_fused(oracle_mod, ob, feats, scale)
    for n, g, r in zip(("O", "LSE", "dQ", "dK", "dV"), got, ref):
        assert_close(n, g, r, dtype)
    deg = np.diff(ob.indptr)
    assert np.all(got[0][deg == 0] == 0) and np.all(got[2][deg == 0] == 0)      # zero-degree: O = dQ = 0, LSE = -inf


@pytest.mark.parametrize("dtype", ["f32", "bf16", "bf16+o32"])
@pytest.mark.parametrize("H,D", SHAPES)
def test_fused_all_tiers_with_hubs(B, oracle_mod, H, D, dtype):
    """warp tier, multi-chunk destination hubs (partial (m,l,acc) merge) and a hot source row (dK/dV partial merge)."""
    side_copy = dtype.endswith("+o32")
    dtype = dtype.split("+")[0]
    w = _hub_workload(7 + H, H, D, dtype)
    ob = _oblock(oracle_mod, w)
    gb = gpu_block(B, w)
    info = gb.info()
    assert info["dst_slots"] >= 4 and info["src_slots"] >= 2 and info["dst_warp_items"] >= info["dst_slots"]
    feats = w.features(ob.U)
    scale = float(math.sqrt(D))                                              # logits ~ N(0,1): softmax far from uniform
    got = run_fused(B, gb, w, feats, scale, side_copy=side_copy)
    ref = oracle_fused(oracle_mod, ob, feats, scale)
    for n, g, r in zip(("O", "LSE", "dQ", "dK", "dV"), got, ref):
        assert_close(n, g, r, dtype)


@pytest.mark.parametrize("scale", [1.0, 1e4])
def test_fused_degree_thresholds_and_large_logits(B, oracle_mod, scale):
    """A spread of degrees from 0 to 16385 (group tier, warp tier, hub rows of up to 257 chunks on this launch-bound side) and
    logits x 1e4 (max subtraction).  The schedule's own thresholds are straddled one by one in
    test_fused_straddles_every_schedule_threshold below."""
    degs = [0, 1, 2, 7, 8, 9, 10, 255, 256, 257, 258, 8191, 8192, 8193, 16384, 16385]
    H, D = 2, 64
    root = np.repeat(np.arange(len(degs), dtype=np.int32), degs)
    r = np.random.default_rng(5)
    nbr = r.integers(0, 2000, size=len(root)).astype(np.int64)
    w = W.Workload("thresholds", 98, 5, len(degs), H, D, "f32", scale, 1, root, nbr, np.arange(len(root), dtype=np.int64),
                   r.random(len(root), dtype=np.float32))
    ob = _oblock(oracle_mod, w)
    gb = gpu_block(B, w)
    feats = w.features(ob.U)
    got = run_fused(B, gb, w, feats, scale)
    ref = oracle_fused(oracle_mod, ob, feats, scale)
    # Saturating logits: |s| ~ scale * |<q,k>|.  fp32 holds a logit and the stored LSE to |s| * 2^-24, so alpha = exp(s - LSE)
    # carries a relative error of that size per edge and ds = alpha*(dalpha - delta) cancels down to it; the extra absolute
    # term is the fp32 rounding budget of DESIGN.md §6.4 (computed by the oracle on absolute values).  At scale = 1 the
    # budget is far below BASELINE.json's bound, which is then the one that binds.
    bud = fp32_budget(oracle_mod, ob.indptr, ob.kv_row, ob.U, feats, scale)
    for n, g, r_ in zip(("O", "LSE", "dQ", "dK", "dV"), got, ref):
        if n in bud:
            assert_close_budget(f"thresholds[scale={scale:g}].{n}", g, r_, "f32", bud[n])
        else:
            assert_close(n, g, r_, "f32")


def _straddle(*thresholds):
    return sorted({d for t in thresholds for d in (t - 1, t, t + 1) if d >= 0})


@pytest.mark.parametrize("side", ["launch_bound", "large"])
def test_fused_straddles_every_schedule_threshold(B, oracle_mod, side):
    """Destination AND source degrees at t-1, t, t+1 for every threshold of the schedule the block actually got
    (tg_block_sched_info): the degree classes (2, 4, 8, 16, 32, 64), the side's group-tier limit, one warp item
    (chunk), the direct hub merge (TG_HUB_DIRECT = 32 chunks) and beyond.  'launch_bound': a side below 2^20 edges
    (group limit 32, chunk 64, one CTA per hub); 'large': >= 2^20 edges (group limit 64, forked tiers, two-level hub merge)."""
    rng = np.random.default_rng(17)
    if side == "launch_bound":
        H, D, dtype, group_max, chunk, filler = 2, 64, "f32", 32, 64, (0, 0)
    else:
        H, D, dtype, group_max, chunk, filler = 8, 16, "bf16", 64, 128, (4000, 260)
    degs = _straddle(1, 2, 4, 8, 16, 32, 64, group_max, chunk, 2 * chunk, 32 * chunk, 33 * chunk) + [0, 0, 3 * 32 * chunk + 5]
    dst_deg = np.array(degs + [filler[1]] * filler[0])
    E = int(dst_deg.sum())
    src_deg = np.array([d for d in degs if d > 0])
    assert src_deg.sum() <= E
    rest = E - int(src_deg.sum())                                     # the remaining edges go to sources of degree ~ 3 and ~ 40
    extra = []
    while rest > 0:
        d = min(rest, int(rng.choice([1, 2, 3, 5, 40])))
        extra.append(d); rest -= d
    src_deg = np.concatenate([src_deg, np.array(extra, dtype=np.int64)])
    root = np.repeat(np.arange(len(dst_deg), dtype=np.int32), dst_deg)
    nbr = rng.permutation(np.repeat(np.arange(len(src_deg), dtype=np.int64) * 3 + 11, src_deg))
    w = W.Workload("straddle_" + side, 97, 17, len(dst_deg), H, D, dtype, 1.0, 1, root, nbr, np.arange(E, dtype=np.int64),
                   rng.random(E, dtype=np.float32))
    ob = _oblock(oracle_mod, w)
    gb = gpu_block(B, w)
    sched = gb.sched_info()
    assert (E >= (1 << 20)) == (side == "large")
    for k in ("dst", "src"):                                           # the thresholds this test was written against
        assert sched[k + "_group_max"] == group_max and sched[k + "_chunk"] == chunk, sched
        assert sched[k + "_hubs"] >= 9 and sched[k + "_max_deg"] == 3 * 32 * chunk + 5
    assert np.array_equal(np.sort(np.diff(ob.t_indptr)), np.sort(src_deg))
    feats = w.features(ob.U)
    got = run_fused(B, gb, w, feats, 1.0)
    ref = oracle_fused(oracle_mod, ob, feats, 1.0)
    bud = fp32_budget(oracle_mod, ob.indptr, ob.kv_row, ob.U, feats, 1.0) if dtype == "f32" else {}
    for n, g, r_ in zip(("O", "LSE", "dQ", "dK", "dV"), got, ref):
        if n in bud:
            assert_close_budget(f"straddle[{side}].{n}", g, r_, dtype, bud[n])
        else:
            assert_close(f"straddle[{side}].{n}", g, r_, dtype)


def test_fused_identity_rows_and_single_source(B, oracle_mod):
    """dedup_mode 0 (per-edge K/V rows, config 1 as written) and U = 1 (all edges share one source row)."""
    w = W.small_random(21, 300, 12, 40, 2, 50, shuffle=True, dedup_mode=0)
    ob = _oblock(oracle_mod, w)
    gb = gpu_block(B, w)
    assert gb.U == w.E
    feats = w.features(ob.U)
    for n, g, r in zip(("O", "LSE", "dQ", "dK", "dV"), run_fused(B, gb, w, feats, 1.5), oracle_fused(oracle_mod, ob, feats, 1.5)):
        assert_close(n, g, r, "f32")
    w = W.small_random(22, 400, 30, 1, 4, 32, dtype="bf16", shuffle=True)
    ob = _oblock(oracle_mod, w)
    gb = gpu_block(B, w)
    assert gb.U == 1
    feats = w.features(1)
    for n, g, r in zip(("O", "LSE", "dQ", "dK", "dV"), run_fused(B, gb, w, feats, 3.0), oracle_fused(oracle_mod, ob, feats, 3.0)):
        assert_close(n, g, r, "bf16")


def test_fused_bitwise_reproducible(B):
    """no float atomics anywhere: two runs give identical bits."""
    w = _hub_workload(3, 8, 16, "bf16")
    gb = gpu_block(B, w)
    feats = w.features(gb.U)
    a = run_fused(B, gb, w, feats, 4.0)
    b = run_fused(B, gb, w, feats, 4.0)
    for x, y in zip(a, b):
        assert np.array_equal(x, y, equal_nan=True)


def test_block_from_csr_and_empty_blocks(B, oracle_mod):
    """tg_block_from_csr wraps index arrays the caller already has (here: the oracle's); empty blocks are TG_OK."""
    w = _hub_workload(11, 4, 32, "f32", hub_deg=3000)
    ob = _oblock(oracle_mod, w)
    gb = B.block_from_csr(dev(ob.indptr), dev(ob.kv_row), ob.U, dev(ob.t_indptr), dev(ob.t_edge), dev(ob.t_dst))
    assert gb.info()["E"] == w.E and gb.info()["U"] == ob.U
    feats = w.features(ob.U)
    for n, g, r in zip(("O", "LSE", "dQ", "dK", "dV"), run_fused(B, gb, w, feats, 1.5), oracle_fused(oracle_mod, ob, feats, 1.5)):
        assert_close(n, g, r, "f32")
    # R = 3 destinations without any edge: O = 0, LSE = -inf, dQ = 0, nothing to write on the source side
    e = B.block_build(3, dev(np.zeros(0, np.int32)), dev(np.zeros(0, np.int64)), None, None, 1)
    q = torch.randn(3, 8, 16, device="cuda").bfloat16()
    kv = torch.zeros(0, 8, 16, device="cuda", dtype=torch.bfloat16)
    O, lse = B.attn_fused_fwd(e, q, kv, kv, 1.0)
    dQ, dK, dV = B.attn_fused_bwd(e, q, kv, kv, O, lse, q, 1.0)
    torch.cuda.synchronize()
    assert float(O.float().abs().max()) == 0.0 and bool(torch.isneginf(lse).all()) and float(dQ.float().abs().max()) == 0.0
    assert dK.shape[0] == 0 and dV.shape[0] == 0
    e0 = B.block_build(0, dev(np.zeros(0, np.int32)), dev(np.zeros(0, np.int64)), None, None, 1)
    q0 = torch.zeros(0, 8, 16, device="cuda", dtype=torch.bfloat16)
    O0, lse0 = B.attn_fused_fwd(e0, q0, kv, kv, 1.0)
    assert O0.shape[0] == 0 and lse0.shape[0] == 0


def test_fused_cuda_graph_capture_and_side_stream(B):
    """The fused calls only enqueue (the group tiers fork onto the library's auxiliary streams and join back):
    they can be captured into a CUDA graph on a non-default stream, and the replay gives the eager bits."""
    w = W.config4(0, R=30000)                     # E ~ 1.5 M: large enough for the fork / join path
    gb = gpu_block(B, w)
    q, k, v, do = (dev(x, torch.bfloat16) for x in w.features(gb.U))
    O, lse = B.attn_fused_fwd(gb, q, k, v, 1.0)
    dQ, dK, dV = B.attn_fused_bwd(gb, q, k, v, O, lse, do, 1.0)
    torch.cuda.synchronize()
    ref = [t.clone() for t in (O, lse, dQ, dK, dV)]
    for t in (O, lse, dQ, dK, dV):
        t.zero_()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.graph(g, stream=side):
        B.attn_fused_fwd(gb, q, k, v, 1.0, out=(O, lse))
        B.attn_fused_bwd(gb, q, k, v, O, lse, do, 1.0, out=(dQ, dK, dV))
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    for a, b in zip(ref, (O, lse, dQ, dK, dV)):
        assert torch.equal(a, b)


# ------------------------------------------------------------------------------------------------
# unfused operators
# ------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("H,D", SHAPES)
def test_unfused_chain(B, oracle_mod, H, D, dtype):
    w = _hub_workload(40 + H, H, D, dtype, hub_deg=9000)
    ob = _oblock(oracle_mod, w)
    gb = gpu_block(B, w)
    q, k, v, do = w.features(ob.U)
    tq, tk, tv, tdo = (dev(x, TDT[dtype]) for x in (q, k, v, do))
    scale = float(math.sqrt(D))
    # SDDMM
    s_ref = oracle_mod.sddmm(ob.indptr, ob.kv_row, q, k, scale)
    s = B.sddmm(gb, tq, tk, scale)
    assert_close("s", host(s), s_ref, "f32" if dtype == "f32" else "bf16")
    # ESM forward on the oracle's logits (isolates the operator)
    s_in = dev(s_ref.astype(np.float32))
    a_ref = oracle_mod.edge_softmax_fwd(ob.indptr, host(s_in))
    alpha = B.edge_softmax_fwd(gb, s_in)
    assert_close("alpha", host(alpha), a_ref, "f32")
    sums = np.add.reduceat(host(alpha).astype(np.float64), ob.indptr[:-1][np.diff(ob.indptr) > 0], axis=0)
    np.testing.assert_allclose(sums, 1.0, atol=2e-5)
    # AGG forward, weighted and plain
    a_in = dev(a_ref.astype(np.float32))
    y_ref = oracle_mod.aggregate_fwd(ob.indptr, ob.kv_row, host(a_in), v)
    assert_close("Y", host(B.aggregate_fwd(gb, a_in, tv)), y_ref, dtype)
    y0_ref = oracle_mod.aggregate_fwd(ob.indptr, ob.kv_row, None, v)
    assert_close("Y_plain", host(B.aggregate_fwd(gb, None, tv)), y0_ref, dtype)
    # AGG backward: dX through the transposed CSR, dw
    dx_ref, dw_ref = oracle_mod.aggregate_bwd(ob.indptr, ob.kv_row, ob.U, host(a_in), v, do)
    dX, dw = B.aggregate_bwd(gb, a_in, tv, tdo)
    # Long fp32 sums: the hot source row adds ~10^4 terms, thousands of them identical (multi-edges of one hub), and the
    # two hubs' contributions can cancel.  Extra absolute term = the summation part of the fp32 rounding budget of
    # C_BUDGET * u * sqrt(H_SUM) * sum|terms|; sum|terms| comes from the oracle on absolute values.
    gamma = C_BUDGET * U32 * math.sqrt(H_SUM)
    cond, _ = oracle_mod.aggregate_bwd(ob.indptr, ob.kv_row, ob.U, np.abs(host(a_in)), None, np.abs(do), want_dw=False)
    assert_close_budget(f"unfused[{H}x{D},{dtype}].dX", host(dX), dx_ref, dtype, gamma * cond)
    assert_close("dw", host(dw), dw_ref, "f32" if dtype == "f32" else "bf16")
    dx0_ref, _ = oracle_mod.aggregate_bwd(ob.indptr, ob.kv_row, ob.U, None, None, do, want_dw=False)
    dX0, none = B.aggregate_bwd(gb, None, None, tdo, want_dw=False)
    assert none is None
    cond0, _ = oracle_mod.aggregate_bwd(ob.indptr, ob.kv_row, ob.U, None, None, np.abs(do), want_dw=False)
    assert_close_budget(f"unfused[{H}x{D},{dtype}].dX_plain", host(dX0), dx0_ref, dtype, gamma * cond0)
    # ESM backward
    da_in = dev(dw_ref.astype(np.float32))
    ds_ref = oracle_mod.edge_softmax_bwd(ob.indptr, host(a_in), host(da_in))
    assert_close("ds", host(B.edge_softmax_bwd(gb, a_in, da_in)), ds_ref, "f32")


def test_unfused_chain_equals_fused(B, oracle_mod):
    """the DGL-style chain sddmm -> softmax -> aggregate and its backward reproduce the fused path."""
    w = W.small_random(60, 800, 60, 200, 4, 32, shuffle=True)
    gb = gpu_block(B, w)
    q, k, v, do = (dev(x) for x in w.features(gb.U))
    scale = 2.5
    O, lse = B.attn_fused_fwd(gb, q, k, v, scale)
    dQ, dK, dV = B.attn_fused_bwd(gb, q, k, v, O, lse, do, scale)
    alpha = B.edge_softmax_fwd(gb, B.sddmm(gb, q, k, scale))
    O2 = B.aggregate_fwd(gb, alpha, v)
    dV2, dalpha = B.aggregate_bwd(gb, alpha, v, do)
    ds = B.edge_softmax_bwd(gb, alpha, dalpha)
    dQ2 = B.aggregate_fwd(gb, ds, k) * scale
    dK2, _ = B.aggregate_bwd(gb, ds, None, q, want_dw=False)
    for n, x, y in (("O", O, O2), ("dV", dV, dV2), ("dQ", dQ, dQ2), ("dK", dK, dK2 * scale)):
        assert_close(n, host(x), host(y).astype(np.float64), "f32")


# ------------------------------------------------------------------------------------------------
# error behaviour of the boundary
# ------------------------------------------------------------------------------------------------

def test_boundary_errors(B):
    w = W.small_random(70, 50, 9, 30, 2, 50, shuffle=True)
    gb = gpu_block(B, w)
    q, k, v, do = (dev(x) for x in w.features(gb.U))
    with pytest.raises(B.FastTGError) as ei:                                  # (H, D) outside the compiled set
        B.attn_fused_fwd(gb, q[:, :, :48].contiguous(), k[:, :, :48].contiguous(), v[:, :, :48].contiguous(), 1.0)
    assert ei.value.status == 2
    buf = torch.empty(q.numel() + 1, dtype=torch.float32, device="cuda")
    q_mis = buf[1:].view_as(q)                                                # 4-byte offset: not 16-byte aligned
    q_mis.copy_(q)
    with pytest.raises(B.FastTGError) as ei:
        B.attn_fused_fwd(gb, q_mis, k, v, 1.0)
    assert ei.value.status == 3
    assert B.supported(8, 16, torch.bfloat16) and not B.supported(3, 16, torch.float32)
