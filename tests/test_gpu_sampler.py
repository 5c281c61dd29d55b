"""`-m gpu` parity of the device-side temporal neighbour sampler against oracle/sampler_oracle.py:
tg_tcsr_build and tg_sample_neighbors are integer / byte work -- bit-exact (np.array_equal), timestamps included.

Cases: tiny streams with self-loops and repeated endpoints (every k, cutoffs 0..M, unknown nodes); the event streams of
configs 1 and 2 with their own roots (the sampled lists must equal the workload's lists, and the block built from them the
block built from the workload); a config-3-shaped uniform draw (1 M nodes, 5 M events -- the 50 M-event stream of config 3
takes minutes in the oracle's lexsort, the sampler code path does not depend on the stream length); empty inputs.
No expected value comes from the CUDA path.
"""
import numpy as np
import pytest
import torch

from oracle import sampler_oracle as S
import workloads as W
from gpu_util import dev, host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2607_05095_b200 import binding
    binding.lib()
    return binding


def _gpu_tcsr(B, n_nodes, u, v, t):
    return B.tcsr_build(n_nodes, dev(u.astype(np.int64)), dev(v.astype(np.int64)), dev(t.astype(np.float32)))


def _check_tcsr(g, o):
    m2 = int(o.indptr[-1])
    assert np.array_equal(host(g.indptr), o.indptr)
    assert np.array_equal(host(g.nbr)[:m2], o.nbr) and np.array_equal(host(g.eid)[:m2], o.eid)
    assert np.array_equal(host(g.ts)[:m2], o.ts)


def _check_sample(B, g, o, root_node, cutoff, k, mode, seed=0):
    got = B.sample_neighbors(g, dev(np.asarray(root_node, np.int64)), dev(np.asarray(cutoff, np.int64)), k, mode, seed)
    ref = S.sample_recent(o, root_node, cutoff, k) if mode == "recent" else S.sample_uniform(o, root_node, cutoff, k, seed)
    for a, b, n in zip(got, ref, ("root_idx", "nbr_node", "edge_id", "ts")):
        a = host(a)
        assert a.dtype == b.dtype and np.array_equal(a, b), (n, mode, k)
    return got


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_tiny_streams(B, seed):
    r = np.random.default_rng(seed)
    n_nodes, m = 9, 300
    u, v = r.integers(0, n_nodes, m), r.integers(0, n_nodes, m)
    u[::17] = v[::17]                                   # self-loops
    t = np.sort(r.random(m)).astype(np.float32)
    o = S.tcsr_build(n_nodes, u, v, t)
    g = _gpu_tcsr(B, n_nodes, u, v, t)
    _check_tcsr(g, o)
    root_node = r.integers(0, n_nodes, 500)
    cutoff = r.integers(0, m + 1, 500)
    for k in (1, 3, 10, 64):
        _check_sample(B, g, o, root_node, cutoff, k, "recent")
        _check_sample(B, g, o, root_node, cutoff, k, "uniform", seed=seed + 7)
    # zero cutoff: nothing is prior
    got = B.sample_neighbors(g, dev(root_node.astype(np.int64)), dev(np.zeros(500, np.int64)), 10, "recent")
    assert got[0].numel() == 0
    # empty root list
    e = torch.zeros(0, dtype=torch.int64, device="cuda")
    assert B.sample_neighbors(g, e, e, 10, "recent")[0].numel() == 0


def test_empty_stream(B):
    z = np.zeros(0, np.int64)
    g = _gpu_tcsr(B, 5, z, z, z.astype(np.float32))
    assert np.array_equal(host(g.indptr), np.zeros(6, np.int64))
    got = B.sample_neighbors(g, dev(np.array([1, 2], np.int64)), dev(np.array([5, 5], np.int64)), 4, "uniform", 3)
    assert got[0].numel() == 0


def test_tcsr_long_runs_of_nodes_without_events(B):
    """n_nodes >> M: the runs of event-free nodes are longer than the emit kernel fills itself (the search kernel writes
    tc_indptr then), including a run at the tail and self-loops, whose sentinel entries sort behind every node."""
    rng = np.random.default_rng(9)
    n_nodes, M = 1_500_007, 900
    u = rng.integers(0, 400, size=M)
    v = rng.integers(700_000, 700_300, size=M)
    u[::50] = v[::50]                                                        # some self-loops
    t = np.sort(rng.random(M)).astype(np.float32)
    o = S.tcsr_build(n_nodes, u, v, t)
    g = _gpu_tcsr(B, n_nodes, u, v, t)
    _check_tcsr(g, o)
    _check_sample(B, g, o, [int(v[-1]), int(u[3]), n_nodes - 1], [M, M, M], 5, "recent")


def _stream_case(B, oracle_mod, cid, n_nodes, n_events, k, hop2=False):
    seed = 0
    u, v, t = W._event_stream(seed, cid, n_nodes, n_events)
    o = S.tcsr_build(n_nodes, u, v, t)
    g = _gpu_tcsr(B, n_nodes, u, v, t)
    _check_tcsr(g, o)
    rn, rc = W._batch_roots(u, v, n_nodes, 600, seed, cid)
    return u, v, t, o, g, rn, rc


def test_config1_lists_and_block(B, oracle_mod):
    """PAPER.md:311's k = 10 most-recent sampling on config 1's stream: the device lists equal the workload's lists,
    and the block built from them is the oracle's block."""
    u, v, t, o, g, rn, rc = _stream_case(B, oracle_mod, 1, 20_000, 200_000, 10)
    got = _check_sample(B, g, o, rn, rc, 10, "recent")
    w = W.config1(0)
    for a, b in zip(got, (w.root_idx, w.nbr_node, w.edge_id, w.ts)):
        assert np.array_equal(host(a), b)
    blk = B.block_build(w.R, got[0], got[1], got[2], got[3], w.dedup_mode)
    ob = oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, w.dedup_mode)
    for name in ("indptr", "perm", "kv_row", "uniq_node", "t_indptr", "t_edge", "t_dst", "eid_csr", "ts_csr"):
        assert np.array_equal(host(getattr(blk, name)), getattr(ob, name)), name


def test_config2_two_hops(B, oracle_mod):
    u, v, t, o, g, rn, rc = _stream_case(B, oracle_mod, 2, 100_000, 5_000_000, 10)
    w1, w2 = W.config2(0)
    h1 = _check_sample(B, g, o, rn, rc, 10, "recent")
    for a, b in zip(h1, (w1.root_idx, w1.nbr_node, w1.edge_id, w1.ts)):
        assert np.array_equal(host(a), b)
    # hop 2: every hop-1 edge is a root (node = that neighbour, cutoff = that edge's event index); all on the device
    h2 = B.sample_neighbors(g, h1[1], h1[2], 10, "recent")
    for a, b in zip(h2, (w2.root_idx, w2.nbr_node, w2.edge_id, w2.ts)):
        assert np.array_equal(host(a), b)


def test_config3_shaped_uniform(B, oracle_mod):
    """k = 20 uniform-without-replacement over a Zipf(1.1) stream with 12 000 roots (config 3's shape; reading R28)."""
    seed, cid, n_nodes, n_events = 0, 3, 1_000_000, 5_000_000
    u, v, t = W._event_stream(seed, cid, n_nodes, n_events)
    o = S.tcsr_build(n_nodes, u, v, t)
    g = _gpu_tcsr(B, n_nodes, u, v, t)
    _check_tcsr(g, o)
    rn, rc = W._batch_roots(u, v, n_nodes, 4000, seed, cid)
    got = _check_sample(B, g, o, rn, rc, 20, "uniform", seed=2024)
    deg = np.bincount(host(got[0]), minlength=len(rn))
    assert deg.max() == 20 and (deg == 20).mean() > 0.3
    _check_sample(B, g, o, rn, rc, 20, "recent")
