"""Seeded synthetic workload generators for the five BASELINE.json configs.

This module holds NO arithmetic of the method (no sorting into CSR, no softmax, no dot
products): it only draws the sampler's output lists (root, neighbour, edge, timestamp) and
the random feature tensors, exactly as DESIGN.md §4 ("input recipe") states.  Both the CPU
oracle (tests, ``bench.py --impl reference``) and the CUDA path consume the arrays produced
here; neither of them imports the other.

The paper's datasets (Table 3) are not available; these inputs stand in for
them and take their shapes: top-k most-recent sampling with k = 10, small-degree /
long-tailed root degrees (Fig. 3), heavy within-batch node repetition
(Table 1).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

STREAM_ENDPOINTS, STREAM_NEG, STREAM_SAMPLING, STREAM_Q, STREAM_K, STREAM_V, STREAM_DO, \
    STREAM_DEG, STREAM_SRC, STREAM_TS, STREAM_PERM = range(11)


def _rng(seed: int, config_id: int, stream_id: int, sub: int = 0) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([seed, config_id, stream_id, sub]))


def bounded_zipf_cdf(a: float, n: int) -> np.ndarray:
    """float64 CDF of P(k) ∝ k^-a on {1..n}."""
    w = np.arange(1, n + 1, dtype=np.float64) ** (-a)
    cdf = np.cumsum(w)
    cdf /= cdf[-1]
    return cdf


def bounded_zipf(rng: np.random.Generator, cdf: np.ndarray, size: int) -> np.ndarray:
    """Inverse-CDF draw; returns ranks in 0..n-1 (rank 0 is the most likely)."""
    u = rng.random(size)
    k = np.searchsorted(cdf, u, side="left")
    np.minimum(k, len(cdf) - 1, out=k)
    return k


def sorted_uniform_times(rng: np.random.Generator, m: int, t_max: float) -> np.ndarray:
    """m sorted U[0,t_max) draws (order statistics via normalised exponential gaps; no sort)."""
    gaps = rng.standard_exponential(m + 1)
    t = np.cumsum(gaps)
    t = t[:m] / t[m] * t_max
    return t


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round float32 values to the nearest bf16 (RNE) and return them as float32."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + r) & np.uint32(0xFFFF0000)).view(np.float32)


def bf16_bits(x_rounded: np.ndarray) -> np.ndarray:
    """uint16 bit patterns of float32 values that are already bf16-representable."""
    return (np.ascontiguousarray(x_rounded, dtype=np.float32).view(np.uint32) >> np.uint32(16)).astype(np.uint16)


@dataclass
class Workload:
    """One mini-batch block as the sampler would hand it over (COO lists, sampler order)."""
    name: str
    config_id: int
    seed: int
    R: int
    H: int
    D: int
    dtype: str            # "f32" | "bf16" (storage type of row tensors)
    scale: float
    dedup_mode: int       # 0: K,V are per-edge rows [E,H,D]; 1: unique-row remap
    root_idx: np.ndarray  # int32 [E]
    nbr_node: np.ndarray  # int64 [E]
    edge_id: np.ndarray   # int64 [E]
    ts: np.ndarray        # float32 [E]
    hop: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def E(self) -> int:
        return int(self.root_idx.shape[0])

    @property
    def F(self) -> int:
        return self.H * self.D

    def num_unique_rows(self) -> int:
        """Number of K/V rows the block will index (sizing only)."""
        if self.dedup_mode == 0:
            return self.E
        return int(np.unique(self.nbr_node).shape[0])

    def features(self, U: int | None = None):
        """Q[R,H,D], K[U,H,D], V[U,H,D], dO[R,H,D] as float32 (bf16-rounded if dtype == 'bf16')."""
        if U is None:
            U = self.num_unique_rows()
        sub = self.hop
        sd = 1.0 / np.sqrt(self.D)
        q = _rng(self.seed, self.config_id, STREAM_Q, sub).standard_normal((self.R, self.H, self.D), dtype=np.float32) * np.float32(sd)
        k = _rng(self.seed, self.config_id, STREAM_K, sub).standard_normal((U, self.H, self.D), dtype=np.float32) * np.float32(sd)
        v = _rng(self.seed, self.config_id, STREAM_V, sub).standard_normal((U, self.H, self.D), dtype=np.float32) * np.float32(sd)
        do = _rng(self.seed, self.config_id, STREAM_DO, sub).standard_normal((self.R, self.H, self.D), dtype=np.float32)
        if self.dtype == "bf16":
            q, k, v, do = (round_to_bf16(a) for a in (q, k, v, do))
        return q, k, v, do


# ----------------------------------------------------------------------------------------------
# Event-stream configs (1-3)
# ----------------------------------------------------------------------------------------------

def _event_stream(seed, cid, n_nodes, n_events, zipf_a=1.1, t_max=1e6):
    cdf = bounded_zipf_cdf(zipf_a, n_nodes)
    rank_to_id = _rng(seed, cid, STREAM_PERM).permutation(n_nodes).astype(np.int32)
    r = _rng(seed, cid, STREAM_ENDPOINTS)
    u = rank_to_id[bounded_zipf(r, cdf, n_events)]
    v = rank_to_id[bounded_zipf(r, cdf, n_events)]
    t = sorted_uniform_times(_rng(seed, cid, STREAM_TS), n_events, t_max)
    return u, v, t


def _incidence_lists(u, v, root_nodes):
    """For the given root node ids: (node-sorted) lists of incident event indices and the other endpoint."""
    n = int(max(u.max(), v.max(), root_nodes.max())) + 1
    is_root = np.zeros(n, dtype=bool)
    is_root[root_nodes] = True
    a = np.flatnonzero(is_root[u])                 # events where u is a root node: neighbour is v
    b = np.flatnonzero(is_root[v] & (u != v))      # events where v is a root node: neighbour is u
    node = np.concatenate([u[a], v[b]]).astype(np.int64)
    other = np.concatenate([v[a], u[b]]).astype(np.int64)
    idx = np.concatenate([a, b]).astype(np.int64)
    order = np.lexsort((idx, node))
    node, other, idx = node[order], other[order], idx[order]
    uniq, start = np.unique(node, return_index=True)
    end = np.append(start[1:], len(node))
    lut = {int(x): (int(s), int(e)) for x, s, e in zip(uniq, start, end)}
    return lut, other, idx


def _sample_block(u, v, t, root_node, root_cutoff, k, mode, rng):
    """Temporal neighbour sampling: per root, up to k prior incident events (index < cutoff).
    mode 'recent': the k most recent; 'uniform': k uniformly without replacement."""
    lut, other, idx = _incidence_lists(u, v, np.unique(root_node))
    roots, nbrs, eids = [], [], []
    for i, (x, c) in enumerate(zip(root_node.tolist(), root_cutoff.tolist())):
        se = lut.get(x)
        if se is None:
            continue
        s, e = se
        p = s + int(np.searchsorted(idx[s:e], c, side="left"))   # entries [s,p) are prior events
        cnt = p - s
        if cnt == 0:
            continue
        if mode == "recent":
            sel = np.arange(max(s, p - k), p)
        else:
            sel = s + np.sort(rng.choice(cnt, size=min(k, cnt), replace=False))
        roots.append(np.full(len(sel), i, dtype=np.int32))
        nbrs.append(other[sel])
        eids.append(idx[sel])
    if roots:
        root_idx = np.concatenate(roots)
        nbr = np.concatenate(nbrs)
        eid = np.concatenate(eids)
    else:
        root_idx = np.zeros(0, np.int32); nbr = np.zeros(0, np.int64); eid = np.zeros(0, np.int64)
    ts = t[eid].astype(np.float32)
    return root_idx, nbr, eid, ts


def _batch_roots(u, v, n_nodes, batch, seed, cid):
    m = len(u)
    ev = np.arange(m - batch, m)
    neg = _rng(seed, cid, STREAM_NEG).integers(0, n_nodes, size=batch)
    root_node = np.concatenate([u[ev], v[ev], neg]).astype(np.int64)
    root_cutoff = np.concatenate([ev, ev, ev]).astype(np.int64)
    return root_node, root_cutoff


def config1(seed: int = 0, n_nodes=20_000, n_events=200_000, batch=600, k=10, dedup_mode=0) -> Workload:
    """Tiny single-layer TGAT block, fp32 (BASELINE.json configs[0])."""
    cid = 1
    u, v, t = _event_stream(seed, cid, n_nodes, n_events)
    rn, rc = _batch_roots(u, v, n_nodes, batch, seed, cid)
    root_idx, nbr, eid, ts = _sample_block(u, v, t, rn, rc, k, "recent", None)
    return Workload("config1_tgat_tiny_f32", cid, seed, len(rn), 2, 50, "f32", 1.0, dedup_mode, root_idx, nbr, eid, ts)


def config2(seed: int = 0, n_nodes=100_000, n_events=5_000_000, batch=600, k=10):
    """Two-hop TGAT block, fp32 (configs[1]); returns (hop-1 block, hop-2 block)."""
    cid = 2
    u, v, t = _event_stream(seed, cid, n_nodes, n_events)
    rn, rc = _batch_roots(u, v, n_nodes, batch, seed, cid)
    r1, n1, e1, t1 = _sample_block(u, v, t, rn, rc, k, "recent", None)
    w1 = Workload("config2_hop1_f32", cid, seed, len(rn), 2, 50, "f32", 1.0, 1, r1, n1, e1, t1, hop=0)
    # hop 2: one root per hop-1 edge (node = that neighbour, cutoff = that edge's event index)
    r2, n2, e2, t2 = _sample_block(u, v, t, n1.copy(), e1.copy(), k, "recent", None)
    w2 = Workload("config2_hop2_f32", cid, seed, len(n1), 2, 50, "f32", 1.0, 1, r2, n2, e2, t2, hop=1)
    return w1, w2


def config3(seed: int = 0, n_nodes=1_000_000, n_events=50_000_000, batch=4000, k=20) -> Workload:
    """Large-batch one-hop block, bf16 storage (configs[2])."""
    cid = 3
    u, v, t = _event_stream(seed, cid, n_nodes, n_events)
    rn, rc = _batch_roots(u, v, n_nodes, batch, seed, cid)
    root_idx, nbr, eid, ts = _sample_block(u, v, t, rn, rc, k, "uniform", _rng(seed, cid, STREAM_SAMPLING))
    return Workload("config3_large_batch_bf16", cid, seed, len(rn), 4, 32, "bf16", 1.0, 1, root_idx, nbr, eid, ts)


# ----------------------------------------------------------------------------------------------
# Degree-distribution configs (4-5)
# ----------------------------------------------------------------------------------------------

def _degree_block(seed, cid, R, deg_a, deg_max, n_src_nodes, src_a=1.2):
    deg = bounded_zipf(_rng(seed, cid, STREAM_DEG), bounded_zipf_cdf(deg_a, deg_max), R).astype(np.int64) + 1
    E = int(deg.sum())
    root_idx = np.repeat(np.arange(R, dtype=np.int32), deg)
    rank_to_id = _rng(seed, cid, STREAM_PERM).permutation(n_src_nodes).astype(np.int64)
    nbr = rank_to_id[bounded_zipf(_rng(seed, cid, STREAM_SRC), bounded_zipf_cdf(src_a, n_src_nodes), E)]
    eid = np.arange(E, dtype=np.int64)
    ts = (_rng(seed, cid, STREAM_TS).random(E, dtype=np.float32) * np.float32(1e6)).astype(np.float32)
    return root_idx, nbr, eid, ts


def config4(seed: int = 0, R=200_000, deg_max=4096, n_src_nodes=5_000_000, dedup_mode=1) -> Workload:
    """Skewed large block, bf16 storage; the roofline target (configs[3])."""
    cid = 4
    root_idx, nbr, eid, ts = _degree_block(seed, cid, R, 1.5, deg_max, n_src_nodes)
    return Workload("config4_skewed_bf16", cid, seed, R, 8, 16, "bf16", 1.0, dedup_mode, root_idx, nbr, eid, ts)


def config5(seed: int = 0, R=50_000, deg_max=200_000, n_src_nodes=5_000_000) -> Workload:
    """Full-neighbourhood hub stress, fp32, logits with standard deviation 8 (configs[4])."""
    cid = 5
    root_idx, nbr, eid, ts = _degree_block(seed, cid, R, 1.3, deg_max, n_src_nodes)
    return Workload("config5_hub_stress_f32", cid, seed, R, 2, 64, "f32", 64.0, 1, root_idx, nbr, eid, ts)


def small_random(seed: int, R: int, max_deg: int, n_src: int, H: int, D: int, dtype="f32", scale=1.0,
                 dedup_mode=1, shuffle=False, zero_frac=0.1) -> Workload:
    """Small random block for unit tests: degrees U{0..max_deg} (a fraction forced to zero), sources U{0..n_src-1}."""
    r = _rng(seed, 99, 0)
    deg = r.integers(0, max_deg + 1, size=R)
    deg[r.random(R) < zero_frac] = 0
    E = int(deg.sum())
    root_idx = np.repeat(np.arange(R, dtype=np.int32), deg)
    nbr = r.integers(0, max(n_src, 1), size=E).astype(np.int64) * 7 + 3
    eid = r.permutation(E).astype(np.int64) + 1000
    ts = r.random(E, dtype=np.float32)
    if shuffle and E > 0:
        p = r.permutation(E)
        root_idx, nbr, eid, ts = root_idx[p], nbr[p], eid[p], ts[p]
    return Workload(f"small_R{R}_d{max_deg}", 99, seed, R, H, D, dtype, scale, dedup_mode, root_idx, nbr, eid, ts)
