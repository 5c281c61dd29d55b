"""CPU oracle of the temporal neighbour sampler.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

What it follows (reference = /root/reference/PAPER.md, FAST, arxiv/paper_2607_05095):
  * "top-k recent neighbor sampling [18] with k=10" ............ PAPER.md:311 (§6.1, Baselines and Settings)
  * the sampler walks TGL's T-CSR (per-node, time-sorted) ........ PAPER.md:412 (§7, Sampler-Based Acceleration)
  * each root node and its sampled neighbourhood are one task .... PAPER.md:233-247 (§4.4; the CPU thread binding of
    Algorithm 2 is the paper's own answer for its CPU and is out of scope)
  * uniform-in-time sampling of prior neighbours ................. BASELINE.json configs[2] ("up to 20 uniform-in-time
    sampled prior neighbors")
Readings: R20 "prior" = events with stream index strictly below the root's cutoff, incident to the
root node in either direction, a self-loop counted once; R27 ties in time are broken by the event index (the stream is
time-sorted, so "most recent" = largest event index); R28 the uniform draw is Floyd's sampling without replacement
driven by a counter-based generator (SplitMix64 outputs indexed by (seed, root, draw)), positions emitted ascending.

Plain NumPy / pure-Python loops over roots, no blocking, no vectorised tricks: written to be checked by eye.
Pins (tests/test_oracle_sampler.py): brute force over the raw event list on tiny streams; the bench generator's own
dictionary-based sampler (workloads._sample_block) on config 1; SplitMix64's published test
vector; Floyd's algorithm against exhaustive subset frequencies; validity properties of every draw.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

MASK64 = (1 << 64) - 1
GOLDEN = 0x9E3779B97F4A7C15
MAX_K = 64          # draws of one root are the outputs  64*root + 1 .. 64*root + k  of the stream


def splitmix64_output(seed: int, n: int) -> int:
    """The n-th output (n >= 1) of SplitMix64 seeded with `seed` (Steele, Lea, Flood 2014; Vigna's reference code):
    state_n = seed + n * GOLDEN (mod 2^64), output = the 64-bit finaliser of state_n.  Counter-based: no carried state."""
    z = (seed + n * GOLDEN) & MASK64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
    return z ^ (z >> 31)


def rand_below(seed: int, root: int, draw: int, n: int) -> int:
    """Integer in [0, n): the high 64 bits of (64-bit output) * n  (multiply-shift range reduction, no rejection)."""
    return (splitmix64_output(seed, MAX_K * root + draw + 1) * n) >> 64


@dataclass
class TCSR:
    """Per-node incidence lists in event (= time) order: entries indptr[x]..indptr[x+1] of `nbr` (other endpoint),
    `eid` (event index, ascending inside a node) and `ts` (event time)."""
    indptr: np.ndarray   # int64 [N+1]
    nbr: np.ndarray      # int64 [M2]
    eid: np.ndarray      # int64 [M2]
    ts: np.ndarray       # float32 [M2]


def tcsr_build(n_nodes: int, u: np.ndarray, v: np.ndarray, t: np.ndarray) -> TCSR:
    """Event i = (u[i], v[i]) at time t[i] is listed under u[i] with neighbour v[i] and, unless u[i] == v[i], under v[i]
    with neighbour u[i] (reading R20).  Inside a node the entries are in ascending event index.  The grouping is a
    library sort (np.lexsort by (node, event index)); tests pin it against plain per-node Python lists."""
    u, v = np.asarray(u, np.int64), np.asarray(v, np.int64)
    ev = np.arange(len(u), dtype=np.int64)
    two = u != v
    node = np.concatenate([u, v[two]])
    other = np.concatenate([v, u[two]])
    idx = np.concatenate([ev, ev[two]])
    order = np.lexsort((idx, node))
    node, other, idx = node[order], other[order], idx[order]
    indptr = np.zeros(n_nodes + 1, np.int64)
    np.cumsum(np.bincount(node, minlength=n_nodes), out=indptr[1:])
    return TCSR(indptr, other, idx, np.asarray(t, np.float32)[idx])


def _prior_range(g: TCSR, node: int, cutoff: int):
    """[s, p): the node's entries with event index strictly below the cutoff (eid ascends inside a node: a library
    binary search; tests pin it against a linear scan)."""
    s, e = int(g.indptr[node]), int(g.indptr[node + 1])
    return s, s + int(np.searchsorted(g.eid[s:e], cutoff, side="left"))


def _emit(g: TCSR, picks):
    roots = np.array([i for i, _ in picks], np.int32)
    pos = np.array([p for _, p in picks], np.int64)
    return roots, g.nbr[pos].astype(np.int64), g.eid[pos].astype(np.int64), g.ts[pos].astype(np.float32)


def sample_recent(g: TCSR, root_node, root_cutoff, k: int):
    """Per root i: the (up to) k most recent prior incident events of root_node[i], oldest first.
    Returns tg_block_build's inputs: root_idx int32 [E] (the root's index i), nbr_node int64, edge_id int64, ts float32."""
    picks = []
    for i in range(len(root_node)):
        s, p = _prior_range(g, int(root_node[i]), int(root_cutoff[i]))
        for q in range(max(s, p - k), p):
            picks.append((i, q))
    return _emit(g, picks)


def floyd_sample(seed: int, root: int, n: int, k: int):
    """k distinct integers of [0, n) (all of them if n <= k), ascending.  Robert Floyd's algorithm (Bentley & Floyd,
    CACM 30(9), 1987): for j = n-k .. n-1 draw t uniform in [0, j]; take t unless already taken, else take j."""
    if n <= k:
        return list(range(n))
    chosen = []
    for d, j in enumerate(range(n - k, n)):
        t = rand_below(seed, root, d, j + 1)
        chosen.append(j if t in chosen else t)
    return sorted(chosen)


def sample_uniform(g: TCSR, root_node, root_cutoff, k: int, seed: int):
    """Per root i: up to k of its prior incident events, uniformly without replacement (reading R28), oldest first."""
    assert k <= MAX_K
    picks = []
    for i in range(len(root_node)):
        s, p = _prior_range(g, int(root_node[i]), int(root_cutoff[i]))
        for off in floyd_sample(seed, i, p - s, k):
            picks.append((i, s + off))
    return _emit(g, picks)
