"""Pins of oracle/sampler_oracle.py, `-m "not gpu"`.

  * tcsr_build ........ plain per-node Python lists built by walking the events in order
  * _prior_range ...... linear scan
  * sample_recent ..... brute force over the RAW event list (no T-CSR at all) on tiny streams; the bench generator's own
                        dictionary-based sampler (workloads._sample_block) on config 1 (k = 10 most recent)
  * splitmix64_output . the published SplitMix64 test vector (seed 1234567; Vigna's splitmix64.c, reproduced in the test
                        suites of the xoshiro generators)
  * floyd_sample ...... exhaustive subset frequencies on tiny (n, k); always k distinct sorted values below n
  * sample_uniform .... every pick is a prior incident event of its root, distinct, ascending, min(k, count) of them;
                        k >= count reduces to "all prior events" = sample_recent with k = count
"""
import itertools

import numpy as np
import pytest

from oracle import sampler_oracle as S
import workloads as W


def _tiny_stream(seed, n_nodes=7, m=60):
    r = np.random.default_rng(seed)
    u = r.integers(0, n_nodes, m)
    v = r.integers(0, n_nodes, m)
    t = np.sort(r.random(m)).astype(np.float32)
    return u, v, t


def test_tcsr_against_python_lists():
    for seed in range(5):
        u, v, t = _tiny_stream(seed)
        g = S.tcsr_build(7, u, v, t)
        lists = [[] for _ in range(7)]
        for i in range(len(u)):
            lists[int(u[i])].append((i, int(v[i])))
            if u[i] != v[i]:
                lists[int(v[i])].append((i, int(u[i])))
        for x in range(7):
            s, e = int(g.indptr[x]), int(g.indptr[x + 1])
            assert [(int(a), int(b)) for a, b in zip(g.eid[s:e], g.nbr[s:e])] == lists[x]
            assert np.array_equal(g.ts[s:e], t[g.eid[s:e]])
        assert g.indptr[-1] == len(u) + int((u != v).sum())      # a self-loop is listed once


def test_prior_range_against_linear_scan():
    u, v, t = _tiny_stream(3)
    g = S.tcsr_build(7, u, v, t)
    for x in range(7):
        for c in range(0, 62):
            s, p = S._prior_range(g, x, c)
            q = s
            while q < g.indptr[x + 1] and g.eid[q] < c:
                q += 1
            assert (s, p) == (int(g.indptr[x]), q)


def _brute_recent(u, v, t, root_node, cutoff, k):
    """No T-CSR: for every root walk the whole event list backwards from cutoff-1 (definition of PAPER.md:311 + R20)."""
    out = []
    for i, (x, c) in enumerate(zip(root_node, cutoff)):
        found = []
        for e in range(int(c) - 1, -1, -1):
            if u[e] == x or v[e] == x:
                found.append((i, int(v[e]) if u[e] == x else int(u[e]), e, np.float32(t[e])))
                if len(found) == k:
                    break
        out.extend(reversed(found))        # oldest first
    return out


@pytest.mark.parametrize("k", [1, 3, 10])
def test_recent_brute_force(k):
    for seed in range(4):
        u, v, t = _tiny_stream(seed)
        g = S.tcsr_build(7, u, v, t)
        r = np.random.default_rng(100 + seed)
        root_node = r.integers(0, 7, 25)
        cutoff = r.integers(0, 61, 25)
        ri, nb, ei, ts = S.sample_recent(g, root_node, cutoff, k)
        ref = _brute_recent(u, v, t, root_node, cutoff, k)
        assert [(int(a), int(b), int(c), np.float32(d)) for a, b, c, d in zip(ri, nb, ei, ts)] == ref


def test_recent_matches_bench_generator_config1():
    """workloads.config1 draws its block with its own sampler (dictionary of incidence ranges); same lists expected."""
    seed, cid = 0, 1
    u, v, t = W._event_stream(seed, cid, 20_000, 200_000)
    rn, rc = W._batch_roots(u, v, 20_000, 600, seed, cid)
    g = S.tcsr_build(20_000, u, v, t)
    ri, nb, ei, ts = S.sample_recent(g, rn, rc, 10)
    w = W.config1(seed)
    assert np.array_equal(ri, w.root_idx) and np.array_equal(nb, w.nbr_node) and np.array_equal(ei, w.edge_id)
    assert np.array_equal(ts, w.ts)


def test_splitmix64_published_vector():
    # SplitMix64, seed 1234567: first five outputs as printed with the reference implementation
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "splitmix64_seed1234567.txt")
    expect = [int(ln) for ln in open(path).read().splitlines() if ln and not ln.startswith("#")]
    assert len(expect) == 5
    assert [S.splitmix64_output(1234567, n) for n in range(1, 6)] == expect


def test_rand_below_is_uniform():
    n = 7
    cnt = np.zeros(n)
    for root in range(2000):
        for d in range(5):
            x = S.rand_below(42, root, d, n)
            assert 0 <= x < n
            cnt[x] += 1
    exp = cnt.sum() / n
    assert ((cnt - exp) ** 2 / exp).sum() < 30.0        # chi-square, 6 dof: P(> 30) ~ 4e-5


@pytest.mark.parametrize("n,k", [(5, 2), (6, 3), (4, 1)])
def test_floyd_subsets_equally_likely(n, k):
    subsets = {c: 0 for c in itertools.combinations(range(n), k)}
    trials = 6000
    for root in range(trials):
        pick = tuple(S.floyd_sample(7, root, n, k))
        assert pick in subsets                           # k distinct ascending values below n
        subsets[pick] += 1
    exp = trials / len(subsets)
    chi = sum((c - exp) ** 2 / exp for c in subsets.values())
    assert chi < 3.0 * len(subsets) + 20                 # far beyond any plausible fluctuation of a fair draw, far below a biased one
    assert S.floyd_sample(7, 0, 3, 5) == [0, 1, 2]       # fewer candidates than k: all of them


def test_uniform_validity_and_reduction():
    for seed in range(3):
        u, v, t = _tiny_stream(seed, m=80)
        g = S.tcsr_build(7, u, v, t)
        r = np.random.default_rng(seed)
        root_node = r.integers(0, 7, 30)
        cutoff = r.integers(0, 81, 30)
        for k in (2, 5, 64):
            ri, nb, ei, ts = S.sample_uniform(g, root_node, cutoff, k, seed=9)
            for i in range(30):
                x, c = int(root_node[i]), int(cutoff[i])
                mine = ei[ri == i]
                prior = [e for e in range(c) if u[e] == x or v[e] == x]
                assert len(mine) == min(k, len(prior))
                assert np.all(np.diff(mine) > 0) and set(mine.tolist()) <= set(prior)
            assert np.all(np.diff(ri) >= 0)
            j = np.flatnonzero(ei >= 0)
            assert np.array_equal(nb[j], np.where(u[ei] == root_node[ri], v[ei], u[ei]))
        # k >= every count: identical to "all prior events"
        allr = S.sample_recent(g, root_node, cutoff, 64)
        allu = S.sample_uniform(g, root_node, cutoff, 64, seed=1)
        for a, b in zip(allr, allu):
            assert np.array_equal(a, b)
