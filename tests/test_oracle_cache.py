"""Pins of the NEXT-2 oracle (oracle/cache_oracle.py: Algorithm 1 + ID-compression / cache reconstruction).

* reconstruct o lookup o unique == plain fancy indexing of the full feature table by the original ids (the definition
  SlimCache must preserve: the reconstructed rows ARE the rows of the ids), bit for bit;
* the paper's only worked numbers (Figure 5): 12 occurrences -> 7 unique rows transferred without a cache;
* Algorithm 1: the selected sets respect the budget, are prefixes of the frequency orders, and maximise the total access
  frequency among ALL subsets of that size (brute force on small universes); a hand example with a tie;
* degenerate budgets (0, everything) and an exhausted node list.
"""
import itertools

import numpy as np
import pytest

from oracle import cache_oracle as CO


def test_reconstruct_is_plain_indexing():
    rng = np.random.default_rng(0)
    n_ids, F = 500, 6
    table = rng.standard_normal((n_ids, F)).astype(np.float32)
    ids = rng.zipf(1.3, size=3000) % n_ids
    uniq, inv = np.unique(ids, return_inverse=True)
    slot = -np.ones(n_ids, np.int32)
    hot = rng.choice(n_ids, size=120, replace=False)
    slot[hot] = rng.permutation(120)
    cache = np.zeros((120, F), np.float32)
    cache[slot[hot]] = table[hot]
    m, fresh = CO.cache_lookup(uniq, slot)
    assert len(fresh) == int((slot[uniq] < 0).sum()) and np.all(slot[fresh] < 0)
    assert np.array_equal(fresh, uniq[slot[uniq] < 0])                       # order of the unique ids is kept
    X = CO.reconstruct(inv, m, table[fresh], cache)
    assert np.array_equal(X, table[ids])


def test_paper_example_12_to_7():
    ids = np.array([3, 5, 3, 9, 1, 5, 3, 7, 9, 2, 1, 8])                     # 12 occurrences, 7 distinct ids (counts are the paper's)
    uniq, inv = np.unique(ids, return_inverse=True)
    m, fresh = CO.cache_lookup(uniq, -np.ones(10, np.int32))
    assert len(ids) == 12 and len(fresh) == 7 and np.array_equal(m, np.arange(7))


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_greedy_is_optimal_and_respects_budget(seed):
    rng = np.random.default_rng(seed)
    nV, nE = 6, 7
    batches = [(rng.integers(0, nV, 5), rng.integers(0, nE, 6)) for _ in range(8)]
    for alpha in (0.0, 0.2, 0.5, 0.77, 1.0):
        H_N, H_E, f_v, f_e = CO.greedy_select(alpha, batches, nV, nE)
        n = len(H_N) + len(H_E)
        assert n == int(np.ceil(alpha * (nV + nE) - 1e-12)) and len(set(H_N)) == len(H_N) and len(set(H_E)) == len(H_E)
        # prefixes of the (descending) frequency orders
        assert np.array_equal(f_v[H_N], np.sort(f_v)[::-1][:len(H_N)]) and np.array_equal(f_e[H_E], np.sort(f_e)[::-1][:len(H_E)])
        # brute force: no subset of the same size has a larger total frequency
        allf = np.concatenate([f_v, f_e])
        best = max(sum(c) for c in itertools.combinations(allf.tolist(), n)) if n else 0
        assert int(f_v[H_N].sum() + f_e[H_E].sum()) == best


def test_greedy_hand_example_tie_and_exhaustion():
    # nodes: f = [3, 1]; edges: f = [3, 2, 0]  (batches are id sets: one count per batch)
    batches = [([0, 1], [0, 1]), ([0], [0, 1]), ([0], [0])]
    H_N, H_E, f_v, f_e = CO.greedy_select(0.6, batches, 2, 3)                # budget 0.6 * 5 = 3 picks
    assert f_v.tolist() == [3, 1] and f_e.tolist() == [3, 2, 0]
    # pick 1: f_v = 3 is not > f_e = 3 -> edge 0; pick 2: 3 > 2 -> node 0; pick 3: 1 > 2 false -> edge 1
    assert H_E.tolist() == [0, 1] and H_N.tolist() == [0]
    H_N, H_E, _, _ = CO.greedy_select(1.0, batches, 2, 3)                    # everything, lists exhausted without error
    assert sorted(H_N.tolist()) == [0, 1] and sorted(H_E.tolist()) == [0, 1, 2]
