"""NEXT-2 (SlimCache) parity: the library's Algorithm 1 (host C++, no GPU needed) and its device half against
oracle/cache_oracle.py, bit for bit (integer / byte work)."""
import numpy as np
import pytest

from oracle import cache_oracle as CO


@pytest.fixture(scope="module")
def B():
    from paper_2607_05095_b200 import build, binding
    build.build()
    binding.lib()
    return binding


@pytest.mark.parametrize("seed,alpha", [(0, 0.0), (1, 0.1), (2, 0.37), (3, 1.0), (4, 0.5)])
def test_greedy_select_matches_oracle(B, seed, alpha):
    rng = np.random.default_rng(seed)
    nV, nE = 300, 700
    batches = [(rng.zipf(1.4, 80) % nV, rng.zipf(1.2, 150) % nE) for _ in range(12)]
    rN, rE, _, _ = CO.greedy_select(alpha, batches, nV, nE)
    gN, gE = B.cache_greedy_select(alpha, batches, nV, nE)
    assert np.array_equal(gN, rN) and np.array_equal(gE, rE)


def test_greedy_select_edge_cases(B):
    assert all(len(x) == 0 for x in B.cache_greedy_select(0.5, [], 0, 0))
    gN, gE = B.cache_greedy_select(1.0, [([0, 0, 1], [2])], 2, 3)          # a batch counts an id once; everything selected
    rN, rE, _, _ = CO.greedy_select(1.0, [([0, 0, 1], [2])], 2, 3)
    assert np.array_equal(gN, rN) and np.array_equal(gE, rE) and len(gN) == 2 and len(gE) == 3
    with pytest.raises(B.FastTGError):
        B.cache_greedy_select(0.5, [([5], [0])], 2, 3)                       # id outside [0, n)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,F", [("float32", 100), ("bfloat16", 128), ("float32", 7), ("bfloat16", 50)])
def test_lookup_and_reconstruct(B, dtype, F):
    import torch
    rng = np.random.default_rng(F)
    n_ids, n_occ, n_hot = 50_000, 400_000, 9_000
    table = rng.standard_normal((n_ids, F)).astype(np.float32)
    ids = rng.zipf(1.2, size=n_occ) % n_ids
    uniq, inv = np.unique(ids, return_inverse=True)
    slot = -np.ones(n_ids, np.int32)
    hot = rng.choice(n_ids, size=n_hot, replace=False)
    slot[hot] = rng.permutation(n_hot).astype(np.int32)
    tdt = getattr(torch, dtype)
    t_table = torch.from_numpy(table).to(tdt)                                 # the storage-dtype table is the ground truth
    cache = torch.zeros(n_hot, F, dtype=tdt)
    cache[torch.from_numpy(slot[hot]).long()] = t_table[torch.from_numpy(hot).long()]
    rm, rfresh = CO.cache_lookup(uniq, slot)
    gm, gfresh = B.cache_lookup(torch.from_numpy(uniq).cuda(), torch.from_numpy(slot).cuda())
    assert np.array_equal(gm.cpu().numpy(), rm) and np.array_equal(gfresh.cpu().numpy(), rfresh)
    fresh_rows = t_table[torch.from_numpy(rfresh).long()].cuda()
    X = B.feature_reconstruct(torch.from_numpy(inv.astype(np.int32)).cuda(), gm, fresh_rows, cache.cuda())
    torch.cuda.synchronize()
    ref = t_table[torch.from_numpy(ids).long()]
    assert torch.equal(X.cpu(), ref)                                          # bit-exact: byte work
    ref_o = CO.reconstruct(inv[:500], rm, fresh_rows.cpu().float().numpy(), cache.float().numpy())
    assert np.array_equal(X[:500].cpu().float().numpy(), ref_o)
    X2 = B.feature_reconstruct(None, gm, fresh_rows, cache.cuda())            # one row per unique id
    assert torch.equal(X2.cpu(), t_table[torch.from_numpy(uniq).long()])
