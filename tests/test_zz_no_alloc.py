"""tg_cache_lookup_static -- the cache lookup for callers that cannot allocate device memory.

Some users of this library run where a device allocation is not an option: a serving process whose memory pool was
sized at start-up and is fully handed out, a plug-in that gets its tensors from a host framework and has no allocator
of its own, a thread that must never wait on cudaMalloc's device-wide lock.  They cannot give tg_cache_lookup its
workspace, so the library carries a small fixed scratch array for them (about 17 KB per GPU, at most 2^22 unique ids per
call).  This file checks that the entry point built on it returns exactly what tg_cache_lookup returns -- the work is
integer, so the comparison is bit for bit, as in tests/test_cache.py -- on two calls in a row that share the scratch
(the second one smaller, so that it runs over what the first left behind), that a request beyond the limit is refused
without a launch, and that the second call leaves the amount of free device memory untouched.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (first use of the scratch on the device happens here) and after the
rest of the suite."""
import ctypes as C

import numpy as np
import pytest


@pytest.fixture(scope="module")
def B():
    from paper_2607_05095_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def _case(seed, n_ids, n_occ, n_hot):
    rng = np.random.default_rng(seed)
    uniq = np.unique(rng.zipf(1.15, size=n_occ) % n_ids).astype(np.int64)
    slot = -np.ones(n_ids, np.int32)
    hot = rng.choice(n_ids, size=n_hot, replace=False)
    slot[hot] = rng.permutation(n_hot).astype(np.int32)
    return uniq, slot


@pytest.mark.gpu
def test_static_scratch_lookup_matches_workspace_lookup_twice(B):
    import torch
    # several scan tiles of 1024 ids and a ragged tail; the second call is shorter than the first
    cases = [_case(11, 900_000, 1_500_000, 120_000), _case(12, 200_000, 150_001, 30_000)]
    assert len(cases[0][0]) > len(cases[1][0]) > 4 * 1024 and len(cases[0][0]) % 1024 != 0
    U_max = max(len(u) for u, _ in cases)
    map_out = torch.empty(U_max, dtype=torch.int32, device="cuda")          # the caller's outputs, allocated once up front
    fresh_out = torch.empty(U_max, dtype=torch.int64, device="cuda")
    for call, (uniq, slot) in enumerate(cases):
        d_uniq, d_slot = torch.from_numpy(uniq).cuda(), torch.from_numpy(slot).cuda()
        ref_map, ref_fresh = B.cache_lookup(d_uniq, d_slot)                   # existing path: caller workspace
        torch.cuda.synchronize()
        map_out.fill_(-7)
        fresh_out.fill_(-7)
        torch.cuda.synchronize()
        free_before, held_before = torch.cuda.mem_get_info()[0], torch.cuda.memory_allocated()
        n_fresh = B.cache_lookup_static(d_uniq, d_slot, map_out, fresh_out)
        torch.cuda.synchronize()
        if call > 0:   # the first use on a device may load device code; after that a call must not cost a byte
            assert torch.cuda.mem_get_info()[0] >= free_before and torch.cuda.memory_allocated() == held_before
        U = len(uniq)
        assert n_fresh == ref_fresh.numel() and 0 < n_fresh < U
        assert torch.equal(map_out[:U], ref_map), f"call {call}: map differs from tg_cache_lookup"
        assert torch.equal(fresh_out[:n_fresh], ref_fresh), f"call {call}: fresh_ids differ from tg_cache_lookup"
        assert bool((map_out[U:] == -7).all()) and bool((fresh_out[n_fresh:] == -7).all()), "wrote past the valid outputs"


@pytest.mark.gpu
def test_static_scratch_lookup_limits(B):
    import torch
    L = B.lib()
    n = C.c_int64(-1)
    before = L.tg_launch_count()
    st = L.tg_cache_lookup_static(C.c_int64(B.CACHE_STATIC_MAX_IDS + 1), None, None, None, None, C.byref(n), None)
    assert st == 4 and n.value == 0 and L.tg_launch_count() == before         # TG_ERR_WORKSPACE, nothing launched
    assert b"TG_CACHE_STATIC_MAX_IDS" in L.tg_last_error()
    assert L.tg_cache_lookup_static(C.c_int64(0), None, None, None, None, C.byref(n), None) == 0 and n.value == 0
    # a call of exactly one id works (smallest non-empty input)
    uniq = torch.tensor([3], dtype=torch.int64, device="cuda")
    slot = torch.tensor([-1, -1, -1, 5], dtype=torch.int32, device="cuda")
    m = torch.empty(1, dtype=torch.int32, device="cuda")
    f = torch.empty(1, dtype=torch.int64, device="cuda")
    assert B.cache_lookup_static(uniq, slot, m, f) == 0 and int(m[0]) == -6
