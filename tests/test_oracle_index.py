"""Pins for the oracle's index structures (ora_block_build).

The paper's compression triple (uni_ID, inv_Idx, ind_ptr) prints no values, only the
counts "12 -> 7" of Fig. 5(a); so the oracle is pinned by library routines it does not itself call
(np.unique, np.argsort, scipy.sparse), by brute force and by invariants (SURVEY.md §8(c) pins table).
"""
import os

import numpy as np
import pytest
import scipy.sparse as sp

import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _cases():
    yield W.small_random(1, 40, 6, 12, 2, 4, shuffle=True)
    yield W.small_random(2, 300, 20, 50, 2, 4, shuffle=True)
    yield W.small_random(3, 300, 20, 50, 2, 4, shuffle=False)
    yield W.small_random(4, 5, 200, 3, 2, 4, shuffle=True)          # few destinations, heavy multi-edges
    yield W.small_random(5, 100, 3, 1, 2, 4, shuffle=True)           # a single source row (U = 1)
    yield W.config1(seed=0)


@pytest.mark.parametrize("w", list(_cases()), ids=lambda w: w.name)
@pytest.mark.parametrize("dedup", [0, 1])
def test_block_vs_library_routines(oracle_mod, w, dedup):
    b = oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, dedup)
    E = w.E
    # group-by: stable argsort + bincount prefix sum (numpy)
    perm = np.argsort(w.root_idx, kind="stable").astype(np.int32)
    indptr = np.concatenate([[0], np.cumsum(np.bincount(w.root_idx, minlength=w.R))]).astype(np.int32)
    assert np.array_equal(b.perm, perm)
    assert np.array_equal(b.indptr, indptr)
    assert np.array_equal(b.eid_csr, w.edge_id[perm]) and np.array_equal(b.ts_csr, w.ts[perm])
    # scipy: COO -> CSR keeps input order inside a row when data = arange (sum_duplicates not called)
    if E:
        csr = sp.coo_matrix((np.arange(E), (w.root_idx, np.arange(E))), shape=(w.R, E)).tocsr()
        assert np.array_equal(csr.indptr, b.indptr)
    nbr_csr = w.nbr_node[perm]
    if dedup:
        uniq, inv = np.unique(nbr_csr, return_inverse=True)
        assert b.U == len(uniq)
        assert np.array_equal(b.uniq_node, uniq)
        assert np.array_equal(b.kv_row, inv.astype(np.int32))
    else:
        assert b.U == E
        assert np.array_equal(b.kv_row, np.arange(E, dtype=np.int32))
        assert np.array_equal(b.uniq_node, nbr_csr)
    # transposed CSR == structure of csr.T with data = CSR position
    t_edge = np.argsort(b.kv_row, kind="stable").astype(np.int32)
    t_indptr = np.concatenate([[0], np.cumsum(np.bincount(b.kv_row, minlength=b.U))]).astype(np.int32)
    dst_of = np.repeat(np.arange(w.R, dtype=np.int32), np.diff(indptr))
    assert np.array_equal(b.t_edge, t_edge)
    assert np.array_equal(b.t_indptr, t_indptr)
    assert np.array_equal(b.t_dst, dst_of[t_edge])
    if E:
        a = sp.csr_matrix((np.arange(E) + 1, b.kv_row, b.indptr), shape=(w.R, b.U))
        # multi-edges: keep them distinct by going through COO with explicit ordering
        coo_r, coo_c = dst_of, b.kv_row
        order = np.lexsort((np.arange(E), coo_c))
        assert np.array_equal(b.t_edge, order.astype(np.int32))
        assert a.shape == (w.R, b.U)


@pytest.mark.parametrize("w", list(_cases()), ids=lambda w: w.name)
def test_block_invariants(oracle_mod, w):
    b = oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, 1)
    E = w.E
    assert b.indptr[0] == 0 and b.indptr[-1] == E and np.all(np.diff(b.indptr) >= 0)
    assert np.array_equal(np.sort(b.perm), np.arange(E))
    assert np.all(np.diff(w.root_idx[b.perm]) >= 0)
    for v in range(w.R):                                  # stable: input order kept inside a destination
        seg = b.perm[b.indptr[v]:b.indptr[v + 1]]
        assert np.all(np.diff(seg) > 0)
    assert np.all(np.diff(b.uniq_node) > 0)               # strictly ascending
    assert np.array_equal(b.uniq_node[b.kv_row], w.nbr_node[b.perm])
    assert np.array_equal(np.sort(b.t_edge), np.arange(E))
    dst_of = np.repeat(np.arange(w.R), np.diff(b.indptr))
    for u in range(b.U):
        seg = b.t_edge[b.t_indptr[u]:b.t_indptr[u + 1]]
        assert len(seg) >= 1                              # an unused unique row cannot exist
        assert np.all(b.kv_row[seg] == u) and np.all(np.diff(seg) > 0)
        assert np.array_equal(b.t_dst[b.t_indptr[u]:b.t_indptr[u + 1]], dst_of[seg])


def test_block_brute_force(oracle_mod):
    """O(E^2) brute force on a tiny shuffled input."""
    w = W.small_random(11, 9, 5, 6, 1, 2, shuffle=True)
    b = oracle_mod.block_build(w.R, w.root_idx, w.nbr_node, w.edge_id, w.ts, 1)
    E = w.E
    pos = 0
    for v in range(w.R):
        assert b.indptr[v] == pos
        for e in range(E):
            if w.root_idx[e] == v:
                assert b.perm[pos] == e
                pos += 1
    assert b.indptr[w.R] == pos == E
    uniq = sorted(set(w.nbr_node.tolist()))
    assert b.uniq_node.tolist() == uniq
    for e in range(E):
        assert uniq[b.kv_row[e]] == w.nbr_node[b.perm[e]]
    j = 0
    for u in range(len(uniq)):
        assert b.t_indptr[u] == j
        for e in range(E):
            if b.kv_row[e] == u:
                assert b.t_edge[j] == e
                assert b.indptr[b.t_dst[j]] <= e < b.indptr[b.t_dst[j] + 1]
                j += 1
    assert b.t_indptr[len(uniq)] == E


def test_block_paper_counts_12_to_7(oracle_mod):
    """PAPER.md:162 (Fig. 5a): 12 feature rows shrink to 7 unique rows + an inverse index.
    The figure's ids are an image; only the counts are in the text (tests/golden/compression_12_to_7.txt)."""
    rows = [ln.split() for ln in open(os.path.join(GOLDEN, "compression_12_to_7.txt")) if ln.strip() and not ln.startswith("#")]
    ids = np.array([int(x) for x in rows[0]], dtype=np.int64)
    n_in, n_unique = int(rows[1][0]), int(rows[1][1])
    assert len(ids) == n_in == 12
    root = np.repeat(np.arange(4, dtype=np.int32), 3)
    b = oracle_mod.block_build(4, root, ids, None, None, 1)
    assert b.U == n_unique == 7
    assert np.array_equal(b.uniq_node[b.kv_row], ids)       # reconstruction through the inverse index


def test_block_empty_and_errors(oracle_mod):
    b = oracle_mod.block_build(3, np.zeros(0, np.int32), np.zeros(0, np.int64), None, None, 1)
    assert b.U == 0 and b.indptr.tolist() == [0, 0, 0, 0] and b.t_indptr.tolist() == [0]
    b = oracle_mod.block_build(0, np.zeros(0, np.int32), np.zeros(0, np.int64), None, None, 0)
    assert b.U == 0 and b.indptr.tolist() == [0]
    with pytest.raises(ValueError):
        oracle_mod.block_build(2, np.array([0, 2], np.int32), np.array([1, 1], np.int64), None, None, 1)
