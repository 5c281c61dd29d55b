"""CPU ORACLE for NEXT-2: SlimCache's selection and its device half.  TEST INFRASTRUCTURE.

Follows PAPER.md §4.2 (lines 156-201): ID-based compression ("only unique IDs and their corresponding features are
transferred, along with an inverse index for reconstruction on the GPU") and Algorithm 1, the greedy
hot-set selection under a cache budget, step by step in the paper's order and notation.
Plain NumPy / Python loops; shares nothing with paper_2607_05095_b200.

Readings: Alg. 1 line 6 `argsort` is by DESCENDING frequency (the greedy picks the most frequent first),
ties by ascending id; line 8's budget test `i + j < alpha(|V| + |E|)` is a real comparison; when one of the two lists is
exhausted the other one is taken (the paper's loop is silent); line 9 uses a strict `>`, so a tie goes to the edge.
"""
import numpy as np


def greedy_select(alpha, batches, n_nodes, n_edges):
    """Algorithm 1.  batches: iterable of (node_id_array, edge_id_array), each the id SET of one pre-sampled mini-batch.
    Returns (H_N, H_E) as int64 arrays in selection order, and the frequency vectors (f_v, f_e)."""
    f_v = np.zeros(n_nodes, np.int64)                              # line 1
    f_e = np.zeros(n_edges, np.int64)
    for N_k, E_k in batches:                                       # lines 2-5: count frequencies
        f_v[np.unique(np.asarray(N_k, np.int64))] += 1
        f_e[np.unique(np.asarray(E_k, np.int64))] += 1
    s_v = np.argsort(-f_v, kind="stable")                          # line 6 (descending, ties by id)
    s_e = np.argsort(-f_e, kind="stable")
    i = j = 0                                                      # line 7
    H_N, H_E = [], []
    while i + j < alpha * (n_nodes + n_edges) and (i < n_nodes or j < n_edges):   # line 8
        if i < n_nodes and (j >= n_edges or f_v[s_v[i]] > f_e[s_e[j]]):           # line 9
            H_N.append(int(s_v[i])); i += 1                        # lines 10-11
        else:
            H_E.append(int(s_e[j])); j += 1                        # lines 13-14
    return np.array(H_N, np.int64), np.array(H_E, np.int64), f_v, f_e


def cache_lookup(uniq_ids, slot_of_id):
    """Runtime stage: for the batch's unique ids, which rows are resident (slot_of_id[id] >= 0) and which
    must be transferred.  Returns map[U] (>= 0: position among the transferred rows, in the order of uniq_ids;
    < 0: -(cache slot) - 1) and fresh_ids (the ids to transfer, same order)."""
    uniq_ids = np.asarray(uniq_ids, np.int64)
    m = np.zeros(len(uniq_ids), np.int32)
    fresh = []
    for u, x in enumerate(uniq_ids):
        s = int(slot_of_id[x])
        if s >= 0:
            m[u] = -s - 1
        else:
            m[u] = len(fresh)
            fresh.append(int(x))
    return m, np.array(fresh, np.int64)


def reconstruct(inv_idx, map_, fresh_rows, cache_rows):
    """X[i] = the feature row of occurrence i: through the inverse index to the unique id, then from the transferred
    rows or from the resident cache."""
    inv_idx = np.asarray(inv_idx)
    out = np.zeros((len(inv_idx),) + fresh_rows.shape[1:], fresh_rows.dtype)
    for i, u in enumerate(inv_idx):
        m = int(map_[u])
        out[i] = fresh_rows[m] if m >= 0 else cache_rows[-m - 1]
    return out
