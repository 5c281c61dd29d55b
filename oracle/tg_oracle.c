/*
 * tg_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision restatement of what libfasttg computes, written from the
 * paper's definitions before any CUDA kernel existed.  It shares no code, header, table or
 * helper with paper_2607_05095_b200/csrc.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.
 *
 * What it follows (reference = /root/reference/PAPER.md, FAST, arxiv/paper_2607_05095):
 *   - compression triple uni_ID / inv_Idx / ind_ptr ........ PAPER.md:162 (§4.2), PAPER.md:287 (§5)
 *   - AGG  h_v = sum_{u in N_in(v)} v_u ...................... PAPER.md:215 (§4.3 "Balanced Aggregate"), Eq.(1)
 *   - ESM  numerically stable softmax: max-reduce, sum-reduce,
 *          element-wise division, per destination ........... PAPER.md:225 (§4.3 "Edge Softmax")
 *   - backward of AGG / ESM ("forward and backward") ......... PAPER.md:231, 287; formulas are the
 *          textbook derivatives, DESIGN.md §3 readings R4-R6
 *   - SDDMM per-edge logits (DGL gSDDMM, only named) ......... PAPER.md:94; DESIGN.md §3 reading R1
 *
 * Every op is the definition written out as loops.  No blocking, no fusion, no online softmax,
 * no splitting.  `#pragma omp parallel for` appears only over independent output rows.
 *
 * Pins (tests/test_oracle_*.py): np.unique / scipy.sparse for the index structures, brute force,
 * closed forms (single neighbour, equal logits, two-neighbour sigmoid), shift invariance,
 * torch float64 scaled_dot_product_attention on regular blocks, torch float64 autograd on a
 * padded-dense formulation, central finite differences, gradient identities.
 *
 * Conventions: row-major contiguous; E edges in destination-grouped CSR order; v(e) = the
 * destination whose indptr range holds e; r(e) = kv_row[e].
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------ */
/* Index structures (integer, exact).  DESIGN.md §3 readings R7-R10.                             */
/* ------------------------------------------------------------------------------------------ */

static int cmp_i64(const void* a, const void* b) {
    int64_t x = *(const int64_t*)a, y = *(const int64_t*)b;
    return (x > y) - (x < y);
}

/* rank of key in ascending distinct array u[0..n): plain binary search */
static int64_t rank_of(const int64_t* u, int64_t n, int64_t key) {
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        int64_t mid = lo + (hi - lo) / 2;
        if (u[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

/*
 * ind_ptr / perm: stable group-by-destination of the sampler's COO list (PAPER.md:229 CSR, 287).
 * uni_ID / inv_Idx: ascending distinct neighbour ids and each edge's rank.
 * Transposed CSR for the backward gather (north_star; not in the paper, which scatters with
 * atomics).
 * Returns 0 on success, 1 on an out-of-range root index, 2 on allocation failure.
 */
int ora_block_build(int64_t R, int64_t E, const int32_t* root_idx, const int64_t* nbr_node,
                    const int64_t* edge_id, const float* ts, int dedup_mode,
                    int32_t* indptr, int32_t* perm, int32_t* kv_row, int64_t* uniq_node,
                    int32_t* t_indptr, int32_t* t_edge, int32_t* t_dst,
                    int64_t* eid_csr, float* ts_csr, int64_t* U_out) {
    int64_t e, v, u;
    /* 1. indptr = exclusive prefix sum of bincount(root_idx) */
    for (v = 0; v <= R; ++v) indptr[v] = 0;
    for (e = 0; e < E; ++e) {
        if (root_idx[e] < 0 || root_idx[e] >= R) return 1;
        indptr[root_idx[e] + 1] += 1;
    }
    for (v = 0; v < R; ++v) indptr[v + 1] += indptr[v];
    /* perm = stable argsort of root_idx: walk the input in order, append to its destination */
    int32_t* cursor = (int32_t*)malloc(sizeof(int32_t) * (size_t)(R + 1));
    int32_t* dst_of = (int32_t*)malloc(sizeof(int32_t) * (size_t)(E + 1));
    if (!cursor || !dst_of) { free(cursor); free(dst_of); return 2; }
    for (v = 0; v < R; ++v) cursor[v] = indptr[v];
    for (e = 0; e < E; ++e) {
        int32_t pos = cursor[root_idx[e]]++;
        perm[pos] = (int32_t)e;
        dst_of[pos] = root_idx[e];
    }
    free(cursor);
    /* 4. pass-through arrays in CSR order */
    for (e = 0; e < E; ++e) {
        if (eid_csr && edge_id) eid_csr[e] = edge_id[perm[e]];
        if (ts_csr && ts) ts_csr[e] = ts[perm[e]];
    }
    /* 2. unique rows */
    int64_t U;
    if (dedup_mode == 0) {
        U = E;
        for (e = 0; e < E; ++e) { kv_row[e] = (int32_t)e; uniq_node[e] = nbr_node[perm[e]]; }
    } else {
        int64_t* sorted = (int64_t*)malloc(sizeof(int64_t) * (size_t)(E + 1));
        if (!sorted) { free(dst_of); return 2; }
        for (e = 0; e < E; ++e) sorted[e] = nbr_node[e];
        qsort(sorted, (size_t)E, sizeof(int64_t), cmp_i64);
        U = 0;
        for (e = 0; e < E; ++e)
            if (e == 0 || sorted[e] != sorted[e - 1]) uniq_node[U++] = sorted[e];
        free(sorted);
        for (e = 0; e < E; ++e) kv_row[e] = (int32_t)rank_of(uniq_node, U, nbr_node[perm[e]]);
    }
    /* 3. transposed CSR: stable group-by-row of the CSR positions */
    for (u = 0; u <= U; ++u) t_indptr[u] = 0;
    for (e = 0; e < E; ++e) t_indptr[kv_row[e] + 1] += 1;
    for (u = 0; u < U; ++u) t_indptr[u + 1] += t_indptr[u];
    int32_t* tcur = (int32_t*)malloc(sizeof(int32_t) * (size_t)(U + 1));
    if (!tcur) { free(dst_of); return 2; }
    for (u = 0; u < U; ++u) tcur[u] = t_indptr[u];
    for (e = 0; e < E; ++e) {
        int32_t pos = tcur[kv_row[e]]++;
        t_edge[pos] = (int32_t)e;
        t_dst[pos] = dst_of[e];
    }
    free(tcur);
    free(dst_of);
    *U_out = U;
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* Floating-point definitions, double precision.                                               */
/* ------------------------------------------------------------------------------------------ */

/* s[e,h] = scale * <A[v(e),h,:], B[r(e),h,:]>   (R1; gSDDMM named at PAPER.md:94) */
void ora_sddmm(int64_t R, int64_t H, int64_t D, const int32_t* indptr, const int32_t* kv_row,
               const double* A, const double* B, double scale, double* s) {
    int64_t F = H * D;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t v = 0; v < R; ++v)
        for (int64_t e = indptr[v]; e < indptr[v + 1]; ++e)
            for (int64_t h = 0; h < H; ++h) {
                const double* a = A + v * F + h * D;
                const double* b = B + (int64_t)kv_row[e] * F + h * D;
                double acc = 0.0;
                for (int64_t d = 0; d < D; ++d) acc += a[d] * b[d];
                s[e * H + h] = scale * acc;
            }
}

/* ESM forward: max reduction, sum reduction, element-wise division, per (v,h). */
void ora_edge_softmax_fwd(int64_t R, int64_t H, const int32_t* indptr, const double* s, double* alpha) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t v = 0; v < R; ++v)
        for (int64_t h = 0; h < H; ++h) {
            int64_t b = indptr[v], en = indptr[v + 1];
            if (b == en) continue;
            double m = -INFINITY, l = 0.0;
            for (int64_t e = b; e < en; ++e) if (s[e * H + h] > m) m = s[e * H + h];
            for (int64_t e = b; e < en; ++e) l += exp(s[e * H + h] - m);
            for (int64_t e = b; e < en; ++e) alpha[e * H + h] = exp(s[e * H + h] - m) / l;
        }
}

/* ESM backward: ds = alpha * (dalpha - sum_{N(v)} alpha*dalpha)   (softmax Jacobian) */
void ora_edge_softmax_bwd(int64_t R, int64_t H, const int32_t* indptr, const double* alpha,
                          const double* dalpha, double* ds) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t v = 0; v < R; ++v)
        for (int64_t h = 0; h < H; ++h) {
            double dot = 0.0;
            for (int64_t e = indptr[v]; e < indptr[v + 1]; ++e) dot += alpha[e * H + h] * dalpha[e * H + h];
            for (int64_t e = indptr[v]; e < indptr[v + 1]; ++e)
                ds[e * H + h] = alpha[e * H + h] * (dalpha[e * H + h] - dot);
        }
}

/* AGG forward: Y[v] = sum_{e in N(v)} w[e,h] * X[r(e)];  w == NULL -> plain sum. */
void ora_aggregate_fwd(int64_t R, int64_t H, int64_t D, const int32_t* indptr, const int32_t* kv_row,
                       const double* w, const double* X, double* Y) {
    int64_t F = H * D;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t v = 0; v < R; ++v) {
        for (int64_t i = 0; i < F; ++i) Y[v * F + i] = 0.0;
        for (int64_t e = indptr[v]; e < indptr[v + 1]; ++e)
            for (int64_t h = 0; h < H; ++h) {
                double we = w ? w[e * H + h] : 1.0;
                const double* x = X + (int64_t)kv_row[e] * F + h * D;
                for (int64_t d = 0; d < D; ++d) Y[v * F + h * D + d] += we * x[d];
            }
    }
}

/* AGG backward: dX[u] = sum_{e: r(e)=u} w[e,h]*dY[v(e)];  dw[e,h] = <dY[v(e),h,:], X[r(e),h,:]>.
 * Written as the scatter the definition states (serial over edges). */
void ora_aggregate_bwd(int64_t R, int64_t U, int64_t H, int64_t D, const int32_t* indptr, const int32_t* kv_row,
                       const double* w, const double* X, const double* dY, double* dX, double* dw) {
    int64_t F = H * D;
    for (int64_t i = 0; i < U * F; ++i) dX[i] = 0.0;
    for (int64_t v = 0; v < R; ++v)
        for (int64_t e = indptr[v]; e < indptr[v + 1]; ++e)
            for (int64_t h = 0; h < H; ++h) {
                double we = w ? w[e * H + h] : 1.0;
                const double* g = dY + v * F + h * D;
                double* dx = dX + (int64_t)kv_row[e] * F + h * D;
                for (int64_t d = 0; d < D; ++d) dx[d] += we * g[d];
                if (dw && X) {
                    const double* x = X + (int64_t)kv_row[e] * F + h * D;
                    double acc = 0.0;
                    for (int64_t d = 0; d < D; ++d) acc += g[d] * x[d];
                    dw[e * H + h] = acc;
                }
            }
}

/*
 * Fused attention forward = SDDMM -> ESM -> alpha-weighted AGG, as three plain stages per
 * destination (definitions in DESIGN.md §2).  LSE[v,h] = m + ln l.  Zero-degree destination:
 * O = 0, LSE = -inf (R5).  alpha_out (nullable) receives alpha[E,H].
 */
void ora_attn_fwd(int64_t R, int64_t H, int64_t D, const int32_t* indptr, const int32_t* kv_row,
                  const double* Q, const double* K, const double* V, double scale,
                  double* O, double* LSE, double* alpha_out) {
    int64_t F = H * D;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t v = 0; v < R; ++v) {
        int64_t b = indptr[v], en = indptr[v + 1], n = en - b;
        for (int64_t i = 0; i < F; ++i) O[v * F + i] = 0.0;
        if (n == 0) { for (int64_t h = 0; h < H; ++h) LSE[v * H + h] = -INFINITY; continue; }
        double* s = (double*)malloc(sizeof(double) * (size_t)n);
        for (int64_t h = 0; h < H; ++h) {
            const double* q = Q + v * F + h * D;
            double m = -INFINITY, l = 0.0;
            for (int64_t e = b; e < en; ++e) {
                const double* k = K + (int64_t)kv_row[e] * F + h * D;
                double acc = 0.0;
                for (int64_t d = 0; d < D; ++d) acc += q[d] * k[d];
                s[e - b] = scale * acc;
                if (s[e - b] > m) m = s[e - b];
            }
            for (int64_t e = b; e < en; ++e) l += exp(s[e - b] - m);
            LSE[v * H + h] = m + log(l);
            for (int64_t e = b; e < en; ++e) {
                double a = exp(s[e - b] - m) / l;
                if (alpha_out) alpha_out[e * H + h] = a;
                const double* x = V + (int64_t)kv_row[e] * F + h * D;
                for (int64_t d = 0; d < D; ++d) O[v * F + h * D + d] += a * x[d];
            }
        }
        free(s);
    }
}

/*
 * Fused attention backward for upstream gradient dO (L = sum dO*O):
 *   dalpha[e,h] = <dO[v(e),h,:], V[r(e),h,:]>;  delta[v,h] = sum_{N(v)} alpha*dalpha;
 *   ds = alpha*(dalpha - delta);
 *   dQ[v]  = scale * sum_{N(v)} ds * K[r(e)];
 *   dK[u]  = scale * sum_{r(e)=u} ds * Q[v(e)];     dV[u] = sum_{r(e)=u} alpha * dO[v(e)].
 * Stage 1 (per destination) recomputes s, alpha as in ora_attn_fwd and stores alpha, ds per edge;
 * stage 2 sums per unique row over the edges that reference it (row lists built by a stable
 * counting sort, the same definition as the transposed CSR).  Returns 0, or 2 on allocation failure.
 */
int ora_attn_bwd(int64_t R, int64_t U, int64_t H, int64_t D, const int32_t* indptr, const int32_t* kv_row,
                 const double* Q, const double* K, const double* V, const double* dO, double scale,
                 double* dQ, double* dK, double* dV) {
    int64_t F = H * D, E = indptr[R];
    double* alpha = (double*)malloc(sizeof(double) * (size_t)(E * H + 1));
    double* ds = (double*)malloc(sizeof(double) * (size_t)(E * H + 1));
    int32_t* dst_of = (int32_t*)malloc(sizeof(int32_t) * (size_t)(E + 1));
    int32_t* tptr = (int32_t*)calloc((size_t)(U + 2), sizeof(int32_t));
    int32_t* tedge = (int32_t*)malloc(sizeof(int32_t) * (size_t)(E + 1));
    if (!alpha || !ds || !dst_of || !tptr || !tedge) { free(alpha); free(ds); free(dst_of); free(tptr); free(tedge); return 2; }
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t v = 0; v < R; ++v) {
        int64_t b = indptr[v], en = indptr[v + 1];
        for (int64_t i = 0; i < F; ++i) dQ[v * F + i] = 0.0;
        for (int64_t e = b; e < en; ++e) dst_of[e] = (int32_t)v;
        for (int64_t h = 0; h < H; ++h) {
            const double* q = Q + v * F + h * D;
            const double* g = dO + v * F + h * D;
            double m = -INFINITY, l = 0.0, delta = 0.0;
            for (int64_t e = b; e < en; ++e) {
                const double* k = K + (int64_t)kv_row[e] * F + h * D;
                double acc = 0.0;
                for (int64_t d = 0; d < D; ++d) acc += q[d] * k[d];
                ds[e * H + h] = scale * acc;            /* holds s for now */
                if (scale * acc > m) m = scale * acc;
            }
            for (int64_t e = b; e < en; ++e) l += exp(ds[e * H + h] - m);
            for (int64_t e = b; e < en; ++e) alpha[e * H + h] = exp(ds[e * H + h] - m) / l;
            for (int64_t e = b; e < en; ++e) {
                const double* x = V + (int64_t)kv_row[e] * F + h * D;
                double da = 0.0;
                for (int64_t d = 0; d < D; ++d) da += g[d] * x[d];
                ds[e * H + h] = da;                     /* holds dalpha for now */
                delta += alpha[e * H + h] * da;
            }
            for (int64_t e = b; e < en; ++e) {
                ds[e * H + h] = alpha[e * H + h] * (ds[e * H + h] - delta);
                const double* k = K + (int64_t)kv_row[e] * F + h * D;
                for (int64_t d = 0; d < D; ++d) dQ[v * F + h * D + d] += scale * ds[e * H + h] * k[d];
            }
        }
    }
    for (int64_t e = 0; e < E; ++e) tptr[kv_row[e] + 1] += 1;
    for (int64_t u = 0; u < U; ++u) tptr[u + 1] += tptr[u];
    {
        int32_t* cur = (int32_t*)malloc(sizeof(int32_t) * (size_t)(U + 1));
        if (!cur) { free(alpha); free(ds); free(dst_of); free(tptr); free(tedge); return 2; }
        for (int64_t u = 0; u < U; ++u) cur[u] = tptr[u];
        for (int64_t e = 0; e < E; ++e) tedge[cur[kv_row[e]]++] = (int32_t)e;
        free(cur);
    }
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t u = 0; u < U; ++u) {
        for (int64_t i = 0; i < F; ++i) { dK[u * F + i] = 0.0; dV[u * F + i] = 0.0; }
        for (int64_t j = tptr[u]; j < tptr[u + 1]; ++j) {
            int64_t e = tedge[j], v = dst_of[e];
            for (int64_t h = 0; h < H; ++h)
                for (int64_t d = 0; d < D; ++d) {
                    dK[u * F + h * D + d] += scale * ds[e * H + h] * Q[v * F + h * D + d];
                    dV[u * F + h * D + d] += alpha[e * H + h] * dO[v * F + h * D + d];
                }
        }
    }
    free(alpha); free(ds); free(dst_of); free(tptr); free(tedge);
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* NEXT-1: the full TGAT edge term.  Temporal attention carries "temporal and   */
/* edge information during message passing": every sampled edge adds its own   */
/* row (time encoding / edge-feature projection) to the gathered key and value, and TGAT-style     */
/* logits pass a LeakyReLU.  Definitions (readings R22-R23), per head h:             */
/*   z[e,h]  = scale * <Q[v(e),h,:], K[r(e),h,:] + Ke[e,h,:]>                                      */
/*   s[e,h]  = z > 0 ? z : slope*z            (slope = 1: no non-linearity)                         */
/*   alpha   = softmax over N(v) of s (three plain passes);  LSE = m + ln l                        */
/*   O[v,h,:] = sum_{N(v)} alpha[e,h] * (V[r(e),h,:] + Ve[e,h,:])                                  */
/* Ke, Ve are [E,H,D] in CSR order and may be NULL (= 0).                                          */
/* ------------------------------------------------------------------------------------------ */
void ora_attn_edge_fwd(int64_t R, int64_t H, int64_t D, const int32_t* indptr, const int32_t* kv_row,
                       const double* Q, const double* K, const double* V, const double* Ke, const double* Ve,
                       double scale, double slope, double* O, double* LSE) {
    int64_t F = H * D;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t v = 0; v < R; ++v) {
        int64_t b = indptr[v], en = indptr[v + 1], n = en - b;
        for (int64_t i = 0; i < F; ++i) O[v * F + i] = 0.0;
        if (n == 0) { for (int64_t h = 0; h < H; ++h) LSE[v * H + h] = -INFINITY; continue; }
        double* s = (double*)malloc(sizeof(double) * (size_t)n);
        for (int64_t h = 0; h < H; ++h) {
            const double* q = Q + v * F + h * D;
            double m = -INFINITY, l = 0.0;
            for (int64_t e = b; e < en; ++e) {
                const double* k = K + (int64_t)kv_row[e] * F + h * D;
                double acc = 0.0;
                for (int64_t d = 0; d < D; ++d) acc += q[d] * (k[d] + (Ke ? Ke[e * F + h * D + d] : 0.0));
                double z = scale * acc;
                s[e - b] = z > 0.0 ? z : slope * z;
                if (s[e - b] > m) m = s[e - b];
            }
            for (int64_t e = b; e < en; ++e) l += exp(s[e - b] - m);
            LSE[v * H + h] = m + log(l);
            for (int64_t e = b; e < en; ++e) {
                double a = exp(s[e - b] - m) / l;
                const double* x = V + (int64_t)kv_row[e] * F + h * D;
                for (int64_t d = 0; d < D; ++d) O[v * F + h * D + d] += a * (x[d] + (Ve ? Ve[e * F + h * D + d] : 0.0));
            }
        }
        free(s);
    }
}

/*
 * Backward of the edge term for upstream dO:
 *   dalpha = <dO[v], V[r]+Ve[e]>; delta = sum alpha*dalpha; ds = alpha*(dalpha - delta);
 *   dz = ds * (z > 0 ? 1 : slope);
 *   dQ[v] = scale * sum dz*(K[r]+Ke[e]);  dKe[e] = scale*dz*Q[v];  dVe[e] = alpha*dO[v];
 *   dK[u] = sum_{r(e)=u} dKe[e];  dV[u] = sum_{r(e)=u} dVe[e].
 * dKe, dVe [E,H,D] are always written (they are the per-edge terms of dK, dV).
 */
void ora_attn_edge_bwd(int64_t R, int64_t U, int64_t H, int64_t D, const int32_t* indptr, const int32_t* kv_row,
                       const double* Q, const double* K, const double* V, const double* Ke, const double* Ve,
                       const double* dO, double scale, double slope,
                       double* dQ, double* dK, double* dV, double* dKe, double* dVe) {
    int64_t F = H * D, E = indptr[R];
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t v = 0; v < R; ++v) {
        int64_t b = indptr[v], en = indptr[v + 1], n = en - b;
        for (int64_t i = 0; i < F; ++i) dQ[v * F + i] = 0.0;
        if (n == 0) continue;
        double* z = (double*)malloc(sizeof(double) * (size_t)n * 3);
        double *al = z + n, *da = z + 2 * n;
        for (int64_t h = 0; h < H; ++h) {
            const double* q = Q + v * F + h * D;
            const double* g = dO + v * F + h * D;
            double m = -INFINITY, l = 0.0, delta = 0.0;
            for (int64_t e = b; e < en; ++e) {
                const double* k = K + (int64_t)kv_row[e] * F + h * D;
                double acc = 0.0;
                for (int64_t d = 0; d < D; ++d) acc += q[d] * (k[d] + (Ke ? Ke[e * F + h * D + d] : 0.0));
                z[e - b] = scale * acc;
                double s = z[e - b] > 0.0 ? z[e - b] : slope * z[e - b];
                if (s > m) m = s;
            }
            for (int64_t e = b; e < en; ++e) { double s = z[e - b] > 0.0 ? z[e - b] : slope * z[e - b]; l += exp(s - m); }
            for (int64_t e = b; e < en; ++e) {
                double s = z[e - b] > 0.0 ? z[e - b] : slope * z[e - b];
                al[e - b] = exp(s - m) / l;
                const double* x = V + (int64_t)kv_row[e] * F + h * D;
                double t = 0.0;
                for (int64_t d = 0; d < D; ++d) t += g[d] * (x[d] + (Ve ? Ve[e * F + h * D + d] : 0.0));
                da[e - b] = t;
                delta += al[e - b] * t;
            }
            for (int64_t e = b; e < en; ++e) {
                double dsv = al[e - b] * (da[e - b] - delta);
                double dz = dsv * (z[e - b] > 0.0 ? 1.0 : slope);
                const double* k = K + (int64_t)kv_row[e] * F + h * D;
                for (int64_t d = 0; d < D; ++d) {
                    dQ[v * F + h * D + d] += scale * dz * (k[d] + (Ke ? Ke[e * F + h * D + d] : 0.0));
                    dKe[e * F + h * D + d] = scale * dz * q[d];
                    dVe[e * F + h * D + d] = al[e - b] * g[d];
                }
            }
        }
        free(z);
    }
    for (int64_t i = 0; i < U * F; ++i) { dK[i] = 0.0; dV[i] = 0.0; }
    for (int64_t e = 0; e < E; ++e)      /* plain sequential sum in CSR order */
        for (int64_t i = 0; i < F; ++i) {
            dK[(int64_t)kv_row[e] * F + i] += dKe[e * F + i];
            dV[(int64_t)kv_row[e] * F + i] += dVe[e * F + i];
        }
}

int ora_num_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* thread count of the timing legs (bench.py cpu_baseline at 1 thread and at all cores); no arithmetic */
void ora_set_num_threads(int n) {
#ifdef _OPENMP
    extern void omp_set_num_threads(int);
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
