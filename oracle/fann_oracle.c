/*
 * fann_oracle.c -- CPU oracle for the GPU stage of FusionANNS (arxiv 2409.16576).
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this
 * file.  It shares no code, header, table or helper with the CUDA library in
 * paper_2409_16576_b200/ and neither includes the other.
 *
 * What it computes (per query, section 3 "Online Processing",
 * L125-L133, steps (1)(5)(6)(7) of Fig. 6), written as the plain definitions:
 *
 *   (1) distance lookup table   PAPER.md:L82, L87   -> oracle_build_lut
 *   (5) vector-ID dedup         PAPER.md:L127       -> oracle_dedup
 *   (6) PQ (ADC) distance       PAPER.md:L84 Eq. 1  -> oracle_adc
 *   (7) sort, return top-n      PAPER.md:L133       -> oracle_topk
 *
 * The method reaches exactly a plainly-defined result (set of distinct IDs, a
 * finite sum, the k smallest), so each function below IS that definition:
 * no hashing, no partial selection, no blocking, no SIMD.  Floating point is
 * fp64 throughout; the fp32 value the GPU is compared with is the fp64 result
 * rounded once.  Readings of the paper: squared L2
 * (R1), dedup per query (R6), order (dist asc, id asc) (R11), padding with
 * (+inf, 0xFFFFFFFF) (R12), IDs 0xFFFFFFFF skipped and IDs >= N dropped (R13).
 *
 * Pins (tests/test_oracle_pins.py, `-m "not gpu"`): every function is pinned
 * against something other than itself -- see the list in DESIGN.md "Oracle
 * pins".  No function here is "parity unpinned".  The paper prints no worked
 * numeric example for this path, so no pin is a paper-printed value.
 *
 * Parallelism: `omp parallel for schedule(dynamic)` over queries only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_ID_NONE 0xFFFFFFFFu

/* (1) PAPER.md:L82 "a distance lookup table is first generated, including all
 * distances between a sub-query-vector and centroids per sub-space".
 * lut64[b][m][j] = sum_{t<dsub} (q[b][m*dsub+t] - cb[m][j][t])^2, squared L2. */
void oracle_build_lut(const float *queries, const float *codebooks, uint32_t B,
                      uint32_t M, uint32_t dsub, double *lut64)
{
    const uint32_t d = M * dsub;
    for (uint32_t b = 0; b < B; ++b)
        for (uint32_t m = 0; m < M; ++m)
            for (uint32_t j = 0; j < 256; ++j) {
                double s = 0.0;
                for (uint32_t t = 0; t < dsub; ++t) {
                    double delta = (double)queries[(size_t)b * d + m * dsub + t]
                                 - (double)codebooks[((size_t)m * 256 + j) * dsub + t];
                    s += delta * delta;
                }
                lut64[((size_t)b * M + m) * 256 + j] = s;
            }
}

static int cmp_u32(const void *a, const void *b)
{
    uint32_t x = *(const uint32_t *)a, y = *(const uint32_t *)b;
    return (x > y) - (x < y);
}

/* (5) PAPER.md:L127 "it first deduplicates them": the set of distinct valid
 * IDs, ascending.  Returns U; out must hold n entries. */
uint64_t oracle_dedup(const uint32_t *ids, uint64_t n, uint64_t N, uint32_t *out)
{
    uint64_t c = 0;
    for (uint64_t i = 0; i < n; ++i)
        if (ids[i] != ORACLE_ID_NONE && (uint64_t)ids[i] < N)
            out[c++] = ids[i];
    qsort(out, c, sizeof(uint32_t), cmp_u32);
    uint64_t u = 0;
    for (uint64_t i = 0; i < c; ++i)
        if (u == 0 || out[u - 1] != out[i])
            out[u++] = out[i];
    return u;
}

/* (6) PAPER.md:L84 Eq. 1: dist^(q, v) = sum_{i=1..M} dist(q_i, c_i(v_i)), each
 * term read from the table with the PQ code byte as the address (L87). */
double oracle_adc(const double *lut64_q, const uint8_t *codes, uint32_t M, uint64_t id)
{
    double s = 0.0;
    for (uint32_t m = 0; m < M; ++m)
        s += lut64_q[(size_t)m * 256 + codes[id * M + m]];
    return s;
}

typedef struct { float d; uint32_t id; double d64; } pair_t;

static int cmp_pair(const void *a, const void *b)
{
    const pair_t *x = (const pair_t *)a, *y = (const pair_t *)b;
    if (x->d < y->d) return -1;
    if (x->d > y->d) return 1;
    return (x->id > y->id) - (x->id < y->id);
}

/* (7) PAPER.md:L133 "the GPU sorts all distances and returns the top-n
 * vectors' ID": full sort by (fp32 distance asc, id asc), first min(k, U);
 * the rest padded with (+inf, ORACLE_ID_NONE).  Ascending order is what the
 * re-ranking consumes.  Sorts `p` in place. */
static void topk_pairs(pair_t *p, uint64_t U, uint32_t k, uint32_t *out_ids,
                       float *out_dists, double *out_dists64, uint32_t *out_count)
{
    qsort(p, U, sizeof(pair_t), cmp_pair);
    uint32_t c = (U < k) ? (uint32_t)U : k;
    for (uint32_t i = 0; i < k; ++i) {
        if (i < c) {
            out_ids[i] = p[i].id; out_dists[i] = p[i].d;
            if (out_dists64) out_dists64[i] = p[i].d64;
        } else {
            out_ids[i] = ORACLE_ID_NONE; out_dists[i] = INFINITY;
            if (out_dists64) out_dists64[i] = INFINITY;
        }
    }
    *out_count = c;
}

void oracle_topk(const uint32_t *ids, const float *dists, uint64_t U, uint32_t k,
                 uint32_t *out_ids, float *out_dists, uint32_t *out_count)
{
    pair_t *p = (pair_t *)malloc((U ? U : 1) * sizeof(pair_t));
    for (uint64_t i = 0; i < U; ++i) { p[i].d = dists[i]; p[i].id = ids[i]; p[i].d64 = dists[i]; }
    topk_pairs(p, U, k, out_ids, out_dists, NULL, out_count);
    free(p);
}

/* Steps (1)(5)(6)(7) for one query.  If all_ids/all_d64 are non-NULL they
 * receive the U distinct IDs (ascending) and their fp64 distances. */
static uint64_t one_query(const float *q, const float *codebooks, const uint8_t *codes,
                          uint64_t N, uint32_t M, uint32_t dsub,
                          const uint32_t *ids, uint64_t C, uint32_t k,
                          uint32_t *out_ids, float *out_dists, double *out_dists64,
                          uint32_t *out_count, uint32_t *all_ids, double *all_d64)
{
    double *lut = (double *)malloc((size_t)M * 256 * sizeof(double));
    oracle_build_lut(q, codebooks, 1, M, dsub, lut);
    uint32_t *uniq = (uint32_t *)malloc((C ? C : 1) * sizeof(uint32_t));
    uint64_t U = oracle_dedup(ids, C, N, uniq);
    pair_t *p = (pair_t *)malloc((U ? U : 1) * sizeof(pair_t));
    for (uint64_t i = 0; i < U; ++i) {
        double s = oracle_adc(lut, codes, M, uniq[i]);
        p[i].id = uniq[i]; p[i].d64 = s; p[i].d = (float)s;
        if (all_ids) { all_ids[i] = uniq[i]; all_d64[i] = s; }
    }
    if (out_ids) topk_pairs(p, U, k, out_ids, out_dists, out_dists64, out_count);
    free(p); free(uniq); free(lut);
    return U;
}

/* The whole GPU stage for a batch.  All pointers are host pointers.
 * out_dists64 / out_uniq may be NULL.  Returns the number of threads used. */
int oracle_search(const float *queries, const float *codebooks, const uint8_t *codes,
                  uint64_t N, uint32_t M, uint32_t dsub, uint32_t B,
                  const int64_t *cand_offsets, const uint32_t *cand_ids, uint32_t k,
                  uint32_t *out_ids, float *out_dists, double *out_dists64,
                  uint32_t *out_counts, uint32_t *out_uniq, int nthreads)
{
    const uint32_t d = M * dsub;
    int used = 1;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
    used = nthreads;
#pragma omp parallel for schedule(dynamic) num_threads(nthreads)
#endif
    for (int64_t b = 0; b < (int64_t)B; ++b) {
        uint64_t C = (uint64_t)(cand_offsets[b + 1] - cand_offsets[b]);
        uint64_t U = one_query(queries + (size_t)b * d, codebooks, codes, N, M, dsub,
                               cand_ids + cand_offsets[b], C, k,
                               out_ids + (size_t)b * k, out_dists + (size_t)b * k,
                               out_dists64 ? out_dists64 + (size_t)b * k : NULL,
                               out_counts + b, NULL, NULL);
        if (out_uniq) out_uniq[b] = (uint32_t)U;
    }
    return used;
}

/* One query, every distinct candidate: all_ids[U] ascending, all_d64[U]. */
uint64_t oracle_query_all(const float *q, const float *codebooks, const uint8_t *codes,
                          uint64_t N, uint32_t M, uint32_t dsub,
                          const uint32_t *ids, uint64_t C, uint32_t *all_ids, double *all_d64)
{
    return one_query(q, codebooks, codes, N, M, dsub, ids, C, 0, NULL, NULL, NULL, NULL,
                     all_ids, all_d64);
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
