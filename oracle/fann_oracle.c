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
 * and the rows SURVEY.md 8(f) adds around that path:
 *   (3) list metadata -> candidate IDs   PAPER.md:L125, L150   -> oracle_expand_lists   (NEXT-2)
 *   (8) heuristic re-ranking, Alg. 1     PAPER.md:L164-L182    -> oracle_rerank         (NEXT-1)
 *       page-level I/O dedup, Fig. 8     PAPER.md:L198         -> oracle_page_reads     (NEXT-4)
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

/* NEXT-2, PAPER.md:L125 step (3) "the CPU ... consults the metadata to obtain the vector-IDs
 * in these posting lists" (L150: the metadata holds only the vector-IDs of every list): the candidate list of a
 * query is the concatenation, in probe order, of the ID arrays of the posting lists it probes.  Readings
 * (R21): a probe equal to 0xFFFFFFFF is padding and a probe >= n_lists names no list; both contribute
 * nothing.  Two-pass use: with cand_ids == NULL only cand_offsets[B+1] is written; returns the total. */
uint64_t oracle_expand_lists(const int64_t *list_offsets, const uint32_t *list_ids, uint64_t n_lists,
                             const uint32_t *probes, uint32_t B, uint32_t nprobe,
                             int64_t *cand_offsets, uint32_t *cand_ids)
{
    uint64_t total = 0;
    for (uint32_t b = 0; b < B; ++b) {
        cand_offsets[b] = (int64_t)total;
        for (uint32_t j = 0; j < nprobe; ++j) {
            uint32_t l = probes[(size_t)b * nprobe + j];
            if (l == ORACLE_ID_NONE || (uint64_t)l >= n_lists) continue;
            for (int64_t e = list_offsets[l]; e < list_offsets[l + 1]; ++e) {
                if (cand_ids) cand_ids[total] = list_ids[e];
                ++total;
            }
        }
    }
    cand_offsets[B] = (int64_t)total;
    return total;
}

/* ---------------------------------------------------------------------------------------------------------
 * NEXT-1: heuristic re-ranking, PAPER.md:L164-L182 (section 4.2, Eq. 3 at L174, Algorithm 1
 * at L182).  An iteration with a heuristic stop, so it is followed step by step in the paper's order and
 * notation: a max-heap Q of capacity k, mini-batches of BatchSize tasks, change rate Delta, StabilityCounter.
 *
 * Readings (R22-R25; S20 of SURVEY.md): distance = exact squared L2 on the raw vectors (R1), computed
 * in fp64 and rounded once to fp32 before any comparison (the precision the GPU decides in); Delta's
 * denominator is k (Eq. 3; the pseudo-code's "L" is a garbled k); stop when StabilityCounter >= beta
 * (pseudo-code, L182); "insert ... if its distance is less than the current maximum distance" (L172) is a strict
 * "<" on the distance, and while Q holds fewer than k vectors every task is inserted; the vector that leaves Q
 * is the one with the largest distance, the latest inserted among equals (so Q is at all times the k smallest
 * of the tasks seen so far under the order (distance, position in Tasks)); a task ID equal to 0xFFFFFFFF ends
 * the task list (padding of the top-n list) and an ID >= N is skipped; Q is returned ascending by
 * (distance, position).  Delta < eps is evaluated as (double)c / (double)k < (double)eps.
 * --------------------------------------------------------------------------------------------------------- */
typedef struct { float d; uint32_t pos; uint32_t id; double d64; } heap_item_t;

static int heap_less(const heap_item_t *a, const heap_item_t *b)        /* order (distance, position) */
{
    if (a->d != b->d) return a->d < b->d;
    return a->pos < b->pos;
}

static void heap_sift_up(heap_item_t *h, uint32_t i)
{
    while (i > 0) {
        uint32_t p = (i - 1) / 2;
        if (!heap_less(&h[p], &h[i])) break;
        heap_item_t t = h[p]; h[p] = h[i]; h[i] = t;
        i = p;
    }
}

static void heap_sift_down(heap_item_t *h, uint32_t n, uint32_t i)
{
    for (;;) {
        uint32_t l = 2 * i + 1, r = l + 1, m = i;
        if (l < n && heap_less(&h[m], &h[l])) m = l;
        if (r < n && heap_less(&h[m], &h[r])) m = r;
        if (m == i) break;
        heap_item_t t = h[m]; h[m] = h[i]; h[i] = t;
        i = m;
    }
}

static int cmp_heap_item(const void *a, const void *b)
{
    const heap_item_t *x = (const heap_item_t *)a, *y = (const heap_item_t *)b;
    if (heap_less(x, y)) return -1;
    if (heap_less(y, x)) return 1;
    return 0;
}

/* GetDistance(Tasks[j]) of Algorithm 1 line 6, without the SSD: exact squared L2 in fp64. */
static double exact_dist(const float *q, const float *v, uint32_t d)
{
    double s = 0.0;
    for (uint32_t t = 0; t < d; ++t) {
        double delta = (double)q[t] - (double)v[t];
        s += delta * delta;
    }
    return s;
}

/* Algorithm 1 for one query.  tasks[n]: candidate IDs in ascending PQ-distance order (the GPU stage's top-n,
 * L170).  Writes Q ascending into out_ids/out_dists[k] (padded with 0xFFFFFFFF / +inf), *out_count = |Q|,
 * *out_batches = mini-batches executed.  Returns the number of tasks whose raw vector was read. */
uint32_t oracle_rerank(const float *query, const float *vectors, uint64_t N, uint32_t d,
                       const uint32_t *tasks, uint32_t n, uint32_t batch_size, uint32_t k,
                       float eps, uint32_t beta,
                       uint32_t *out_ids, float *out_dists, double *out_dists64,
                       uint32_t *out_count, uint32_t *out_batches)
{
    heap_item_t *Q = (heap_item_t *)malloc((size_t)(k ? k : 1) * sizeof(heap_item_t));   /* line 1: Q <- NULL */
    uint32_t *S_prev = (uint32_t *)malloc((size_t)(k ? k : 1) * sizeof(uint32_t));
    uint32_t qn = 0, stability = 0, batches = 0, reads = 0;                               /* line 2 */
    uint32_t n_tasks = 0;
    while (n_tasks < n && tasks[n_tasks] != ORACLE_ID_NONE) ++n_tasks;                    /* padding ends the list */
    int done = 0;
    for (uint32_t i = 0; i < n_tasks && !done; i += batch_size) {                         /* line 3 */
        uint32_t prev_n = qn;
        for (uint32_t s = 0; s < qn; ++s) S_prev[s] = Q[s].id;                            /* line 4: S_{n-1} */
        for (uint32_t j = i; j < i + batch_size && j < n_tasks; ++j) {                    /* line 5 */
            uint32_t id = tasks[j];
            if ((uint64_t)id >= N) continue;
            double d64 = exact_dist(query, vectors + (size_t)id * d, d);                  /* line 6 */
            ++reads;
            heap_item_t c; c.d = (float)d64; c.pos = j; c.id = id; c.d64 = d64;
            if (qn < k) {                                                                 /* line 7: Q.insert */
                Q[qn] = c; heap_sift_up(Q, qn); ++qn;
            } else if (k > 0 && c.d < Q[0].d) {
                Q[0] = c; heap_sift_down(Q, qn, 0);
            }
        }
        ++batches;
        uint32_t changed = 0;                                                             /* lines 9-10: Delta */
        for (uint32_t s = 0; s < qn; ++s) {
            int in_prev = 0;
            for (uint32_t t = 0; t < prev_n; ++t) if (S_prev[t] == Q[s].id) { in_prev = 1; break; }
            if (!in_prev) ++changed;
        }
        double delta = (double)changed / (double)k;
        if (delta < (double)eps) {                                                        /* line 11 */
            ++stability;                                                                  /* line 12 */
            if (stability >= beta) done = 1;                                              /* lines 13-14 */
        } else {
            stability = 0;                                                                /* line 17 */
        }
    }
    qsort(Q, qn, sizeof(heap_item_t), cmp_heap_item);                                     /* line 20: return Q */
    for (uint32_t s = 0; s < k; ++s) {
        if (s < qn) {
            out_ids[s] = Q[s].id; out_dists[s] = Q[s].d;
            if (out_dists64) out_dists64[s] = Q[s].d64;
        } else {
            out_ids[s] = ORACLE_ID_NONE; out_dists[s] = INFINITY;
            if (out_dists64) out_dists64[s] = INFINITY;
        }
    }
    *out_count = qn;
    *out_batches = batches;
    free(Q); free(S_prev);
    return reads;
}

/* ---------------------------------------------------------------------------------------------------------
 * NEXT-4: redundancy-aware I/O deduplication, PAPER.md:L198 (section 4.3, Fig. 8).
 * "merging I/Os mapped to the same SSD page within a mini-batch, and exploiting the DRAM buffer to eliminate
 * redundant I/Os in subsequent mini-batches".  For one query: the mapping table gives the page of each task's
 * vector; a mini-batch reads each page it needs once, unless the DRAM buffer already holds it; pages read
 * enter the buffer.
 *
 * Readings (R26): the buffer is per query, unbounded, and starts with the pages whose bit is set in
 * `resident` (may be NULL = empty); a task equal to 0xFFFFFFFF ends the list, an ID >= N is skipped; the
 * pages of a mini-batch are reported in order of first need.  Only the first `max_batches` mini-batches are
 * processed (what Algorithm 1 executed); 0 = all.
 * page_of[N]; out_pages[n] receives the pages read, mini-batch after mini-batch; out_batch_reads[nb] the number
 * of page reads (I/Os) of each mini-batch, nb = ceil(n / batch_size).  Returns the total number of reads.
 * --------------------------------------------------------------------------------------------------------- */
uint32_t oracle_page_reads(const uint32_t *page_of, uint64_t N, const uint32_t *tasks, uint32_t n,
                           uint32_t batch_size, uint32_t max_batches, const uint32_t *resident, uint64_t n_pages,
                           uint32_t *out_pages, uint32_t *out_batch_reads)
{
    uint32_t n_tasks = 0, total = 0, nb = (n + batch_size - 1) / batch_size;
    while (n_tasks < n && tasks[n_tasks] != ORACLE_ID_NONE) ++n_tasks;
    for (uint32_t t = 0; t < nb; ++t) out_batch_reads[t] = 0;
    for (uint32_t i = 0, t = 0; i < n_tasks; i += batch_size, ++t) {
        if (max_batches && t >= max_batches) break;
        for (uint32_t j = i; j < i + batch_size && j < n_tasks; ++j) {
            if ((uint64_t)tasks[j] >= N) continue;
            uint32_t p = page_of[tasks[j]];
            int have = resident && (uint64_t)p < n_pages && ((resident[p >> 5] >> (p & 31)) & 1u);
            for (uint32_t s = 0; s < total && !have; ++s) if (out_pages[s] == p) have = 1;   /* buffer + this batch */
            if (!have) { out_pages[total++] = p; ++out_batch_reads[t]; }
        }
    }
    return total;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
