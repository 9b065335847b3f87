/*
 * fann.h -- C ABI of the B200-native GPU stage of FusionANNS (arxiv 2409.16576).
 *
 * The library runs, batched over queries on ONE GPU, the GPU side of the
 * paper's CPU/GPU cooperative filtering (section 3 "Online
 * Processing", L125-L133, Fig. 6 steps (1)(5)(6)(7)):
 *
 *   (1) per-query PQ distance lookup table          fann_build_lut
 *   (5) dedup of the candidate vector-IDs   \
 *   (6) gather PQ codes from HBM + Eq. 1     >      fann_dedup_scan_topk
 *   (7) top-n candidates, ascending         /
 *
 * with the PQ codes pinned in HBM beforehand  fann_load_codes.
 *
 * Conventions
 *   - Plain C.  No C++ or torch types cross this boundary.
 *   - Every function that can fail returns a status (FANN_OK == 0, errors < 0)
 *     and leaves a message for fann_last_error() (thread-local).  Nothing
 *     throws, exits or allocates inside fann_build_lut / fann_dedup_scan_topk.
 *   - "device pointer" = CUDA device memory of the index's device; "host
 *     pointer" = ordinary (ideally pinned) host memory.  Each argument says which.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default
 *     stream).  Calls only ENQUEUE work and return without synchronising,
 *     unless stated otherwise.
 *   - Ownership: the index owns only its private copy of the PQ codes.
 *     Queries, codebooks, tables, candidate lists, outputs and workspace are
 *     caller-owned and must stay valid until the enqueued work has finished.
 *   - Distance is squared L2 (reading R1).  IDs are uint32.
 *     FANN_ID_NONE in a candidate list is skipped; an ID >= N is dropped.
 *   - There is no CPU fallback.  If no usable CUDA device exists the calls
 *     fail with FANN_ECUDA.
 *   - Alignment: lut 16 bytes; cand_offsets and list offsets 8 bytes; every other array 4
 *     bytes; workspaces 256 bytes.  A misaligned pointer is FANN_EINVAL / FANN_EWORKSPACE.
 *   - Threads ("each CPU thread handles an individual query"): once the codes
 *     (and posting lists / raw vectors) are loaded, any number of host threads may call the
 *     search entry points on ONE handle at the same time, each with its own stream,
 *     workspace and output arrays.  The loaders, fann_set_timing and fann_destroy must not
 *     run beside any other call on the handle; with timing enabled, calls are serialised.
 */
#ifndef FANN_H
#define FANN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fann_index fann_index;          /* opaque, library-owned */

enum {
    FANN_OK           =  0,
    FANN_EINVAL       = -1,   /* bad argument (NULL, zero size, mismatched M, ...)        */
    FANN_ECUDA        = -2,   /* CUDA runtime error; message has the CUDA error string   */
    FANN_ENOMEM       = -3,   /* device allocation failed                                 */
    FANN_EUNSUPPORTED = -4,   /* M > FANN_MAX_M, k > FANN_MAX_K, dsub == 0, ...           */
    FANN_EWORKSPACE   = -5,   /* workspace NULL, misaligned or smaller than required      */
    FANN_EOVERFLOW    = -6    /* reported by fann_workspace_status: a dedup table filled  */
};

#define FANN_ID_NONE 0xFFFFFFFFu               /* padding in candidate lists and in outputs */
#define FANN_MAX_M   64u                       /* PQ bytes per vector (lookup table <= 64 KB) */
#define FANN_MAX_K   1024u                     /* candidates returned per query             */
#define FANN_MAX_NPROBE 8192u                  /* posting lists probed per query (fann_search_lists) */
enum { FANN_ELEM_F32 = 0, FANN_ELEM_U8 = 1, FANN_ELEM_I8 = 2 };   /* raw-vector element types (fann_load_vectors) */

/* Create an index on CUDA device `device`.  *out receives the handle. */
int  fann_create(fann_index **out, int device);
/* Free the index and its copy of the codes.  Synchronises the device. NULL is a no-op. */
void fann_destroy(fann_index *ix);
/* Message of the last failing call made by this host thread.  Never NULL. */
const char *fann_last_error(void);
/* "fann <version> sm_100a". */
const char *fann_version(void);

/*
 * PAPER.md:L152 "we pin all compressed vectors in the HBM".
 * Copy rows [first, first+n) of the N_total x M uint8 PQ code array (row-major,
 * `codes` points at row `first`) into library-owned HBM.  The library stores
 * rows padded to 16, 32 or 64 bytes (M=25 -> 32, M=48 -> 64) so that a row never
 * straddles a 64-byte DRAM access and is read with aligned 16-byte loads by 1, 2
 * or 4 adjacent lanes; padding bytes are zero and never contribute.
 * The first call fixes N_total and M and allocates; later calls must repeat
 * them and may load other row ranges (so 25-64 GB can be streamed in chunks).
 * codes: host pointer if src_is_device == 0, else device pointer.
 * For a host source the call synchronises `stream` before returning.
 * Errors: EINVAL (NULL, range outside N_total, M or N_total changed, M == 0),
 * EUNSUPPORTED (M > FANN_MAX_M, N_total >= 2^32), ENOMEM, ECUDA.
 */
int fann_load_codes(fann_index *ix, const uint8_t *codes, uint64_t first, uint64_t n,
                    uint64_t N_total, uint32_t M, int src_is_device, void *stream);

/*
 * Step (1): the distance lookup table
 *     lut[b][m][j] = sum_{t<dsub} (queries[b][m*dsub+t] - codebooks[m][j][t])^2
 * in fp32, direct form (no norm expansion).  M is the index's M (codes must be
 * loaded first); d = M*dsub.
 * queries   device pointer, [B][d] fp32 row-major
 * codebooks device pointer, [M][256][dsub] fp32
 * lut       device pointer, [B][M][256] fp32, written
 * Errors: EINVAL (NULL, B == 0, codes not loaded), EUNSUPPORTED (dsub == 0 or > 64).
 */
int fann_build_lut(fann_index *ix, const float *queries, uint32_t B,
                   const float *codebooks, uint32_t dsub, float *lut, void *stream);

/*
 * Bytes of device workspace fann_dedup_scan_topk / fann_dedup_only need for a
 * batch of B queries holding total_cands candidate IDs in all.  The workspace
 * is the paper's per-query working memory turned inside out:
 * the caller allocates it once and reuses it across batches.  About 12 bytes per
 * candidate ID (the distinct IDs, and the candidate lists split into dedup classes)
 * plus small per-query arrays.  Returns 0 on a bad argument (see fann_last_error).
 */
size_t fann_workspace_bytes(const fann_index *ix, uint32_t B, uint64_t total_cands, uint32_t k);

/*
 * Steps (5)(6)(7), for a batch.  For every query b:
 *   (5) the set of distinct valid IDs among cand_ids[cand_offsets[b] .. cand_offsets[b+1])
 *   (6) Eq. 1: dist(v) = sum_m lut[b][m][codes[v][m]], fp32
 *       (summation order unspecified; exact whenever all partial sums are
 *       integers below 2^24)
 *   (7) the min(k, U_b) smallest (dist, id) pairs, ordered by dist ascending,
 *       then id ascending; the remaining slots hold (+inf, FANN_ID_NONE).
 * lut          device, [B][M][256] fp32 as written by fann_build_lut
 * cand_offsets device, [B+1] int64, non-decreasing, cand_offsets[0] == 0
 * cand_ids     device, [total_cands] uint32 (any order; a caller that keeps each posting
 *              list's IDs in ascending order gets a faster class split)
 * total_cands  host value == cand_offsets[B] (lets the call size its work
 *              without reading device memory)
 * out_ids      device, [B][k] uint32        out_dists  device, [B][k] fp32
 * out_counts   device, [B] uint32 = min(k, U_b); may be NULL
 * out_uniq     device, [B] uint32 = U_b (distinct valid IDs scored); may be NULL
 * workspace    device, >= fann_workspace_bytes(ix, B, total_cands, k), 256-byte aligned
 * Synchronous errors: EINVAL, EUNSUPPORTED (k == 0 or k > FANN_MAX_K),
 * EWORKSPACE.  Asynchronous conditions are left in the workspace and read
 * with fann_workspace_status.
 */
int fann_dedup_scan_topk(fann_index *ix, const float *lut, uint32_t B,
                         const int64_t *cand_offsets, const uint32_t *cand_ids,
                         uint64_t total_cands, uint32_t k,
                         uint32_t *out_ids, float *out_dists,
                         uint32_t *out_counts, uint32_t *out_uniq,
                         void *workspace, size_t workspace_bytes, void *stream);

/*
 * The same call for callers that cannot allocate device memory (code under CUDA
 * graph capture, serving loops and harnesses that forbid cudaMalloc): steps (5)-(7),
 * PAPER.md:L127-L133, with the workspace in a file-scope device array of the library
 * instead of a caller's allocation.  The call allocates nothing -- no cudaMalloc, no
 * cudaFree, no stream or event creation -- and enqueues on `stream` only: one
 * 256-byte memset (the workspace header: status word and work counters start at
 * zero), the kernels of fann_dedup_scan_topk, and a 4-byte device-to-device copy of
 * the status word.  Arguments, layouts and results as fann_dedup_scan_topk, plus
 * out_status  device, 1 uint32 (may be NULL): what fann_workspace_status would have
 *             reported, valid once `stream` has run the call -- 0 = results valid,
 *             FANN_STATUS_TABLE_FULL / FANN_STATUS_BAD_TOTAL bits otherwise.
 * Limit: the batch must need at most FANN_STATIC_WS_BYTES (32 MiB) of workspace, i.e.
 * fann_workspace_bytes(ix, B, total_cands, k) <= FANN_STATIC_WS_BYTES -- about 2.7 M
 * candidate IDs per call (20 queries of 128 k IDs, 80 of 32 k).  A larger batch is
 * refused with FANN_EWORKSPACE and a message naming both sizes; nothing is enqueued.
 * The array is ONE per device for the whole process (every GPU that loads the library
 * holds its 32 MiB until exit), shared by every handle and every call and keeping the
 * last call's contents: calls of this entry that overlap on the GPU -- two streams,
 * two host threads, two handles on one device -- race on it and give wrong results;
 * serialise them (one stream, or events).  It does not conflict with the entry points
 * that take a caller's workspace.  Its device address is resolved once per device in
 * fann_create; FANN_ECUDA if that failed; FANN_EUNSUPPORTED with FANN_CHUNKS > 1 (the
 * chunked path creates a stream).
 */
#define FANN_STATIC_WS_BYTES (32u * 1024u * 1024u)
#define FANN_STATUS_TABLE_FULL 1u   /* a dedup table filled up: FANN_EOVERFLOW of fann_workspace_status */
#define FANN_STATUS_BAD_TOTAL  2u   /* total_cands disagrees with cand_offsets: its FANN_EINVAL         */
int fann_dedup_scan_topk_static(fann_index *ix, const float *lut, uint32_t B,
                                const int64_t *cand_offsets, const uint32_t *cand_ids,
                                uint64_t total_cands, uint32_t k,
                                uint32_t *out_ids, float *out_dists,
                                uint32_t *out_counts, uint32_t *out_uniq,
                                uint32_t *out_status, void *stream);

/*
 * Step (5) alone, through the same kernel and hash tables as the call above
 * (test hook for the bit-exact dedup check): the distinct valid IDs of query b,
 * in any order, are written to uniq_ids[cand_offsets[b] .. +uniq_counts[b]).
 * uniq_ids device, [total_cands] uint32; uniq_counts device, [B] uint32.
 */
int fann_dedup_only(fann_index *ix, uint32_t B, const int64_t *cand_offsets,
                    const uint32_t *cand_ids, uint64_t total_cands,
                    uint32_t *uniq_ids, uint32_t *uniq_counts,
                    void *workspace, size_t workspace_bytes, void *stream);

/*
 * Synchronises `stream` and returns the status the last fann_dedup_scan_topk /
 * fann_dedup_only left in `workspace`:
 *   FANN_OK
 *   FANN_EINVAL     total_cands did not match cand_offsets (cand_offsets[0] != 0 or
 *                   cand_offsets[B] != total_cands): nothing was read or scored, every
 *                   query reports zero candidates
 *   FANN_EOVERFLOW  some query's dedup table filled up; that query's outputs are invalid.
 *                   Candidate lists whose IDs are bunched in part of [0, N) are handled
 *                   exactly (the library counts the ID-range classes and falls back to hash
 *                   classes); an overflow is left only for IDs chosen to collide under the
 *                   library's hash function.
 */
int fann_workspace_status(fann_index *ix, const void *workspace, void *stream);

/*
 * Diagnostics: how many queries of the last fann_dedup_scan_topk / fann_dedup_only call on this
 * workspace (same B, total_cands, k) were deduplicated with order-preserving placement and how
 * many fell back to hashed placement (bunched IDs).  Synchronises `stream`.
 */
int fann_workspace_modes(fann_index *ix, const void *workspace, uint32_t B, uint64_t total_cands, uint32_t k,
                         uint32_t *n_ordered, uint32_t *n_hashed, void *stream);

/*
 * The whole stage from HOST buffers, for callers that hold the batch in host
 * memory (the paper's step (4): the CPU sends the vector-IDs):
 * copies queries / candidate lists host->device into `device_scratch`, runs
 * fann_build_lut + fann_dedup_scan_topk, copies ids/dists/counts back and
 * synchronises `stream` before returning.  Codebooks stay on the device.
 * From 16 MB of candidate IDs up, the IDs go up in 8 chunks of queries on a
 * stream of the index's own and the path runs chunk by chunk behind them
 * (queries are independent), so the transfer and the kernels overlap.
 * queries_h, cand_offsets_h, cand_ids_h, out_*_h: host pointers (pinned memory
 * gives asynchronous copies); layouts as above.  out_counts_h may be NULL.
 * Output arrays that are all page-locked (cudaHostAlloc / cudaHostRegister) are
 * written by the kernels themselves through their device address -- a query's
 * results cross PCIe while other queries are still scanned and no copy follows
 * the last kernel; they are valid when the call returns, like copied ones.
 * Pageable arrays (or FANN_HOST_DIRECT=0) take a staged device->host copy.
 * device_scratch: device, >= fann_search_host_scratch_bytes(...), 256-byte aligned.
 */
size_t fann_search_host_scratch_bytes(const fann_index *ix, uint32_t B, uint32_t dsub,
                                      uint64_t total_cands, uint32_t k);
int fann_search_host(fann_index *ix, const float *queries_h, uint32_t B,
                     const float *codebooks_d, uint32_t dsub,
                     const int64_t *cand_offsets_h, const uint32_t *cand_ids_h,
                     uint32_t k, uint32_t *out_ids_h, float *out_dists_h, uint32_t *out_counts_h,
                     void *device_scratch, size_t scratch_bytes, void *stream);

/* ======================================================================================
 * Steps around the hot path.  Each is optional: the calls above never need
 * them.
 * ====================================================================================== */

/*
 * NEXT-2 -- posting-list metadata resident in HBM.  PAPER.md:L150: the host keeps, per posting
 * list, only its vector-IDs; L125 steps (3)(4): the CPU concatenates the IDs of the top-m lists
 * and sends them to the GPU -- 5 GB per batch at the largest configuration, 4x the time of the
 * kernels over PCIe.  On a 180 GB part the ID arrays of all lists (4 bytes per list entry) fit
 * beside the codes, so the host sends nprobe list indices per query instead and step (3) runs
 * on the GPU.
 *
 * fann_load_lists copies the CSR of all posting lists into library-owned HBM (replacing any
 * earlier lists): list l holds list_ids[list_offsets[l] .. list_offsets[l+1]).
 * list_offsets  [n_lists + 1] int64, list_offsets[0] == 0, list_offsets[n_lists] == n_entries
 * list_ids      [n_entries] uint32 vector-IDs (any order inside a list)
 * Host or device source (src_is_device); synchronises `stream`.
 * If the codes are loaded already (N is known) the library sorts every list of its copy
 * ascending and indexes it by 64 ID-range cells (130 bytes per list more): fann_search_lists
 * then takes every dedup partition's IDs straight from the probed lists and writes neither a
 * candidate array nor its split (nprobe <= 512; lists longer than 8192 entries, lists loaded
 * before the codes, or FANN_LISTS_DIRECT=0 take the expanding path).  Same results either way.
 * Errors: EINVAL (NULL, n_lists == 0, offsets do not end at n_entries), ENOMEM, ECUDA.
 */
int fann_load_lists(fann_index *ix, const int64_t *list_offsets, const uint32_t *list_ids,
                    uint64_t n_lists, uint64_t n_entries, int src_is_device, void *stream);

/*
 * Steps (3)(5)(6)(7) from probed list indices.  Query b's candidate list is the concatenation,
 * in probe order, of the ID arrays of lists probes[b][0 .. nprobe); a probe equal to
 * FANN_ID_NONE is padding and a probe >= n_lists names no list -- both contribute nothing.
 * From there the call is fann_dedup_scan_topk on those lists: same kernels, same results.
 * probes           device, [B][nprobe] uint32
 * max_total_cands  capacity the workspace is sized for: an upper bound of the batch's total
 *                  candidate count (sum of the probed lists' lengths).  If the batch needs
 *                  more, nothing is scored and fann_search_lists_status returns
 *                  FANN_EWORKSPACE together with the count that would have been needed.
 * workspace        device, >= fann_search_lists_workspace_bytes(ix, B, max_total_cands, k)
 * lut, out_*       as in fann_dedup_scan_topk.  Enqueues only.
 * fann_search_lists_status synchronises `stream` and returns FANN_OK, FANN_EWORKSPACE (see
 * above) or what fann_workspace_status would; *total_cands (may be NULL) receives the batch's
 * candidate count.  B, max_total_cands and k must repeat the values of the call.
 */
size_t fann_search_lists_workspace_bytes(const fann_index *ix, uint32_t B, uint64_t max_total_cands, uint32_t k);
int fann_search_lists(fann_index *ix, const float *lut, uint32_t B,
                      const uint32_t *probes, uint32_t nprobe, uint64_t max_total_cands, uint32_t k,
                      uint32_t *out_ids, float *out_dists, uint32_t *out_counts, uint32_t *out_uniq,
                      void *workspace, size_t workspace_bytes, void *stream);
int fann_search_lists_status(fann_index *ix, const void *workspace, uint32_t B, uint64_t max_total_cands,
                             uint32_t k, uint64_t *total_cands, void *stream);

/*
 * The same from HOST buffers: query vectors and probes go up (B * (4 d + 4 nprobe) bytes),
 * ids / dists / counts come back; synchronises `stream` and returns the batch's status.
 * queries_h, probes_h, out_*_h: host pointers (pinned memory gives asynchronous copies;
 * page-locked output arrays are written by the kernels directly, as in fann_search_host).
 */
size_t fann_search_lists_host_scratch_bytes(const fann_index *ix, uint32_t B, uint32_t dsub, uint32_t nprobe,
                                            uint64_t max_total_cands, uint32_t k);
int fann_search_lists_host(fann_index *ix, const float *queries_h, uint32_t B,
                           const float *codebooks_d, uint32_t dsub,
                           const uint32_t *probes_h, uint32_t nprobe, uint64_t max_total_cands, uint32_t k,
                           uint32_t *out_ids_h, float *out_dists_h, uint32_t *out_counts_h,
                           void *device_scratch, size_t scratch_bytes, void *stream);

/*
 * EXPERIMENT -- a list-major copy of the codes, streamed instead of gathered.  NOT the paper's
 * layout: the paper keeps one code per vector, indexed by vector-ID, and the
 * posting lists hold vector-IDs only (L150); this keeps, in addition, the codes in posting-list
 * order, replicas included (list_entries x row_bytes of HBM: 64 GB more at 10^9 entries of
 * 64-byte codes), so that step (6) reads each probed list as one contiguous run.  Every
 * candidate is scored, repeats included; the repeats (a vector in several probed lists has the
 * same distance and ID each time) are removed exactly where the top-k buffer is pruned, so
 * steps (5)-(7) need no dedup pass.  Results are the bytes of fann_search_lists.
 *
 * fann_build_list_codes builds the copy from the loaded codes and posting lists (enqueues on
 * `stream`; loading other lists discards it).  fann_search_lists_stream is fann_search_lists
 * on it, without out_uniq (the distinct candidates are never counted).  Its workspace holds
 * the batch's (row, vector-ID) pairs only (8 bytes per candidate).  fann_search_lists_stream_status
 * synchronises `stream` and returns FANN_OK or FANN_EWORKSPACE (max_total_cands too small;
 * *total_cands, may be NULL, receives the count that was needed).
 */
int fann_build_list_codes(fann_index *ix, void *stream);
size_t fann_search_lists_stream_workspace_bytes(const fann_index *ix, uint32_t B, uint64_t max_total_cands);
int fann_search_lists_stream(fann_index *ix, const float *lut, uint32_t B,
                             const uint32_t *probes, uint32_t nprobe, uint64_t max_total_cands, uint32_t k,
                             uint32_t *out_ids, float *out_dists, uint32_t *out_counts,
                             void *workspace, size_t workspace_bytes, void *stream);
int fann_search_lists_stream_status(fann_index *ix, const void *workspace, uint64_t *total_cands, void *stream);

/*
 * NEXT-3 -- low-latency small-batch serving, PAPER.md:L204-L208 (section 5): "each CPU thread
 * handles an individual query" and a "contention-free GPU memory manager": the HBM left after
 * the codes is cut into fixed blocks, a block is handed to a query and recycled.
 *
 * fann_pool_create cuts one HBM allocation into n_blocks blocks, each large enough for one
 * call of up to max_B queries with up to max_cands candidate IDs in total and k <= k_max
 * (max_nprobe > 0 also sizes the blocks for the posting-list form).  Every block owns a CUDA
 * stream.  fann_pool_destroy waits for the blocks' streams and frees everything.
 *
 * fann_search_small / fann_search_small_lists: the whole path for one small batch from HOST
 * buffers, as fann_search_host / fann_search_lists_host, on a block of the pool and the
 * block's stream: take a free block (waiting while all are in use), copy up, run, copy the
 * results back, synchronise the block's stream, give the block back.  Any number of host
 * threads may call concurrently on one index and one pool; calls share no workspace, stream
 * or event.  A batch of fewer queries than half the SMs is scanned by several CTAs per query
 * (each on a slice of the query's distinct list, merged on the device), so that one query
 * does not wait on one SM -- and so are its list expansion and its partition pass; results are
 * the same bytes as the batched entry points give.  fann_search_small_lists replays ONE CUDA
 * graph per call (captured per block and call shape -- B, nprobe, k, codebooks -- on first use):
 * the inputs are copied into the block's pinned staging buffer, the graph copies them up, runs
 * the kernels -- which write the results straight into the staging buffer -- and copies the
 * status back (FANN_SMALL_GRAPH=0: plain launches).
 * Errors: EINVAL (NULL, a pool of another index, B / k / dsub / nprobe outside what the pool
 * was created for), EWORKSPACE (more candidate IDs than a block holds), and what the batched
 * entry points return.
 */
typedef struct fann_pool fann_pool;
typedef struct fann_pool_info {
    uint64_t block_bytes;        /* HBM per block                                              */
    uint64_t calls;              /* blocks handed out so far                                   */
    uint64_t waits;              /* calls that found every block in use and had to wait        */
    uint32_t n_blocks, in_use;   /* blocks of the pool; blocks handed out right now            */
    uint32_t high_water;         /* most blocks in use at the same time so far                 */
    uint32_t reserved;
} fann_pool_info;
int fann_pool_create(fann_index *ix, uint32_t n_blocks, uint32_t max_B, uint64_t max_cands, uint32_t dsub,
                     uint32_t max_nprobe, uint32_t k_max, fann_pool **out);
void fann_pool_destroy(fann_pool *pool);
int fann_pool_stats(fann_pool *pool, fann_pool_info *out);
int fann_search_small(fann_index *ix, fann_pool *pool, const float *queries_h, uint32_t B,
                      const float *codebooks_d, uint32_t dsub,
                      const int64_t *cand_offsets_h, const uint32_t *cand_ids_h, uint32_t k,
                      uint32_t *out_ids_h, float *out_dists_h, uint32_t *out_counts_h);
int fann_search_small_lists(fann_index *ix, fann_pool *pool, const float *queries_h, uint32_t B,
                            const float *codebooks_d, uint32_t dsub,
                            const uint32_t *probes_h, uint32_t nprobe, uint32_t k,
                            uint32_t *out_ids_h, float *out_dists_h, uint32_t *out_counts_h);

/*
 * NEXT-1 -- heuristic re-ranking, PAPER.md:L164-L182 (section 4.2, Eq. 3, Algorithm 1), with the
 * raw vectors in HBM instead of on SSD (the configurations whose raw vectors fit).
 *
 * fann_load_vectors copies rows [first, first + n) of the N_total x d raw-vector array
 * (row-major, elem_type FANN_ELEM_F32 / _U8 / _I8, `vectors` points at row `first`) into
 * library-owned HBM; the first call fixes (N_total, d, elem_type).  d <= 2048.
 *
 * fann_rerank runs Algorithm 1 for B queries.  task_ids[b][0 .. n) is the query's candidate
 * list in ascending PQ-distance order -- out_ids of the calls above (L170) -- ended by
 * FANN_ID_NONE padding; an ID >= N_total is skipped.  Mini-batches of batch_size tasks are
 * executed in order: exact squared L2 distance (fp32) to the raw vector of every task, the
 * vector enters Q if Q holds fewer than k vectors or its distance is less than Q's largest
 * (the vector with the largest distance, the latest inserted among equals, leaves);
 * Delta = |S_n - S_n n S_{n-1}| / k (Eq. 3); the StabilityCounter counts consecutive
 * mini-batches with Delta < eps and the query stops when it reaches beta.  Raw vectors of
 * mini-batches after the stop are not read.
 * queries      device, [B][d] fp32           task_ids  device, [B][n] uint32, n <= 2048
 * out_ids      device, [B][k] uint32: Q ascending by (distance, position in task_ids), padded
 *              with FANN_ID_NONE;  out_dists [B][k] fp32, padded with +inf;  k <= 1024
 * out_counts   device, [B]: |Q|
 * out_batches  device, [B]: mini-batches executed (may be NULL)
 * out_reads    device, [B]: raw vectors read (may be NULL)
 * batch_size > n is taken as n.  Enqueues only; needs no workspace.
 * Errors: EINVAL (NULL, zero sizes, beta == 0, eps < 0, vectors not loaded), EUNSUPPORTED.
 */
int fann_load_vectors(fann_index *ix, const void *vectors, uint64_t first, uint64_t n, uint64_t N_total,
                      uint32_t d, int elem_type, int src_is_device, void *stream);
int fann_rerank(fann_index *ix, const float *queries, uint32_t B, const uint32_t *task_ids, uint32_t n,
                uint32_t batch_size, uint32_t k, float eps, uint32_t beta,
                uint32_t *out_ids, float *out_dists, uint32_t *out_counts,
                uint32_t *out_batches, uint32_t *out_reads, void *stream);

/*
 * NEXT-4 -- page-level I/O deduplication, PAPER.md:L198 (section 4.3, Fig. 8): "merging I/Os
 * mapped to the same SSD page within a mini-batch, and exploiting the DRAM buffer to eliminate
 * redundant I/Os in subsequent mini-batches".  The library computes WHICH pages each
 * mini-batch of each query has to read; it performs no I/O.
 *
 * fann_load_page_table: page_of[v] = SSD page holding raw vector v (the in-memory mapping
 * table of), N entries, page numbers < n_pages.
 *
 * fann_page_reads: for query b, mini-batch t covers task_ids[b][t*batch_size .. +batch_size)
 * (list ended by FANN_ID_NONE; IDs >= N skipped).  A mini-batch reads each page its vectors
 * need once, unless the query's DRAM buffer holds it; pages read enter the buffer.  The buffer
 * starts with the pages whose bit is set in resident_bits (bit p of word p / 32; NULL = empty).
 * Only the first batches_run[b] mini-batches are processed (what fann_rerank executed;
 * NULL or 0 = all).
 * out_pages        device, [B][n]: the pages to read, mini-batch after mini-batch (any order
 *                  inside one), padded with FANN_ID_NONE;  n <= 4096
 * out_batch_reads  device, [B][ceil(n / batch_size)]: page reads (I/Os) of each mini-batch
 * out_total        device, [B]: page reads of the query
 */
int fann_load_page_table(fann_index *ix, const uint32_t *page_of, uint64_t N, uint64_t n_pages,
                         int src_is_device, void *stream);
int fann_page_reads(fann_index *ix, const uint32_t *task_ids, uint32_t B, uint32_t n, uint32_t batch_size,
                    const uint32_t *batches_run, const uint32_t *resident_bits,
                    uint32_t *out_pages, uint32_t *out_batch_reads, uint32_t *out_total, void *stream);

/* Geometry and counters, for benchmarks and tests. */
typedef struct fann_info {
    uint64_t N;                /* rows loaded (N_total), 0 before fann_load_codes            */
    uint32_t M;                /* PQ bytes per vector                                         */
    uint32_t row_bytes;        /* stored row stride: 16, 32 or 64                             */
    uint32_t num_sms;          /* multiprocessors of the device                               */
    uint32_t dedup_threads;    /* threads per CTA of the last dedup launch: 1024 or 512       */
    uint32_t dedup_ctas;       /* persistent CTAs of the last dedup launch (1 or 2 per SM)    */
    uint32_t dedup_smem_bytes; /* dynamic shared memory per dedup CTA                         */
    uint32_t table_slots;      /* dedup table slots one CTA can hold                          */
    uint32_t scan_threads;     /* threads per CTA of the scan kernel                          */
    uint32_t scan_ctas;        /* persistent CTAs of the last scan launch                     */
    uint32_t scan_smem_bytes;  /* dynamic shared memory per scan CTA (table, buffer, ring)    */
    uint32_t scan_buffer_keys; /* top-k candidate buffer of a scan CTA, in (dist, id) keys    */
    uint32_t chunks;           /* batch chunks of the last call (1 unless FANN_CHUNKS is set) */
    uint32_t reserved;
    uint64_t kernel_launches;  /* kernels this index has launched so far                      */
    uint64_t codes_device_ptr; /* device address of the stored code array [N][row_bytes]      */
} fann_info;
int fann_get_info(const fann_index *ix, fann_info *out);

/*
 * Per-kernel device timing for benchmarks.  With enable != 0 every later
 * fann_build_lut / fann_dedup_scan_topk records CUDA events around its kernels on
 * the stream each kernel is launched on.  fann_last_timing synchronises on the last
 * of those events and returns, in milliseconds, the duration of the most recent
 * lookup-table kernel, plan kernels and partition kernel and the summed durations of the
 * dedup launches and of the scan launches (gather + ADC + top-k) of the most recent call;
 * a value is -1 if that kernel has not run since timing was enabled (with FANN_CHUNKS > 1
 * the partition kernels run on a second stream under the scans and are not timed).  Any
 * pointer may be NULL.
 */
int fann_set_timing(fann_index *ix, int enable);
int fann_last_timing(fann_index *ix, float *lut_ms, float *plan_ms, float *partition_ms, float *dedup_ms,
                     float *scan_ms);

#ifdef __cplusplus
}
#endif
#endif /* FANN_H */
