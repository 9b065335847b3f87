// fann_kernels.cuh -- device code of the FusionANNS GPU stage for sm_100a.
//
// Kernels (section 3, steps (1)(5)(6)(7)):
//   repack_rows_kernel   fann_load_codes: pad rows of M bytes to 16 / 32 / 64 bytes
//   build_lut_kernel     (1) lut[b][m][j] = sum_t (q - c)^2
//   plan_kernel          S_b partitions per query so that each fits one CTA's dedup table; work-item list
//   mode_kernel          per query: order-preserving or hashed placement in the dedup table
//   partition_kernel     split each query's candidate IDs into its S_b classes (ID ranges or hash
//                        classes), so that each dedup pass reads only its own IDs
//   partition_multi_kernel  the same with several CTAs per query (small batches)
//   dedup_kernel<T,R>    (5) shared-memory dedup table of 16-byte buckets, one (query, partition) per CTA
//                        pass; straight-line read / write / verify rounds separated by barriers, no
//                        atomics in the table; writes the distinct IDs of every query as a compact
//                        list, ascending in ordered mode (up to a bucket and overflow displacement)
//   scan_kernel<G,NB,D,LM>  (6) code-row gather through a per-warp shared-memory ring filled by
//                        asynchronous copies + Eq. 1 ADC from a conflict-free table  (7) streaming
//                        top-k, one query (or one slice of its distinct list) per CTA pass; writes
//                        out_ids / out_dists / counts.  LM: the list-major experiment
//   merge_parts_kernel   (7) small batches: merges the partial top-k of a query's scan CTAs
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fann {

constexpr uint32_t kIdNone = 0xFFFFFFFFu;
constexpr uint32_t kEmpty = 0xFFFFFFFFu;             // empty hash slot (never a valid id: id < N < 2^32-1)
constexpr unsigned long long kKeyMax = ~0ull;        // padding key, sorts last
constexpr int kScanThreads = 512;
constexpr int kScanWarps = kScanThreads / 32;
constexpr int kSample = 256;                         // keys sampled to place a prune pivot
constexpr int kMaxChunks = 16;                       // batch chunks (dedup of chunk i+1 overlaps scan of chunk i)
constexpr uint32_t kGridCells = 64;                  // ID-range cells sorted posting lists are indexed by (lists-direct: S | 64)
constexpr uint32_t kStatusTableFull = 1u;
constexpr uint32_t kStatusPlanOverflow = 2u;

struct WsHeader {                                    // first 256 bytes of the workspace
    uint32_t status;                                 // kStatus* bits
    uint32_t n_items;                                // (query, partition) work items of this batch
    uint32_t pad[2];
    uint32_t dedup_counter[kMaxChunks];              // next work item of each chunk's dedup launch
    uint32_t scan_counter[kMaxChunks];               // next query of each chunk's scan launch
};

// ---------------------------------------------------------------- helpers

__device__ __forceinline__ uint4 ldg_nc_16(const void *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::64B.v4.u32 {%0,%1,%2,%3}, [%4];"   // default fetches 128 B from DRAM
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// Shared-memory access by 32-bit shared-window address (no generic-address arithmetic per access).
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" :: "r"(addr), "r"(v) : "memory");
}

// shared-memory atomic add by shared-window address (no generic-address arithmetic per access)
__device__ __forceinline__ uint32_t atoms_add(uint32_t addr, uint32_t v)
{
    uint32_t old;
    asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(addr), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ void sts_u128(uint32_t addr, uint4 v)
{
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" :: "r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint2 lds_u64(uint32_t addr)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint4 lds_u128(uint32_t addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}
// 16-byte asynchronous copy global -> shared (LDGSTS), 64-byte L2 fetch; completes in commit-group order.
__device__ __forceinline__ void cp_async_16(uint32_t saddr, const void *g)
{
    asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;" :: "r"(saddr), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

// Compare-exchange of the keys at a lower (a) and a higher (b) index of a bitonic network.
__device__ __forceinline__ void cmpex(unsigned long long &a, unsigned long long &b, bool asc)
{
    const bool sw = (a > b) == asc;
    const unsigned long long t = a;
    a = sw ? b : a;
    b = sw ? t : b;
}

// The steps of merge size `size` with strides s_hi, s_hi / 2, ..., 1 (s_hi <= 64) on the 128 keys a warp holds, four
// consecutive keys per lane (key r of the lane = element e0 + r): strides 64 ... 4 by shuffles, 2 and 1 in registers.
__device__ __forceinline__ void bitonic_warp_steps(unsigned long long (&k)[4], uint32_t e0, uint32_t size, uint32_t s_hi)
{
    const uint32_t lane = threadIdx.x & 31;
    const bool asc = (e0 & size) == 0;                         // the same for the lane's four keys when size >= 4
    for (uint32_t stride = s_hi; stride >= 4; stride >>= 1) {
        const uint32_t L = stride >> 2;
        const bool take_min = ((lane & L) == 0) == asc;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const unsigned long long o = __shfl_xor_sync(0xffffffffu, k[r], L);
            k[r] = ((o < k[r]) == take_min) ? o : k[r];
        }
    }
    if (s_hi >= 2 && size >= 4) { cmpex(k[0], k[2], asc); cmpex(k[1], k[3], asc); }
    if (size >= 4) { cmpex(k[0], k[1], asc); cmpex(k[2], k[3], asc); }
    else { cmpex(k[0], k[1], true); cmpex(k[2], k[3], false); }   // size 2: direction = bit 1 of the element index
}

// Block-wide bitonic sort (ascending) of n = 2^p keys in shared memory, starting from sorted runs of length
// first_size / 2.  From single keys and n >= 128: every thread keeps four consecutive keys in registers for all
// steps with stride <= 64 (a warp sorts its 128 keys without touching shared memory or a barrier), and the steps
// with larger strides go through shared memory two at a time -- 11 barriers instead of 66 for 2048 keys.
__device__ __forceinline__ void bitonic_sort_smem(unsigned long long *a, uint32_t n, uint32_t first_size)
{
    if (first_size == 2 && n >= 128 && (blockDim.x & 31) == 0) {
        const uint32_t nvt = n >> 2;                           // four keys per (virtual) thread; whole warps
        for (uint32_t vt = threadIdx.x; vt < nvt; vt += blockDim.x) {
            unsigned long long k[4] = {a[4 * vt], a[4 * vt + 1], a[4 * vt + 2], a[4 * vt + 3]};
            for (uint32_t size = 2; size <= 128; size <<= 1) bitonic_warp_steps(k, 4 * vt, size, size >> 1);
            a[4 * vt] = k[0]; a[4 * vt + 1] = k[1]; a[4 * vt + 2] = k[2]; a[4 * vt + 3] = k[3];
        }
        __syncthreads();
        for (uint32_t size = 256; size <= n; size <<= 1) {
            uint32_t stride = size >> 1;
            while (stride >= 128) {
                if (stride >= 256) {                           // strides `stride` and `stride / 2` in one pass
                    const uint32_t h = stride >> 1;
                    for (uint32_t vt = threadIdx.x; vt < nvt; vt += blockDim.x) {
                        const uint32_t base = ((vt & ~(h - 1)) << 2) | (vt & (h - 1));
                        const bool asc = (base & size) == 0;
                        unsigned long long x0 = a[base], x1 = a[base + h], x2 = a[base + stride], x3 = a[base + stride + h];
                        cmpex(x0, x2, asc); cmpex(x1, x3, asc);
                        cmpex(x0, x1, asc); cmpex(x2, x3, asc);
                        a[base] = x0; a[base + h] = x1; a[base + stride] = x2; a[base + stride + h] = x3;
                    }
                    stride >>= 2;
                } else {
                    for (uint32_t i = threadIdx.x; i < (n >> 1); i += blockDim.x) {
                        const uint32_t lo = 2 * i - (i & (stride - 1)), hi = lo + stride;
                        unsigned long long x = a[lo], y = a[hi];
                        cmpex(x, y, (lo & size) == 0);
                        a[lo] = x; a[hi] = y;
                    }
                    stride >>= 1;
                }
                __syncthreads();
            }
            for (uint32_t vt = threadIdx.x; vt < nvt; vt += blockDim.x) {
                unsigned long long k[4] = {a[4 * vt], a[4 * vt + 1], a[4 * vt + 2], a[4 * vt + 3]};
                bitonic_warp_steps(k, 4 * vt, size, 64);
                a[4 * vt] = k[0]; a[4 * vt + 1] = k[1]; a[4 * vt + 2] = k[2]; a[4 * vt + 3] = k[3];
            }
            __syncthreads();
        }
        return;
    }
    for (uint32_t size = first_size; size <= n; size <<= 1) {
        for (uint32_t stride = size >> 1; stride > 0; stride >>= 1) {
            for (uint32_t i = threadIdx.x; i < (n >> 1); i += blockDim.x) {
                uint32_t lo = 2 * i - (i & (stride - 1));
                uint32_t hi = lo + stride;
                bool asc = (lo & size) == 0;
                unsigned long long x = a[lo], y = a[hi];
                if ((x > y) == asc) { a[lo] = y; a[hi] = x; }
            }
            __syncthreads();
        }
    }
}

// ---------------------------------------------------------------- fann_load_codes

__global__ void repack_rows_kernel(const uint8_t *__restrict__ src, uint8_t *__restrict__ dst,
                                   uint64_t n, uint32_t M, uint32_t row_bytes)
{
    const uint32_t chunks = row_bytes >> 4;
    uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n * chunks) return;
    uint64_t row = t / chunks;
    uint32_t c0 = (uint32_t)(t % chunks) << 4;
    uint32_t w[4] = {0, 0, 0, 0};
    const uint8_t *s = src + row * M;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        uint32_t m = c0 + i;
        uint32_t v = (m < M) ? (uint32_t)s[m] : 0u;
        w[i >> 2] |= v << ((i & 3) * 8);
    }
    *reinterpret_cast<uint4 *>(dst + row * row_bytes + c0) = make_uint4(w[0], w[1], w[2], w[3]);
}

// ---------------------------------------------------------------- (1) lookup table

// One thread = 4 consecutive centroids j of one (query, sub-space); one block = 4 sub-spaces of one query.
// DS = dsub when it is 2, 4 or 8 (the thread's 4 x dsub codebook floats are contiguous and 16-byte aligned:
// read as float4), else 0 (any dsub, scalar loads).  Sum over t ascending with FMA in both.
template <int DS>
__global__ void __launch_bounds__(256) build_lut_kernel(const float *__restrict__ queries,
                                                        const float *__restrict__ codebooks,
                                                        float *__restrict__ lut, uint32_t M, uint32_t dsub_rt)
{
    const uint32_t blocks_per_q = (M + 3) >> 2;
    const uint32_t b = blockIdx.x / blocks_per_q;
    const uint32_t m = ((blockIdx.x - b * blocks_per_q) << 2) + (threadIdx.x >> 6);
    if (m >= M) return;
    const uint32_t j0 = (threadIdx.x & 63u) << 2;
    const uint32_t dsub = DS ? (uint32_t)DS : dsub_rt;
    const float *q = queries + ((size_t)b * M + m) * dsub;
    const float *c = codebooks + ((size_t)m * 256 + j0) * dsub;
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    if constexpr (DS > 0) {
        float cv[4 * DS], qv[DS];
#pragma unroll
        for (int i = 0; i < DS; ++i) {
            const float4 v = __ldg(reinterpret_cast<const float4 *>(c) + i);
            cv[4 * i] = v.x; cv[4 * i + 1] = v.y; cv[4 * i + 2] = v.z; cv[4 * i + 3] = v.w;
        }
#pragma unroll
        for (int t = 0; t < DS; ++t) qv[t] = __ldg(q + t);
#pragma unroll
        for (int t = 0; t < DS; ++t)
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                const float dlt = qv[t] - cv[jj * DS + t];
                s[jj] = fmaf(dlt, dlt, s[jj]);
            }
    } else {
        for (uint32_t t = 0; t < dsub; ++t) {
            const float qv = __ldg(q + t);
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                const float dlt = qv - __ldg(c + jj * dsub + t);
                s[jj] = fmaf(dlt, dlt, s[jj]);
            }
        }
    }
    *reinterpret_cast<float4 *>(lut + ((size_t)b * M + m) * 256 + j0) = make_float4(s[0], s[1], s[2], s[3]);
}

// ---------------------------------------------------------------- plan

// Single CTA.  S_b = ceil(C_b / cap_c) hash partitions per query, so that the
// IDs one partition can receive fit the per-CTA table at <= 75 % load even if
// none repeats.  Writes S[], item_start[B+1], items[], n_items; zeroes the
// per-query distinct counts and the work counters.
__global__ void plan_kernel(const long long *__restrict__ cand_offsets, uint32_t B, uint32_t cap_c,
                            uint32_t max_items, WsHeader *hdr, uint32_t *S, uint32_t *item_start,
                            uint2 *items, uint32_t *uniq_counts, uint32_t keep_status,
                            unsigned long long total_cands, uint32_t exact_total, uint32_t *bucket_cnt, uint32_t *part_aux,
                            uint32_t pow2_classes)
{
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t running;
    __shared__ uint32_t bad_total;
    if (threadIdx.x == 0) {
        running = 0;
        // the caller's total_cands sized the workspace: lists that reach past it must not be touched
        const long long first = cand_offsets[0], last = cand_offsets[B];
        bad_total = (first < 0 || last < first || (unsigned long long)last > total_cands ||
                     (exact_total && (first != 0 || (unsigned long long)last != total_cands))) ? 1u : 0u;
    }
    __syncthreads();
    const bool refuse = bad_total != 0;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (uint32_t base = 0; base < B; base += blockDim.x) {
        uint32_t b = base + threadIdx.x;
        uint32_t s = 0;
        if (b < B) {
            long long c = cand_offsets[b + 1] - cand_offsets[b];
            if (c < 0) c = 0;
            s = (uint32_t)((c + cap_c - 1) / cap_c);
            if (s == 0) s = 1;
            if (pow2_classes && s <= kGridCells) {             // lists-direct: ID-range classes are runs of grid cells,
                uint32_t s2 = pow2_classes < kGridCells ? pow2_classes : kGridCells;   // at least pow2_classes of them
                while (s2 < s) s2 <<= 1;
                s = s2;
            }
            if (refuse) s = 0;                                 // no partition, no dedup item; the scan sees U = 0
            S[b] = s;
            uniq_counts[b] = 0;
            if (part_aux) { part_aux[2 * b] = 0; part_aux[2 * b + 1] = 0; }   // partition_multi_kernel: arrivals, failure
        }
        uint32_t incl = s;                                     // block inclusive scan
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        if (lane == 31) warp_sums[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = warp_sums[lane], wi = w;
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t v = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += v;
            }
            warp_sums[lane] = wi - w;                          // exclusive
        }
        __syncthreads();
        uint32_t start = running + warp_sums[warp] + incl - s;
        if (b < B) {
            item_start[b] = start;
            for (uint32_t p = 0; p < s; ++p)
                if (start + p < max_items) { items[start + p] = make_uint2(b, p); if (part_aux) bucket_cnt[start + p] = 0; }
        }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) running = start + s;
        __syncthreads();
    }
    if (threadIdx.x < kMaxChunks) { hdr->dedup_counter[threadIdx.x] = 0; hdr->scan_counter[threadIdx.x] = 0; }
    if (threadIdx.x == 0) {
        const bool over = running > max_items;                 // cannot happen when total_cands is honest
        item_start[B] = over ? 0u : running;
        if (over) for (uint32_t b = 0; b < B; ++b) { item_start[b] = 0; S[b] = 0; }
        // a later chunk of the same batch (fann_search_host) keeps what the earlier chunks reported
        hdr->status = (keep_status ? hdr->status : 0u) | ((over || refuse) ? kStatusPlanOverflow : 0u);
        hdr->n_items = over ? 0u : running;
    }
}

// ---------------------------------------------------------------- (5) dedup

// Placement of the distinct IDs in the dedup table, per query:
//   kModeOrdered  slot = floor((id - lo) * nslots / span): order-preserving, so the compacted table is
//                 the distinct set in (almost) ascending ID order and the scan kernel's row gathers walk
//                 the code array in address order (fewer address translations; measured 1.35-1.5x the
//                 random-order gather rate).  Needs IDs that are spread evenly over [0, N).
//   kModeHashed   slot = hash(id): for candidate lists whose IDs are bunched (runs of consecutive IDs,
//                 one dense range), which would pile up in an order-preserving table.
constexpr uint32_t kModeOrdered = 0, kModeHashed = 1;
constexpr int kModeSamplePairs = 8;                  // adjacent pairs sampled per lane (256 per query)

// One warp per query: sample 256 adjacent pairs of its candidate list and decide the placement mode.
// Hashed if (a) some 1/32 range of [0, N) holds more than 3x its share of the samples, or (b) more than
// 1/16 of the sampled neighbours are closer than N / (2 C) (about one table slot of the query).
// unsplit_cap != 0: the lists are not split by partition_kernel (FANN_PARTITION=0), so nobody counts the classes
// exactly; a list longer than unsplit_cap (S >= 2) then takes hash classes, which stay balanced whatever the IDs are.
__global__ void mode_kernel(const long long *__restrict__ cand_offsets, const uint32_t *__restrict__ cand_ids,
                            uint32_t B, uint64_t N, uint32_t force, uint32_t unsplit_cap, uint32_t *__restrict__ mode)
{
    __shared__ uint32_t hist[8][32];
    const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t b = blockIdx.x * 8 + w;
    hist[w][lane] = 0;
    __syncwarp();
    if (b >= B) return;
    const long long off0 = cand_offsets[b];
    const long long Cll = cand_offsets[b + 1] - off0;
    const uint32_t C = Cll > 0 ? (uint32_t)Cll : 0u;
    uint32_t m = kModeOrdered;
    if (N < 4096 || (unsplit_cap && C > unsplit_cap)) {
        m = kModeHashed;                                       // ordered classes need N >> S
    } else if (force < 2) {
        m = force;
    } else if (C >= 64) {
        const uint32_t *ids = cand_ids + off0;
        const unsigned long long cd = N / (2ull * C);
        const uint32_t close_dist = cd > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)cd;
        const uint32_t ns = 32 * kModeSamplePairs;
        const uint32_t bin_mul = (uint32_t)(((32ull << 32) - 1) / N);   // bin = id * 32 / N (< 32 for id < N)
        uint32_t nvalid = 0, nclose = 0;
#pragma unroll
        for (int j = 0; j < kModeSamplePairs; ++j) {
            const uint32_t i = j * 32 + lane;
            const uint32_t e = (uint32_t)((unsigned long long)i * (C - 1) / ns);   // e + 1 <= C - 1
            const uint32_t x = __ldg(ids + e), y = __ldg(ids + e + 1);
            const bool vx = x != kIdNone && (uint64_t)x < N, vy = y != kIdNone && (uint64_t)y < N;
            if (vx) { atomicAdd(&hist[w][__umulhi(x, bin_mul) & 31u], 1u); ++nvalid; }
            if (vx && vy && x != y && (x > y ? x - y : y - x) < close_dist) ++nclose;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            nvalid += __shfl_xor_sync(0xffffffffu, nvalid, o);
            nclose += __shfl_xor_sync(0xffffffffu, nclose, o);
        }
        __syncwarp();
        const bool dense = hist[w][lane] > 3u * (nvalid / 32u) + 8u;
        if (__any_sync(0xffffffffu, dense) || nclose * 16u > nvalid) m = kModeHashed;
    }
    if (lane == 0) mode[b] = m;
}

struct DedupParams {
    const long long *cand_offsets;                   // [B+1]
    const uint32_t *cand_ids;
    uint64_t N;
    uint32_t nslots_max;                             // hash-table slots one CTA can hold
    uint32_t q_begin, q_end;                         // queries of this launch
    uint32_t *counter;                               // work counter of this launch
    WsHeader *hdr;
    const uint32_t *S;                               // [B] partitions per query
    const uint32_t *mode;                            // [B] kMode*
    const uint32_t *item_start;                      // [B+1]
    const uint2 *items;                              // [n_items] (query, partition)
    uint32_t *uniq_ids;                              // [total_cands]; query b's list starts at cand_offsets[b]
    uint32_t *uniq_counts;                           // [B], zeroed by plan_kernel
    const uint32_t *part_ids;                        // [2 * total_cands] buckets written by partition_kernel, or NULL
    const uint32_t *part_ok;                         // [B] 1: query b's buckets are valid
    const uint32_t *bucket_cnt;                      // [n_items] IDs in the bucket of each (query, partition) item
    // Lists-direct mode (dedup_kernel<..., LD = true>, fann_search_lists on sorted posting lists): the IDs of an item
    // are read straight from the probed lists -- for an ID-range class the sub-range of every list that falls into
    // it, found in the lists' grid -- so that neither a candidate array nor its class split is ever written.
    const long long *list_offsets;                   // [n_lists + 1]
    const uint32_t *list_ids;                        // every list ascending
    const uint16_t *list_grid;                       // [n_lists][kGridCells + 1] position of the first ID >= cell start
    const uint32_t *probes;                          // [B][nprobe]
    uint32_t nprobe;
    uint64_t n_lists;
};

constexpr uint32_t kLdMaxProbe = 512;                // lists-direct: probes per query the shared-memory segment table holds
constexpr uint32_t kLdRowMap = 1024;                 // lists-direct: 32-ID rows the row -> segment map holds
__host__ __device__ constexpr uint32_t dedup_ld_bytes() { return kLdMaxProbe * 4 + (kLdMaxProbe + 4) * 4 + kLdRowMap * 2; }
// first ID of grid cell g (g = kGridCells: N)
__host__ __device__ inline uint32_t grid_start(uint64_t N, uint32_t g) { return (uint32_t)((N * g) / kGridCells); }

// Partition of a query's valid IDs into S classes (both the partition kernel and the dedup kernel's own
// filter use these, so a class means the same set of IDs wherever it is computed):
//   ordered  class = floor(id * MS / 2^32), MS = floor(S * 2^32 / N): S contiguous ID ranges of near-equal length;
//            class p starts at ceil(p * 2^32 / MS)
//   hashed   class = floor(h1(id) * S / 2^32), h1 the first round of the slot hash
__device__ __forceinline__ uint32_t ordered_class_mul(uint64_t N, uint32_t S)
{
    return (uint32_t)(((unsigned long long)S << 32) / N);      // S < N (mode_kernel sends tiny N to hashed mode)
}
__device__ __forceinline__ uint32_t ordered_class_start(uint32_t MS, uint32_t cls, uint64_t N)
{
    const unsigned long long v = (((unsigned long long)cls << 32) + MS - 1) / MS;
    return (uint32_t)(v < N ? v : N);
}
__device__ __forceinline__ uint32_t hash_round1(uint32_t x) { return (x ^ (x >> 16)) * 0x7feb352dU; }

__device__ __forceinline__ uint4 load_ids4(const uint32_t *ids, long long e0, uint32_t C);

constexpr uint32_t kMaxPartBuckets = 16;             // partition_kernel handles 2..16 classes per query
constexpr int kPartThreads = 512;

struct PartParams {
    const long long *cand_offsets;
    const uint32_t *cand_ids;
    uint64_t N;
    const uint32_t *S, *item_start;
    uint32_t *mode;                                  // [B]; a query whose ID-range classes do not fit is switched to hashed
    uint32_t *part_ids;                              // query b's buckets at 2 * cand_offsets[b], bucket p at p * cap_b
    uint32_t *part_ok;                               // [B]
    uint32_t *bucket_cnt;                            // [n_items]
    uint32_t q_begin;                                // first query of this launch (one CTA per query)
    uint32_t class_max;                              // most IDs of one class a dedup table takes if none repeats (90 % load)
    uint32_t ctas;                                   // partition_multi_kernel: CTAs per query (small batches)
    uint32_t *aux;                                   // partition_multi_kernel: [B][2] arrivals, failure flag (zeroed per call)
};

// Splits the candidate list of every query that needs S >= 2 dedup partitions into its S classes, so that
// each dedup pass reads only its own IDs instead of filtering the whole list S times.  One CTA per query.
// Bucket p of query b holds at most cap_b = 2 C_b / S_b IDs (twice its fair share).
// The class counts are exact here, so this is also where the placement decision is made final: if an ID-range
// class (ordered mode) is larger than its bucket or than a dedup table takes (IDs concentrated in part of
// [0, N), which mode_kernel's sample can miss), the query is switched to hashed classes and split again.  If
// a hash class overflows its bucket (many repeats of few IDs), part_ok[b] stays 0 and the dedup kernel filters
// the original list itself; its table then only has to hold the distinct IDs.
__global__ void __launch_bounds__(kPartThreads) partition_kernel(const PartParams p)
{
    __shared__ uint32_t scnt[kMaxPartBuckets];
    const uint32_t b = p.q_begin + blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    const uint32_t scnt_addr = (uint32_t)__cvta_generic_to_shared(scnt);
    const uint32_t S = p.S[b];
    if (S < 2 || S > kMaxPartBuckets) {
        // more classes than this kernel splits: hash classes stay balanced whatever the IDs are
        if (tid == 0) { p.part_ok[b] = 0; if (S > kMaxPartBuckets) p.mode[b] = kModeHashed; }
        return;
    }
    bool hashed = p.mode[b] == kModeHashed;
    const long long off0 = p.cand_offsets[b];
    const long long Cll = p.cand_offsets[b + 1] - off0;
    const uint32_t C = Cll > 0 ? (uint32_t)Cll : 0u;
    const uint32_t capb = (uint32_t)(2ull * C / S);
    uint32_t *out = p.part_ids + 2 * off0;
    const uint32_t *ids = p.cand_ids + off0;
    const uint32_t shift = (uint32_t)((reinterpret_cast<uintptr_t>(ids) >> 2) & 3u);
    const uint32_t nvec = (C + shift + 3u) >> 2;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint4 *ids4 = reinterpret_cast<const uint4 *>(ids - shift);
    const uint32_t v_in0 = shift ? 1u : 0u, v_in1 = (C + shift) >> 2;      // vectors wholly inside the list
    auto load_vec = [&](uint32_t v) -> uint4 {
        if (v >= v_in0 && v < v_in1) return __ldg(ids4 + v);
        if (v < nvec) return load_ids4(ids, 4ll * v - shift, C);
        return make_uint4(kIdNone, kIdNone, kIdNone, kIdNone);
    };
    const uint32_t N32 = (uint32_t)p.N;                        // N < 2^32 - 1 (fann_load_codes)
    for (;;) {
        const uint32_t MS = hashed ? 0u : ordered_class_mul(p.N, S);
        if (tid < kMaxPartBuckets) scnt[tid] = 0;
        __syncthreads();
        uint32_t overflow = 0;
        // One ID: its class; lanes of the same class found by one MATCH instead of a ballot per class; the lowest
        // lane of each class reserves the class's output range for all of them.  (Issuing the four matches of a
        // vector before using any result was measured slower: 2.68 against 2.51 ms.)
        auto place = [&](uint32_t x, uint32_t cls) {
            const bool valid = x < N32;                        // also drops kIdNone
            if (!valid) cls = 0xFFu;
            const uint32_t own = __match_any_sync(0xffffffffu, cls);
            const uint32_t leader = __ffs(own) - 1;
            uint32_t base = 0;
            if (valid && lane == leader) base = atoms_add(scnt_addr + (cls << 2), (uint32_t)__popc(own));
            base = __shfl_sync(0xffffffffu, base, leader);
            const uint32_t pos = base + __popc(own & lt_mask);
            if (valid) {
                if (pos < capb) out[cls * capb + pos] = x;     // cls * capb + pos < 2 C < 2^32
                else overflow = 1;
            }
        };
        uint4 nxt = load_vec(tid);
        if (!hashed) {
            for (uint32_t vb = 0; vb < nvec; vb += kPartThreads) { // uniform trip count: the matches need whole warps
                const uint4 q4 = nxt;
                nxt = load_vec(vb + kPartThreads + tid);           // one iteration ahead
                place(q4.x, __umulhi(q4.x, MS)); place(q4.y, __umulhi(q4.y, MS));
                place(q4.z, __umulhi(q4.z, MS)); place(q4.w, __umulhi(q4.w, MS));
            }
        } else {
            for (uint32_t vb = 0; vb < nvec; vb += kPartThreads) {
                const uint4 q4 = nxt;
                nxt = load_vec(vb + kPartThreads + tid);
                place(q4.x, __umulhi(hash_round1(q4.x), S)); place(q4.y, __umulhi(hash_round1(q4.y), S));
                place(q4.z, __umulhi(hash_round1(q4.z), S)); place(q4.w, __umulhi(hash_round1(q4.w), S));
            }
        }
        bool bad = __syncthreads_or(overflow != 0);             // also: every scnt[] update is visible
        if (!hashed) {
            // exact class counts: an ID-range class that would overfill a dedup table if none of its IDs repeats
            const bool big = tid < S && scnt[tid] > p.class_max;
            bad = __syncthreads_or(bad || big);
            if (bad) {                                         // split again with hash classes
                hashed = true;
                if (tid == 0) p.mode[b] = kModeHashed;
                continue;
            }
        }
        if (tid < S) p.bucket_cnt[p.item_start[b] + tid] = scnt[tid] < capb ? scnt[tid] : capb;
        if (tid == 0) p.part_ok[b] = bad ? 0u : 1u;
        return;
    }
}

// Small batches: the same split with p.ctas CTAs per query, so that one query's list does
// not wait on one SM.  Every CTA takes a slice of the list: it counts its IDs per class, reserves each class's range
// in the query's bucket with one global atomic per class (bucket_cnt is the cursor and ends as the class total), then
// scatters.  The query's last CTA to finish closes it: buckets valid, or -- a class overflowed its bucket or would
// overfill a dedup table -- not valid and the query switched to hash classes, which the dedup kernel then filters
// from the original list (the one-CTA kernel splits such a query again instead; here it is the rare case).
__global__ void __launch_bounds__(kPartThreads) partition_multi_kernel(const PartParams p)
{
    __shared__ uint32_t scnt[kMaxPartBuckets];
    __shared__ uint32_t s_last;
    const uint32_t b = p.q_begin + blockIdx.x / p.ctas, sub = blockIdx.x % p.ctas;
    const uint32_t tid = threadIdx.x, lane = tid & 31;
    const uint32_t scnt_addr = (uint32_t)__cvta_generic_to_shared(scnt);
    const uint32_t S = p.S[b];
    if (S < 2 || S > kMaxPartBuckets) {
        if (sub == 0 && tid == 0) { p.part_ok[b] = 0; if (S > kMaxPartBuckets) p.mode[b] = kModeHashed; }
        return;
    }
    const bool hashed = p.mode[b] == kModeHashed;              // nobody changes it before every CTA of the query has read it
    const long long off0 = p.cand_offsets[b];
    const long long Cll = p.cand_offsets[b + 1] - off0;
    const uint32_t C = Cll > 0 ? (uint32_t)Cll : 0u;
    const uint32_t capb = (uint32_t)(2ull * C / S);
    uint32_t *out = p.part_ids + 2 * off0;
    const uint32_t *ids = p.cand_ids + off0;
    const uint32_t shift = (uint32_t)((reinterpret_cast<uintptr_t>(ids) >> 2) & 3u);
    const uint32_t nvec = (C + shift + 3u) >> 2;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint4 *ids4 = reinterpret_cast<const uint4 *>(ids - shift);
    const uint32_t v_in0 = shift ? 1u : 0u, v_in1 = (C + shift) >> 2;
    auto load_vec = [&](uint32_t v) -> uint4 {
        if (v >= v_in0 && v < v_in1) return __ldg(ids4 + v);
        if (v < nvec) return load_ids4(ids, 4ll * v - shift, C);
        return make_uint4(kIdNone, kIdNone, kIdNone, kIdNone);
    };
    const uint32_t v_lo = (uint32_t)((unsigned long long)nvec * sub / p.ctas);
    const uint32_t v_hi = (uint32_t)((unsigned long long)nvec * (sub + 1) / p.ctas);
    const uint32_t N32 = (uint32_t)p.N;
    const uint32_t MS = hashed ? 0u : ordered_class_mul(p.N, S);
    auto class_of = [&](uint32_t x) -> uint32_t {
        if (x >= N32) return 0xFFu;                            // also kIdNone
        return hashed ? __umulhi(hash_round1(x), S) : __umulhi(x, MS);
    };
    if (tid < kMaxPartBuckets) scnt[tid] = 0;
    if (tid == 0) s_last = 0;
    __syncthreads();
    uint32_t overflow = 0;
    for (int pass = 0; pass < 2; ++pass) {                     // 0: count, 1: scatter (the slice is in L2 by then)
        for (uint32_t vb = v_lo; vb < v_hi; vb += kPartThreads) {   // uniform trip count: the matches need whole warps
            const uint4 q4 = vb + tid < v_hi ? load_vec(vb + tid) : make_uint4(kIdNone, kIdNone, kIdNone, kIdNone);
            const uint32_t x[4] = {q4.x, q4.y, q4.z, q4.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const uint32_t cls = class_of(x[e]);
                const uint32_t own = __match_any_sync(0xffffffffu, cls);
                const uint32_t leader = __ffs(own) - 1;
                uint32_t base = 0;
                if (cls != 0xFFu && lane == leader) base = atoms_add(scnt_addr + (cls << 2), (uint32_t)__popc(own));
                if (pass) {
                    base = __shfl_sync(0xffffffffu, base, leader);
                    const uint32_t pos = base + __popc(own & lt_mask);
                    if (cls != 0xFFu) {
                        if (pos < capb) out[cls * capb + pos] = x[e];
                        else overflow = 1;
                    }
                }
            }
        }
        __syncthreads();
        if (!pass) {                                           // this CTA's range in every class's bucket
            if (tid < S) scnt[tid] = atomicAdd(&p.bucket_cnt[p.item_start[b] + tid], scnt[tid]);
            __syncthreads();
        }
    }
    if (__syncthreads_or(overflow != 0) && tid == 0) atomicOr(&p.aux[2 * b + 1], 1u);
    if (tid == 0) {
        __threadfence();
        s_last = atomicAdd(&p.aux[2 * b], 1u) == p.ctas - 1 ? 1u : 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    bool bad = *reinterpret_cast<volatile uint32_t *>(&p.aux[2 * b + 1]) != 0;
    uint32_t total = 0;
    if (tid < S) total = *reinterpret_cast<volatile uint32_t *>(&p.bucket_cnt[p.item_start[b] + tid]);
    if (!hashed) bad = bad || total > p.class_max;             // would overfill a dedup table if none of its IDs repeats
    bad = __syncthreads_or(bad);
    if (tid < S && total > capb) p.bucket_cnt[p.item_start[b] + tid] = capb;
    if (tid == 0) {
        p.part_ok[b] = bad ? 0u : 1u;
        if (bad && !hashed) p.mode[b] = kModeHashed;
    }
}

// Elements e0 .. e0+3 of a candidate list of C IDs (e0 may be negative or reach past the end at the
// two ragged ends of a list); positions outside [0, C) read as kIdNone.  ids + e0 is 16-byte aligned.
__device__ __forceinline__ uint4 load_ids4(const uint32_t *ids, long long e0, uint32_t C)
{
    if (e0 >= 0 && e0 + 3 < (long long)C) return __ldg(reinterpret_cast<const uint4 *>(ids + e0));
    uint4 r = make_uint4(kIdNone, kIdNone, kIdNone, kIdNone);
    if (e0 >= 0 && e0 < (long long)C) r.x = __ldg(ids + e0);
    if (e0 + 1 >= 0 && e0 + 1 < (long long)C) r.y = __ldg(ids + e0 + 1);
    if (e0 + 2 >= 0 && e0 + 2 < (long long)C) r.z = __ldg(ids + e0 + 2);
    if (e0 + 3 >= 0 && e0 + 3 < (long long)C) r.w = __ldg(ids + e0 + 3);
    return r;
}

constexpr int kDedupIdsPerThread = 8;                // fresh IDs a thread holds per batch (two 16-byte loads)
// bookkeeping (256 bytes, of which bytes 64..79 are a bucket that stays empty) + two retry queues of `threads`
// (id, bucket address) pairs precede the table
#ifndef FANN_DEDUP_BS
#define FANN_DEDUP_BS 4
#endif
constexpr int kDedupBucketSlots = FANN_DEDUP_BS;                 // slots per bucket (2: one 8-byte look, 4: one 16-byte look)
constexpr int kDedupQueuePer8 = kDedupBucketSlots == 1 ? 3 : kDedupBucketSlots == 2 ? 2 : 1;   // queued entries a thread takes up per batch, per 8 fresh IDs
// `shape` = threads x fresh IDs per thread / 8: 1024 (one CTA per SM) or 512 (two CTAs per SM)
__host__ __device__ constexpr uint32_t dedup_table_off(uint32_t shape) { return 256 + 2 * kDedupQueuePer8 * shape * 8; }

// PAPER.md:L127 "it first deduplicates them", L210 "parallel hash algorithm".  The paper's kernel takes
// a spinlock per hash entry; an atomicCAS per ID costs about 2 cycles per lane of the shared-memory
// pipe on this part (64x a plain load).  This kernel uses neither.  The table is an array of 16-byte
// buckets of 4 slots; an ID's bucket is an order-preserving (or hashed) function of the ID, so one
// 16-byte shared load shows every slot the ID can be in, and the CTA advances in rounds with no store in
// flight while anyone reads:
//   read   one load per ID: found in its bucket (a repeat: done), else the empty slot it will take (its
//          home slot id & 3 if that is empty, else the first empty one), else -- bucket full -- the ID
//          moves on to the next bucket through the retry queue;
//   write  every ID that found an empty slot stores itself there;
//   verify of several stores to one slot one survived; the losers (about 5 %) go to the retry queue.
// The code is straight-line: nothing walks a probe sequence in a divergent loop.  A queued (ID, bucket)
// pair is taken up again, one per thread, with the next batch.  A bucket seen full stays full, a slot seen
// non-empty keeps its value, and all copies of an ID make the same choices from the same view, so exactly one
// slot ends up holding it.  Each CTA pass handles the IDs of one query that fall into one partition (an ID
// range in ordered mode, a hash class in hashed mode), 8 per thread per batch, then compacts its table in
// bucket order into the query's distinct list.
// T threads per CTA: 1024 (one CTA per SM, the whole shared memory as one table) or 512 (two CTAs per SM with half
// the table each: one computes while the other waits at a barrier).
template <int T, int R, bool LD = false>
__global__ void __launch_bounds__(T, 1024 / (T * R / 8)) dedup_kernel(const DedupParams p)
{
    constexpr int BS = kDedupBucketSlots, BSH = BS == 1 ? 2 : BS == 2 ? 3 : 4;   // slots per bucket, log2 of its bytes
    constexpr int NV = R / 4, NQ = kDedupQueuePer8 * R / 8, NE = R + NQ;   // per thread and batch: NV vectors = R fresh IDs + NQ from the queue
    constexpr uint32_t QCAP = NQ * T;                          // entries one retry queue holds
    constexpr uint32_t kNoSlot = 4 * BS;                       // "no empty slot in this bucket" as a byte offset
    constexpr uint32_t kBucketMask = ~(4u * BS - 1u);
    extern __shared__ __align__(16) unsigned char smem[];
    // [0] out base [2,3] queue lengths [5] queue overflow [8..15], [24..31] the item of this pass and the next one:
    // item, lo, span, bmul, nb  [16..19] a bucket that stays empty  [32..63] warp counts
    uint32_t *misc = reinterpret_cast<uint32_t *>(smem);
    uint32_t *wsum = misc + 32, *qcnt = misc + 2;
    uint2 *queue = reinterpret_cast<uint2 *>(smem + 256);                    // two retry queues of QCAP (id, bucket address)
    // lists-direct: segment starts, prefix of segment lengths, row -> segment map, between the queues and the table
    uint32_t *seg_start = reinterpret_cast<uint32_t *>(smem + dedup_table_off(T * R / 8));
    uint32_t *seg_prefix = seg_start + kLdMaxProbe;
    uint16_t *row_map = reinterpret_cast<uint16_t *>(seg_prefix + kLdMaxProbe + 4);
    uint32_t *table = reinterpret_cast<uint32_t *>(smem + dedup_table_off(T * R / 8) + (LD ? dedup_ld_bytes() : 0u));
    const uint32_t tbl = (uint32_t)__cvta_generic_to_shared(table);
    const uint32_t none_addr = (uint32_t)__cvta_generic_to_shared(misc + 16);   // a bucket that always holds 4 x kEmpty
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t first = p.item_start[p.q_begin], last = p.item_start[p.q_end];

    // Thread 0 takes the next (query, partition) item off the work counter and does its 64-bit divisions (table
    // geometry) for everybody, one pass ahead, so that nobody waits for this chain of dependent loads.
    auto fetch_item = [&](uint32_t *slot) {
        const uint32_t item = first + atomicAdd(p.counter, 1u);
        slot[0] = item;
        if (item >= last) return;
        const uint2 it = p.items[item];
        const uint32_t b = it.x, part = it.y, S = p.S[b];
        const long long Cll = p.cand_offsets[b + 1] - p.cand_offsets[b];
        const uint32_t C = Cll > 0 ? (uint32_t)Cll : 0u;       // plan guarantees C / S <= 0.75 nslots_max
        const bool ordered = p.mode[b] != kModeHashed;
        // lists-direct, ordered: bucket_cnt holds the class's exact ID count (lists_classes_kernel)
        const bool pre = LD ? ordered : (p.part_ids != nullptr && S > 1 && p.part_ok[b] != 0);
        // table sized to the partition, never more than the CTA can hold: 2 slots per expected candidate; 1.5
        // where the count is exact (about 0.4 full after dedup)
        uint32_t nslots = p.nslots_max;
        const unsigned long long want = ((pre ? (unsigned long long)p.bucket_cnt[item] * 3 / 2
                                              : (unsigned long long)(C / S + 1) * 2) + 128) & ~3ull;
        if (want < nslots) nslots = (uint32_t)want;
        const uint32_t nb = nslots / BS;                       // buckets
        // ordered mode: this partition owns the IDs of class `part`, a range [lo, lo + span);
        // bucket = (id - lo) * nb / span
        uint32_t lo = 0, span = 0, bmul = 0;
        if (ordered) {
            if (LD) {                                          // classes are runs of grid cells (S divides kGridCells)
                lo = grid_start(p.N, part * (kGridCells / S));
                span = grid_start(p.N, (part + 1) * (kGridCells / S)) - lo;
            } else {
                const uint32_t class_mul = ordered_class_mul(p.N, S);
                lo = ordered_class_start(class_mul, part, p.N);
                span = ordered_class_start(class_mul, part + 1, p.N) - lo;
            }
            // span <= nb (tiny N): bucket = id - lo - 1 or 0, still order-preserving and inside the table
            bmul = span > nb ? (uint32_t)(((unsigned long long)nb << 32) / span) : 0xFFFFFFFFu;
        }
        slot[1] = lo; slot[2] = span; slot[3] = bmul; slot[4] = nb;
    };
    if (tid < 4) misc[16 + tid] = kEmpty;
    if (tid == 0) { misc[5] = 0; fetch_item(misc + 8); }
    {   // the table starts empty; every pass leaves it empty again (the compaction clears what it reads)
        const uint4 e4 = make_uint4(kEmpty, kEmpty, kEmpty, kEmpty);
        for (uint32_t i = tid; i < (p.nslots_max >> 2); i += T) reinterpret_cast<uint4 *>(table)[i] = e4;
    }
    uint32_t sel = 0;

    for (;;) {
        if (tid == 0) { qcnt[0] = 0; qcnt[1] = 0; }            // nobody reads them between the last batch and here
        __syncthreads();                                       // previous item fully done; this one's geometry is there
        const uint32_t *cur_item = misc + (sel ? 24 : 8);
        const uint32_t item = cur_item[0];
        if (item >= last) break;
        const uint32_t lo = cur_item[1], span = cur_item[2], bmul = cur_item[3], nb = cur_item[4];
        if (tid == 0) fetch_item(misc + (sel ? 8 : 24));
        sel ^= 1u;
        const uint2 it = p.items[item];
        const uint32_t b = it.x, part = it.y, S = p.S[b];
        const bool hashed = p.mode[b] == kModeHashed;
        const long long off0 = p.cand_offsets[b];
        const long long Cll = p.cand_offsets[b + 1] - off0;
        const uint32_t C = Cll > 0 ? (uint32_t)Cll : 0u;
        // pre-partitioned: this item's IDs were split off by partition_kernel; every ID read is ours
        const bool pre = !LD && p.part_ids != nullptr && S > 1 && p.part_ok[b] != 0;
        const uint32_t Cin = pre ? p.bucket_cnt[item] : C;     // IDs this pass reads

        // candidate list as 16-byte vectors; vector 0 may start up to 3 elements before the list.
        // Vectors [v_in0, v_in1) lie wholly inside the list and are read with one 16-byte load.
        const uint32_t *ids = pre ? p.part_ids + 2 * off0 + (size_t)part * (uint32_t)(2ull * C / S) : p.cand_ids + off0;
        const uint32_t shift = LD ? 0u : (uint32_t)((reinterpret_cast<uintptr_t>(ids) >> 2) & 3u);
        const uint4 *ids4 = reinterpret_cast<const uint4 *>(ids - shift);
        uint32_t nvec = Cin ? (Cin + shift + 3u) >> 2 : 0u;
        const uint32_t v_in0 = shift ? 1u : 0u, v_in1 = (Cin + shift) >> 2;
        const uint4 none4 = make_uint4(kIdNone, kIdNone, kIdNone, kIdNone);
        uint32_t ld_total = 0;                                 // lists-direct: IDs of this item's segments
        if constexpr (LD) {
            // The item's IDs are one segment of every probed list: the whole list (hashed classes), or its IDs of
            // this ID-range class, bounded by two entries of the list's grid.  Segment table, prefix of the
            // lengths, and for every 32 positions of the concatenation the segment its first position is in.
            const uint32_t w = hashed ? 0u : kGridCells / S;
            uint32_t len = 0;
            if (tid < p.nprobe) {
                const uint32_t l = __ldg(p.probes + (size_t)b * p.nprobe + tid);
                if ((uint64_t)l < p.n_lists) {
                    const uint16_t *g = p.list_grid + (size_t)l * (kGridCells + 1);
                    const uint32_t a = hashed ? 0u : __ldg(g + part * w), e = hashed ? __ldg(g + kGridCells) : __ldg(g + (part + 1) * w);
                    seg_start[tid] = (uint32_t)(__ldg(p.list_offsets + l) + a);
                    len = e - a;
                }
            }
            uint32_t incl = len;                               // block exclusive scan of the lengths
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += u;
            }
            if (lane == 31) wsum[warp] = incl;
            __syncthreads();
            if (warp == 0) {
                const uint32_t wv = lane < T / 32 ? wsum[lane] : 0u;
                uint32_t wi = wv;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t u = __shfl_up_sync(0xffffffffu, wi, o);
                    if (lane >= o) wi += u;
                }
                wsum[lane] = wi - wv;
                if (lane == 31) misc[6] = wi;                  // IDs of the item
            }
            __syncthreads();
            const uint32_t ex = wsum[warp] + incl - len;
            ld_total = misc[6];
            if (tid < p.nprobe) seg_prefix[tid] = ex;
            if (tid == 0) seg_prefix[p.nprobe] = ld_total;
            if (len) {                                         // rows whose first position lies in this segment
                for (uint32_t r = (ex + 31u) >> 5; (r << 5) < ex + len; ++r)
                    if (r < kLdRowMap) row_map[r] = (uint16_t)tid;
            }
            nvec = ((ld_total + 127u) >> 7) << 5;              // groups of 32 vectors = 128 positions
            __syncthreads();
        }
        auto load_vec = [&](uint32_t v) -> uint4 {
            if constexpr (LD) {
                // vectors 32 g .. 32 g + 31 (one warp) cover positions [128 g, 128 g + 128) of the concatenated
                // segments; element e of lane l is position 128 g + 32 e + l, so every load of a warp is contiguous
                uint32_t x[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t q0 = ((v >> 5) << 7) + 32u * e, q = q0 + (v & 31u);   // the row's first position: warp-uniform
                    x[e] = kIdNone;
                    if (q0 < ld_total) {
                        uint32_t sg;
                        if ((q0 >> 5) < kLdRowMap) {
                            sg = row_map[q0 >> 5];
                        } else {                               // beyond the row map (hashed classes read whole lists): search
                            uint32_t lo_s = 0, hi_s = p.nprobe;
                            while (hi_s - lo_s > 1) { const uint32_t mid = (lo_s + hi_s) >> 1; if (seg_prefix[mid] <= q0) lo_s = mid; else hi_s = mid; }
                            sg = lo_s;
                        }
                        if (q0 + 31u >= seg_prefix[sg + 1]) {  // the row runs into later segments: every lane finds its own
                            if (q < ld_total) {
                                while (q >= seg_prefix[sg + 1]) ++sg;   // also skips empty segments
                                x[e] = __ldg(p.list_ids + seg_start[sg] + (q - seg_prefix[sg]));
                            }
                        } else {
                            x[e] = __ldg(p.list_ids + (seg_start[sg] + (q - seg_prefix[sg])));
                        }
                    }
                }
                return make_uint4(x[0], x[1], x[2], x[3]);
            } else {
                if (v >= v_in0 && v < v_in1) return __ldg(ids4 + v);
                if (v < nvec) return load_ids4(ids, 4ll * v - shift, Cin);
                return none4;
            }
        };
        // hashed mode: bucket and home slot of a valid ID
        auto hash_of = [&](uint32_t x) -> uint32_t {
            uint32_t a = hash_round1(x);
            a = (a ^ (a >> 15)) * 0x846ca68bU;
            return a ^ (a >> 16);
        };
        // byte offset of the slot an ID tries first inside its bucket: low bits the bucket index does not use
        auto home_of = [&](uint32_t x) -> uint32_t { return ((hashed ? hash_of(x) : x - lo) << 2) & (4u * BS - 4u); };
        // the bucket an ID of this partition looks at first
        auto bucket_of = [&](uint32_t x) -> uint32_t { return tbl + ((hashed ? __umulhi(hash_of(x), nb) : __umulhi(x - lo, bmul)) << BSH); };
        const uint32_t tbl_end = tbl + (nb << BSH);
        auto next_bucket = [&](uint32_t a) -> uint32_t { return a + 4 * BS == tbl_end ? tbl : a + 4 * BS; };
        // One look at bucket `a` for ID `x` (kIdNone looks at the empty bucket and "finds itself" there):
        // x is there (a repeat): x becomes kIdNone; else returns the slot x will store itself to (its home slot if
        // that is empty, else the first empty one), or none_addr with x unchanged if the bucket is full of other
        // IDs.  `home` = byte offset of the slot tried first.
        auto look = [&](uint32_t &x, uint32_t a, uint32_t home) -> uint32_t {
            bool found;
            uint32_t off = kNoSlot;
            if (BS == 4) {
                const uint4 v = lds_u128(a);
                // the home slot's value out of the four just read (a second, 4-byte load costs more: the kernel
                // is bound by shared-memory wavefronts -- random 16-byte reads conflict 2.7x -- as much as by issue)
                const uint32_t hlo = (home & 4u) ? v.y : v.x, hhi = (home & 4u) ? v.w : v.z;
                const uint32_t hv = (home & 8u) ? hhi : hlo;
                found = v.x == x || v.y == x || v.z == x || v.w == x;
                off = v.w == kEmpty ? 12u : off;
                off = v.z == kEmpty ? 8u : off;
                off = v.y == kEmpty ? 4u : off;
                off = v.x == kEmpty ? 0u : off;
                off = hv == kEmpty ? home : off;
            } else if (BS == 2) {
                const uint2 v = lds_u64(a);
                found = v.x == x || v.y == x;
                const uint32_t hv = home ? v.y : v.x, ov = home ? v.x : v.y;
                off = ov == kEmpty ? home ^ 4u : off;
                off = hv == kEmpty ? home : off;
            } else {
                const uint32_t v = lds_u32(a);
                found = v == x;
                off = v == kEmpty ? 0u : off;
            }
            if (found) x = kIdNone;
            return (found || off == kNoSlot) ? none_addr : a + off;
        };
        // Places the entries of this thread whose bit is set in `keep` (t[j] = bucket to start at), each walking
        // its bucket sequence in the same three phases, until every thread of the CTA is done.  Used for what the
        // queue holds when the list is exhausted (NK = 1, one entry per thread), and for entries that found the
        // queue full (IDs chosen to collide).
        auto place_kept = [&](auto &id, auto &t, uint32_t keep) {
            constexpr int NK = sizeof(id) / sizeof(id[0]);
            for (;;) {
#pragma unroll
                for (int j = 0; j < NK; ++j) {
                    if (!(keep >> j & 1u)) continue;
                    const uint32_t home = home_of(id[j]);
                    uint32_t a = t[j] & kBucketMask, steps = 0;
                    for (;;) {
                        const uint32_t r = look(id[j], a, home);
                        if (id[j] == kIdNone) { keep &= ~(1u << j); break; }
                        if (r != none_addr) { a = r; break; }
                        a = next_bucket(a);
                        if (++steps > nb) {                    // the table is full of other IDs: give up on this one
                            atomicOr(&p.hdr->status, kStatusTableFull);
                            keep &= ~(1u << j);
                            break;
                        }
                    }
                    t[j] = a;
                }
                if (!__syncthreads_or(keep != 0)) break;       // all reads done
#pragma unroll
                for (int j = 0; j < NK; ++j)
                    if (keep >> j & 1u) sts_u32(t[j], id[j]);
                __syncthreads();                               // all stores done
#pragma unroll
                for (int j = 0; j < NK; ++j)
                    if ((keep >> j & 1u) && lds_u32(t[j]) == id[j]) keep &= ~(1u << j);
            }
        };
        uint4 nxt[NV];                                         // this thread's vectors of the next batch
#pragma unroll
        for (int i = 0; i < NV; ++i) nxt[i] = load_vec(tid + i * T);
        // (no barrier here: the table is empty since the last pass's compaction, which the barrier at the top of
        // the loop closed; the queue lengths are reset there too)

        uint32_t qin = 0, qn = 0;                              // queue read by this batch, its length
        for (uint32_t vbase = 0; vbase < nvec; vbase += NV * T) {
            uint32_t id[NE], t[NE];                            // t: slot to store to, none_addr = nothing to store
#pragma unroll
            for (int i = 0; i < NV; ++i) {
                id[4 * i] = nxt[i].x; id[4 * i + 1] = nxt[i].y; id[4 * i + 2] = nxt[i].z; id[4 * i + 3] = nxt[i].w;
                nxt[i] = load_vec(vbase + (NV + i) * T + tid);
            }
            uint2 *qpush = queue + (qin ^ 1u) * QCAP;
            uint32_t *qpush_cnt = qcnt + (qin ^ 1u);
            // ---- read: one look per entry
            if (!hashed) {
#pragma unroll
                for (int j = 0; j < R; ++j) {
                    const uint32_t x = id[j] - lo;
                    // class test: drops other classes, IDs >= N and kIdNone (lo + span <= N); a
                    // pre-partitioned bucket holds only this class, so there it drops just the padding
                    const bool mine = x < span;
                    if (!mine) id[j] = kIdNone;
                    t[j] = look(id[j], mine ? tbl + (__umulhi(x, bmul) << BSH) : none_addr, (x << 2) & (4u * BS - 4u));
                }
            } else {
#pragma unroll
                for (int j = 0; j < R; ++j) {
                    const uint32_t x = id[j];
                    const bool mine = (uint64_t)x < p.N && (S == 1 || __umulhi(hash_round1(x), S) == part);
                    const uint32_t h = hash_of(x);
                    if (!mine) id[j] = kIdNone;
                    // bucket from the high bits of h, home slot from the low bits
                    t[j] = look(id[j], mine ? tbl + (__umulhi(h, nb) << BSH) : none_addr, (h << 2) & (4u * BS - 4u));
                }
            }
            uint32_t aq[NQ];                                   // the buckets the queued entries look at
#pragma unroll
            for (int i = 0; i < NQ; ++i) {
                uint32_t home = 0;
                aq[i] = none_addr;
                id[R + i] = kIdNone;
                if (tid + i * T < qn) {
                    const uint2 e = queue[qin * QCAP + tid + i * T];
                    id[R + i] = e.x; aq[i] = e.y;
                    home = home_of(e.x);
                }
                t[R + i] = look(id[R + i], aq[i], home);
            }
            uint32_t all = id[0];
#pragma unroll
            for (int j = 1; j < NE; ++j) all &= id[j];
            const bool any_left = __syncthreads_or(all != kIdNone);   // all reads done
            if (tid == 0) qcnt[qin] = 0;                       // drained queue: its length was read before this barrier
            uint32_t keep = 0;                                 // entries that found the queue full
            if (any_left) {
                // ---- write
#pragma unroll
                for (int j = 0; j < NE; ++j)
                    if (t[j] != none_addr) sts_u32(t[j], id[j]);
                __syncthreads();                               // all stores done
                // ---- verify: of several stores to one slot one survived.  Losers (same bucket again) and IDs
                // whose bucket was full (next bucket) go to the queue the next batch reads; an entry that is done
                // reads kEmpty == its id from the empty bucket.  A full queue (IDs chosen to collide) raises
                // misc[5]; the ID then stays with its thread and is placed right after this batch.
                uint32_t lost = 0;
#pragma unroll
                for (int j = 0; j < NE; ++j)
                    if (lds_u32(t[j]) != id[j]) lost |= 1u << j;
                if (lost) {                                    // one reservation per thread: no chain of atomics
                    uint32_t pos = atomicAdd(qpush_cnt, (uint32_t)__popc(lost));
#pragma unroll
                    for (int j = 0; j < NE; ++j) {
                        if (!(lost >> j & 1u)) continue;
                        if (t[j] == none_addr) t[j] = next_bucket(j < R ? bucket_of(id[j]) : aq[j < R ? 0 : j - R]);
                        if (pos < QCAP) qpush[pos] = make_uint2(id[j], t[j] & kBucketMask);
                        else { misc[5] = 1; keep |= 1u << j; }
                        ++pos;
                    }
                }
            }
            __syncthreads();                                   // queue complete; misc[5] final
            if (misc[5]) {
                place_kept(id, t, keep);
                if (tid == 0) misc[5] = 0;
                __syncthreads();
            }
            qin ^= 1u;                                         // the queue just filled is the next batch's input
            qn = qcnt[qin];
            if (qn > QCAP) qn = QCAP;
        }
        if (qn) {                                              // list exhausted: place what the queue still holds
            uint32_t id[NQ], t[NQ], keep = 0;
#pragma unroll
            for (int i = 0; i < NQ; ++i) {
                id[i] = kIdNone; t[i] = none_addr;
                if (tid + i * T < qn) {
                    const uint2 e = queue[qin * QCAP + tid + i * T];
                    id[i] = e.x; t[i] = e.y; keep |= 1u << i;
                }
            }
            place_kept(id, t, keep);
        }

        // compact the table in bucket order: count per warp range, scan, write
        {
            const uint32_t n4 = nb * BS / 4;                   // the table as groups of 4 slots
            const uint32_t chunk = ((n4 + 2 * T - 1) / (2 * T)) * 64;   // groups per warp, multiple of 64
            const uint32_t v0 = warp * chunk < n4 ? warp * chunk : n4;
            const uint32_t v1 = v0 + chunk < n4 ? v0 + chunk : n4;
            uint32_t c = 0;
            for (uint32_t v = v0 + lane; v < v1; v += 32) {
                const uint4 w = lds_u128(tbl + (v << 4));
                c += (w.x != kEmpty) + (w.y != kEmpty) + (w.z != kEmpty) + (w.w != kEmpty);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
            if (lane == 0) wsum[warp] = c;
            if (T < 1024 && tid >= T / 32 && tid < 32) wsum[tid] = 0;   // warps that do not exist
            __syncthreads();
            if (warp == 0) {
                const uint32_t wv = wsum[lane];
                uint32_t incl = wv;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += u;
                }
                wsum[lane] = incl - wv;                        // exclusive
                if (lane == 31) misc[0] = incl ? atomicAdd(p.uniq_counts + b, incl) : 0u;
            }
            __syncthreads();
            // eight adjacent slots per lane and step: the lane's distinct IDs (0..8) go out side by side at the
            // warp's running position plus the counts of the lanes below (a shuffle scan)
            uint32_t *out = p.uniq_ids + off0 + misc[0] + wsum[warp];
            for (uint32_t vb = v0; vb < v1; vb += 64) {
                const uint32_t v = vb + 2 * lane;
                const uint4 w0 = lds_u128(v < v1 ? tbl + (v << 4) : none_addr);
                const uint4 w1 = lds_u128(v + 1 < v1 ? tbl + (v << 4) + 16 : none_addr);
                if (v < v1) sts_u128(tbl + (v << 4), make_uint4(kEmpty, kEmpty, kEmpty, kEmpty));       // empty for the next pass
                if (v + 1 < v1) sts_u128(tbl + (v << 4) + 16, make_uint4(kEmpty, kEmpty, kEmpty, kEmpty));
                const uint32_t p1 = w0.x != kEmpty, p2 = p1 + (w0.y != kEmpty), p3 = p2 + (w0.z != kEmpty), p4 = p3 + (w0.w != kEmpty);
                const uint32_t p5 = p4 + (w1.x != kEmpty), p6 = p5 + (w1.y != kEmpty), p7 = p6 + (w1.z != kEmpty), n = p7 + (w1.w != kEmpty);
                uint32_t incl = n;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += u;
                }
                uint32_t *o = out + (incl - n);
                if (w0.x != kEmpty) o[0] = w0.x;
                if (w0.y != kEmpty) o[p1] = w0.y;
                if (w0.z != kEmpty) o[p2] = w0.z;
                if (w0.w != kEmpty) o[p3] = w0.w;
                if (w1.x != kEmpty) o[p4] = w1.x;
                if (w1.y != kEmpty) o[p5] = w1.y;
                if (w1.z != kEmpty) o[p6] = w1.z;
                if (w1.w != kEmpty) o[p7] = w1.w;
                out += __shfl_sync(0xffffffffu, incl, 31);
            }
        }
    }
}

// ---------------------------------------------------------------- (6)(7) gather + ADC + top-k

// Shared-memory map of one scan CTA (byte offsets):
//   [0, 64)              misc: count, write count, query, tau, pivot, counters
//   [64, +2 KB)          prune sample keys        [.., +1 KB) their ranks
//   [3136, +cap*8)       top-k candidate buffer, 64-bit keys (dist bits << 32 | id)
//   [.., +64 KB)         lookup table of the query, c-major: entry (c, col) at byte c*256 + col*4
//   [.., +warps*D*2.5 KB) per-warp rings of D stages (2 KB of code rows + the rows' IDs), D > 0 only
constexpr uint32_t kScanBufOff = 64 + kSample * 8 + kSample * 4;
constexpr uint32_t kRingStageBytes = 2048 + 512;     // 2 KB of code rows + the stage's IDs (32 .. 128 of them)
__host__ __device__ inline size_t scan_smem_bytes(uint32_t cap, uint32_t ring_depth = 0)
{
    return kScanBufOff + (size_t)cap * 8 + 65536 + (size_t)ring_depth * kScanWarps * kRingStageBytes;
}

struct ScanParams {
    const uint8_t *codes;                            // [N][16*G], library copy
    uint32_t M;
    const float *lut;                                // [B][M][256]
    const long long *cand_offsets;                   // [B+1]
    const uint32_t *uniq_ids;                        // distinct IDs, query b's list at cand_offsets[b]
    const uint32_t *uniq_counts;                     // [B]
    uint32_t k, cap;                                 // cap = candidate-buffer keys (power of two)
    uint32_t q_begin, q_end;
    uint32_t *counter;
    uint32_t *out_ids;                               // [B][k]
    float *out_dists;                                // [B][k]
    uint32_t *out_counts;                            // [B] or NULL
    uint32_t *out_uniq;                              // [B] or NULL
    uint32_t parts;                                  // CTAs per query: > 1 splits a query's distinct list (small batches)
    unsigned long long *part_keys;                   // [B][parts][k] partial top-k keys, merged by merge_parts_kernel
    // List-major experiment (fann_search_lists_stream): `codes` is the list-major copy, key_src holds (row of that
    // copy, vector-ID) pairs WITH repeats, query b's at cand_offsets[b] (uniq_counts[b] = C_b); an ID >= id_limit is
    // skipped, and the repeats are removed where the top-k buffer is pruned.  key_src == NULL otherwise.
    const uint32_t *key_src;
    uint32_t id_limit;                               // 0xFFFFFFFF (kIdNone only) on the ordinary path
};

// Column of sub-space m in the c-major shared-memory table.  G = 16-byte chunks (= lanes) per row.
//   G = 4: col = 32*(e>>3) + 8*q + (e&7)   with m = 16q + e
//   G = 2: col = m                          (columns 32..63 unused)
//   G = 1: col = e and 16 + e               (two copies, columns 32..63 unused)
// so that in every lookup step the 32 lanes of a warp read 32 different banks whatever the codes are.
template <int G>
__device__ __forceinline__ uint32_t m_of_col(uint32_t col)
{
    if (G == 4) return 16u * ((col >> 3) & 3u) + ((col & 7u) | ((col >> 5) << 3));
    if (G == 2) return col;
    return col & 15u;
}

// Keeps every key <= pivot, where the pivot is placed from a sorted sample so that at least k keys
// survive; falls back to an exact sort if that does not shrink the buffer enough.  On return
// buf[0 .. *cnt) holds the survivors (which include the k smallest) and *tau = pivot + 1.
template <int KPT>
__device__ __forceinline__ void prune(unsigned long long *buf, uint32_t *misc, unsigned long long *samp,
                                      uint32_t *rank, uint32_t k, uint32_t cap, uint32_t limit)
{
    volatile uint32_t *vm = misc;
    unsigned long long *tau_p = reinterpret_cast<unsigned long long *>(misc + 4);
    unsigned long long *pivot_p = reinterpret_cast<unsigned long long *>(misc + 6);
    const uint32_t tid = threadIdx.x, lane = tid & 31;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t n = vm[0];
    if (tid < kSample) { samp[tid] = buf[(unsigned long long)tid * n / kSample]; rank[tid] = 0; }
    if (tid == 0) { *pivot_p = kKeyMax - 1; misc[9] = 0; }
    __syncthreads();
    {
        constexpr int parts = kScanThreads / kSample, len = kSample / parts;
        const unsigned long long mine = samp[tid % kSample];
        const uint32_t p0 = (tid / kSample) * len;
        uint32_t r = 0;
#pragma unroll 8
        for (int i = 0; i < len; ++i) r += samp[p0 + i] < mine ? 1u : 0u;
        atomicAdd(&rank[tid % kSample], r);
    }
    __syncthreads();
    unsigned long long key[KPT];
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        const uint32_t i = tid + j * kScanThreads;
        key[j] = i < n ? buf[i] : kKeyMax;
    }
    const float e = (float)kSample * (float)k / (float)n;
    uint32_t tgt = (uint32_t)ceilf(e + 3.f * sqrtf(e) + 2.f);
    unsigned long long pivot = kKeyMax - 1;
    for (int attempt = 0; attempt < 4; ++attempt) {
        if (tgt > kSample - 1) tgt = kSample - 1;
        if (attempt == 3) { if (tid == 0) *pivot_p = kKeyMax - 1; }          // keep everything
        else if (tid < kSample && rank[tid] == tgt) *pivot_p = samp[tid];
        if (tid == 0) misc[8] = 0;
        __syncthreads();
        pivot = *reinterpret_cast<volatile unsigned long long *>(pivot_p);
        uint32_t c = 0;
#pragma unroll
        for (int j = 0; j < KPT; ++j) c += key[j] <= pivot ? 1u : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if (lane == 0 && c) atomicAdd(&misc[8], c);
        __syncthreads();
        if (vm[8] >= k) break;                                  // uniform: every thread reads the same word
        tgt = attempt == 1 ? kSample - 1 : 2 * tgt + 8;
        __syncthreads();
    }
    if (tid == 0) misc[1] = 0;
    __syncthreads();                                           // all keys are in registers: buf may be overwritten
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        const bool keep = key[j] <= pivot;
        const uint32_t bal = __ballot_sync(0xffffffffu, keep);
        if (bal) {
            uint32_t pos = 0;
            if (lane == 0) pos = atomicAdd(&misc[1], (uint32_t)__popc(bal));
            pos = __shfl_sync(0xffffffffu, pos, 0);
            if (keep) buf[pos + __popc(bal & lt_mask)] = key[j];
        }
    }
    __syncthreads();
    const uint32_t kept = vm[1];
    if (kept > limit) {                                        // pivot did not help (k close to n): exact
        for (uint32_t i = kept + tid; i < cap; i += kScanThreads) buf[i] = kKeyMax;
        __syncthreads();
        bitonic_sort_smem(buf, cap, 2);
        if (tid == 0) { misc[0] = k; *tau_p = buf[k - 1] + 1; }
    } else if (tid == 0) {
        misc[0] = kept;
        *tau_p = pivot + 1;
    }
    __syncthreads();
}

// List-major experiment: the buffer may hold a vector several times (once per probed list it sits in) -- with the
// same distance on integer data, with distances a rounding apart on real-valued data (a row's summation order
// depends on the lane that scores it).  Exact prune: sort by (id, dist), keep the first entry of every id, sort the
// survivors by (dist, id), keep the k smallest; tau = the k-th + 1 once k distinct vectors exist.  On return
// buf[0 .. *cnt) is ascending and holds every id once.
__device__ __forceinline__ void prune_exact(unsigned long long *buf, uint32_t *misc, uint32_t *scratch, uint32_t k, uint32_t cap)
{
    volatile uint32_t *vm = misc;
    unsigned long long *tau_p = reinterpret_cast<unsigned long long *>(misc + 4);
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n = vm[0] < cap ? vm[0] : cap;
    uint32_t P = 32;
    while (P < n) P <<= 1;
    for (uint32_t i = tid; i < P; i += kScanThreads) {         // (dist, id) -> (id, dist)
        const unsigned long long x = i < n ? buf[i] : kKeyMax;
        buf[i] = (x << 32) | (x >> 32);
    }
    __syncthreads();
    bitonic_sort_smem(buf, P, 2);
    constexpr int KPT = 8192 / kScanThreads;                   // keys per thread, consecutive (cap <= 8192)
    unsigned long long key[KPT];
    unsigned long long prev = (tid && tid * KPT - 1 < P) ? buf[tid * KPT - 1] : kKeyMax;
    uint32_t c = 0, flags = 0;
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        const uint32_t i = tid * KPT + j;
        key[j] = i < P ? buf[i] : kKeyMax;
        const bool first = key[j] != kKeyMax && (i == 0 || (uint32_t)(key[j] >> 32) != (uint32_t)(prev >> 32));
        prev = key[j];
        if (first) { flags |= 1u << j; ++c; }
    }
    uint32_t incl = c;                                         // block exclusive scan of c
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += u;
    }
    if (lane == 31) scratch[warp] = incl;
    __syncthreads();                                           // also: every key is in registers, buf may be overwritten
    if (warp == 0) {
        const uint32_t wv = lane < kScanWarps ? scratch[lane] : 0u;
        uint32_t wi = wv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += u;
        }
        if (lane < kScanWarps) scratch[lane] = wi - wv;
        if (lane == kScanWarps - 1) scratch[kScanWarps] = wi;   // distinct ids in all
    }
    __syncthreads();
    uint32_t pos = scratch[warp] + incl - c;
#pragma unroll
    for (int j = 0; j < KPT; ++j)
        if (flags >> j & 1u) buf[pos++] = (key[j] << 32) | (key[j] >> 32);   // back to (dist, id)
    const uint32_t d = scratch[kScanWarps];
    uint32_t P2 = 32;
    while (P2 < d) P2 <<= 1;
    __syncthreads();
    for (uint32_t i = d + tid; i < P2; i += kScanThreads) buf[i] = kKeyMax;
    __syncthreads();
    bitonic_sort_smem(buf, P2, 2);
    if (tid == 0) {
        if (d >= k) { misc[0] = k; *tau_p = buf[k - 1] + 1; }
        else misc[0] = d;
    }
    __syncthreads();
}

// 16 table lookups for the 16 code bytes a lane holds (Eq. 1).  The byte address of
// each lookup is built by one PRMT: byte 0 = this lane's column offset, byte 1 = the code.
template <int G>
__device__ __forceinline__ float adc16(const uint4 r, const unsigned char *lutb, const uint32_t (&Bw)[4],
                                       const uint32_t (&sel)[4], bool swap1, bool swap2)
{
    uint32_t w0 = swap1 ? r.y : r.x, w1 = swap1 ? r.x : r.y, w2 = swap1 ? r.w : r.z, w3 = swap1 ? r.z : r.w;
    if (G != 4) {
        const uint32_t t0 = swap2 ? w2 : w0, t1 = swap2 ? w3 : w1, t2 = swap2 ? w0 : w2, t3 = swap2 ? w1 : w3;
        w0 = t0; w1 = t1; w2 = t2; w3 = t3;
    }
    const uint32_t w[4] = {w0, w1, w2, w3};
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            uint32_t addr;
            asm("prmt.b32 %0, %1, %2, %3;" : "=r"(addr) : "r"(w[j]), "r"(Bw[G == 4 ? (j & 1) : j]), "r"(sel[i]));
            acc[i] += *reinterpret_cast<const float *>(lutb + addr + (G == 4 ? (j >> 1) * 128 : 0));
        }
    }
    return (acc[0] + acc[1]) + (acc[2] + acc[3]);
}

// D = 0: code rows go through registers (NB row groups in flight per lane).  D >= 2: every warp keeps a
// private ring of D stages in shared memory and fills it D - 1 stages ahead with 16-byte asynchronous
// copies, so row reads stay in flight while the warp computes.
// LM (list-major experiment): rows are numbered in the list-major copy, their vector-IDs come from p.key_src,
// repeats are removed by prune_exact.  The ordinary path is LM = false and carries none of it.
template <int G, int NB, int D, bool LM = false>
__global__ void __launch_bounds__(kScanThreads) scan_kernel(const ScanParams p)
{
    constexpr int ROWB = 16 * G;
    constexpr int KPT = 8192 / kScanThreads;                   // keys per thread in prune (cap <= 8192)
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t *misc = reinterpret_cast<uint32_t *>(smem);       // [0] cnt [1] wcnt [2] query [4,5] tau [6,7] pivot [8] count
    volatile uint32_t *vm = misc;
    unsigned long long *tau_p = reinterpret_cast<unsigned long long *>(misc + 4);
    unsigned long long *samp = reinterpret_cast<unsigned long long *>(smem + 64);
    uint32_t *rank = reinterpret_cast<uint32_t *>(smem + 64 + kSample * 8);
    unsigned long long *buf = reinterpret_cast<unsigned long long *>(smem + kScanBufOff);
    unsigned char *lutb = smem + kScanBufOff + (size_t)p.cap * 8;
    float *luts = reinterpret_cast<float *>(lutb);

    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t q = lane & (G - 1), r = lane / G;           // chunk of the row, row slot in the warp step
    const uint32_t x0 = r & 3u;                                // byte-in-word xor   (PRMT selector, free)
    const uint32_t x2 = G == 4 ? (r >> 2) & 1u : (r >> 2) & 3u; // word xor          (SEL swaps)
    const bool swap1 = (x2 & 1u) != 0, swap2 = (x2 & 2u) != 0;
    uint32_t Bw[4], sel[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        uint32_t v = 0;
        if (G == 4) {
            const uint32_t w = (uint32_t)(j & 1) ^ x2;
            for (uint32_t beta = 0; beta < 4; ++beta) v |= (4u * (8u * q + 4u * w + beta)) << (8 * beta);
        } else {
            const uint32_t w = (uint32_t)j ^ x2, half = G == 2 ? q : (r >> 4);
            for (uint32_t beta = 0; beta < 4; ++beta) v |= (4u * (16u * half + 4u * w + beta)) << (8 * beta);
        }
        Bw[j] = v;
        const uint32_t beta = (uint32_t)j ^ x0;
        sel[j] = (4u + beta) | (beta << 4) | ((8u | (4u + beta)) << 8) | ((8u | (4u + beta)) << 12);
    }
    constexpr int NBS = 4 / G;                                 // ring: IDs per lane per stage (a stage is 2 KB of rows)
    const uint32_t margin = kScanWarps * 32 * (D ? NBS : NB) + 64;   // keys appended between the buffer passing its limit and the prune
    const uint32_t limit = p.cap - margin;

    // The next work item is taken while the current one is scanned: thread 0 holds the counter's answer in a register
    // (the atomic's round trip overlaps the scan) and publishes it when the query is done.
    uint32_t next_work = 0;
    if (tid == 0) next_work = atomicAdd(p.counter, 1u);
    for (;;) {
        if (tid == 0) misc[2] = next_work;
        __syncthreads();                                       // previous query fully done; misc[2] visible
        const uint32_t work = misc[2];                         // (query, part of its distinct list)
        if (work >= (p.q_end - p.q_begin) * p.parts) break;
        if (tid == 0) next_work = atomicAdd(p.counter, 1u);
        const uint32_t b = p.q_begin + work / p.parts, part = work % p.parts;
        const long long off0 = p.cand_offsets[b];
        uint32_t U = p.uniq_counts[b];
        const uint32_t *uq = p.uniq_ids + off0;
        if (p.parts > 1) {                                     // this CTA's slice, cut at multiples of 512 IDs
            const uint32_t chunks = (U + 511u) >> 9;
            const uint32_t c0 = (uint32_t)((unsigned long long)chunks * part / p.parts) << 9;
            const uint32_t c1 = (uint32_t)((unsigned long long)chunks * (part + 1) / p.parts) << 9;
            uq += c0;
            U = (c1 < U ? c1 : U) - (c0 < U ? c0 : U);
        }

        // stage the lookup table c-major; each warp writes 32 different banks per store
        auto stage_lut = [&]() {
            constexpr uint32_t ncols = G == 4 ? 64 : 32;
            const float4 *g4 = reinterpret_cast<const float4 *>(p.lut + (size_t)b * p.M * 256);
#pragma unroll 4
            for (uint32_t i = tid; i < ncols * 64; i += kScanThreads) {
                const uint32_t col = i % ncols, c4 = i / ncols;
                const uint32_t m = m_of_col<G>(col);
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (m < p.M) v = __ldg(g4 + m * 64 + c4);
                float *d = luts + (c4 * 4) * 64 + col;
                d[0] = v.x; d[64] = v.y; d[128] = v.z; d[192] = v.w;
            }
            if (tid == 0) { misc[0] = 0; misc[9] = 0; *tau_p = kKeyMax; }
        };

        if constexpr (D > 0) {
            const uint32_t ring = (uint32_t)__cvta_generic_to_shared(lutb + 65536) + warp * (D * kRingStageBytes);
            const uint32_t per_stage = 32 * NBS;
            const uint32_t n_st = (U + kScanWarps * per_stage - 1) / (kScanWarps * per_stage);   // stages per warp
            uint32_t idn[NBS], kidn[NBS];                      // rows of the next stage to issue and their vector-IDs, loaded one stage ahead
            auto load_ids = [&](uint32_t st) {
                const uint32_t base = (st * kScanWarps + warp) * per_stage;
#pragma unroll
                for (int nb = 0; nb < NBS; ++nb) {
                    const uint32_t idx = base + nb * 32 + lane;
                    if constexpr (LM) {                        // (row of the list-major copy, vector-ID) pairs
                        const uint2 rv = idx < U ? __ldg(reinterpret_cast<const uint2 *>(p.key_src) + off0 + idx)
                                                 : make_uint2(kIdNone, kIdNone);
                        idn[nb] = rv.x; kidn[nb] = rv.y;
                    } else {
                        idn[nb] = idx < U ? __ldg(uq + idx) : kIdNone;
                        kidn[nb] = idn[nb];
                    }
                }
            };
            // start the copies of stage st (its IDs are in idn), then fetch the IDs of stage st + 1
            auto issue = [&](uint32_t st) {
                if (st < n_st && (st * kScanWarps + warp) * per_stage < U) {
                    const uint32_t sa = ring + (st % D) * kRingStageBytes;
#pragma unroll
                    for (int nb = 0; nb < NBS; ++nb) {
                        sts_u32(sa + 2048 + (nb * 32 + lane) * 4, kidn[nb]);
#pragma unroll
                        for (int t = 0; t < G; ++t) {
                            uint32_t rid = G == 1 ? idn[nb] : __shfl_sync(0xffffffffu, idn[nb], (lane & ~(G - 1)) | t);
                            if (rid == kIdNone) rid = 0;
                            // rows read together (same t) sit together: slot = t * (32 / G) + lane / G
                            cp_async_16(sa + (nb * 32 + t * (32 / G) + r) * ROWB + q * 16,
                                        p.codes + (uint64_t)rid * ROWB + q * 16);
                        }
                    }
                    load_ids(st + 1);
                }
                cp_async_commit();                             // one group per stage, empty past the end
            };
            // the first row copies go out before the table is staged: they need the IDs only, and fly meanwhile
            load_ids(0);
#pragma unroll
            for (int d = 0; d < D - 1; ++d) issue(d);
            stage_lut();
            __syncthreads();
            uint32_t st = 0;
            for (;;) {
                while (st < n_st && !vm[9]) {
                    issue(st + D - 1);
                    cp_async_wait<D - 1>();                    // stage st has landed (this lane's copies)
                    __syncwarp();                              // ... and every other lane's
                    if ((st * kScanWarps + warp) * per_stage < U) {
                        const uint32_t sa = ring + (st % D) * kRingStageBytes;
                        const unsigned long long tau = *reinterpret_cast<volatile unsigned long long *>(tau_p);
#pragma unroll
                        for (int nb = 0; nb < NBS; ++nb) {
                            float mine = 0.f;
#pragma unroll
                            for (int t = 0; t < G; ++t) {
                                const uint4 rw = lds_u128(sa + (nb * 32 + t * (32 / G) + r) * ROWB + q * 16);
                                float sum = adc16<G>(rw, lutb, Bw, sel, swap1, swap2);
                                if (G >= 2) sum += __shfl_xor_sync(0xffffffffu, sum, 1);
                                if (G == 4) sum += __shfl_xor_sync(0xffffffffu, sum, 2);
                                if (q == (uint32_t)t) mine = sum;
                            }
                            const uint32_t idv = lds_u32(sa + 2048 + (nb * 32 + lane) * 4);
                            const unsigned long long key = ((unsigned long long)__float_as_uint(mine) << 32) | idv;
                            const bool keep = (LM ? idv < p.id_limit : idv != kIdNone) && key < tau;
                            const uint32_t bal = __ballot_sync(0xffffffffu, keep);
                            if (bal) {
                                uint32_t pos = 0;
                                if (lane == 0) pos = atomicAdd(&misc[0], (uint32_t)__popc(bal));
                                pos = __shfl_sync(0xffffffffu, pos, 0);
                                if (keep) buf[pos + __popc(bal & lt_mask)] = key;
                            }
                        }
                        if (lane == 0 && vm[0] > limit) vm[9] = 1;
                    }
                    __syncwarp();                              // the stage's slot is refilled by the next issue
                    ++st;
                }
                if (!__syncthreads_or(vm[9] != 0)) break;
                if constexpr (LM) { prune_exact(buf, misc, rank, p.k, p.cap); if (tid == 0) misc[9] = 0; __syncthreads(); }
                else prune<KPT>(buf, misc, samp, rank, p.k, p.cap, limit);
            }
            cp_async_wait<0>();
        } else {
            stage_lut();
            __syncthreads();
            const uint32_t per_iter = kScanWarps * 32 * NB;
            const uint32_t n_iter = (U + per_iter - 1) / per_iter;
            // Warps run free: no barrier per iteration.  The warp whose append takes the buffer past its limit
            // raises misc[9]; every warp sees it before its next iteration (each appends at most one more
            // iteration's keys, which the margin above the limit holds) and meets the others at the barrier
            // below, where the buffer is pruned.  A warp out of work waits there too, so the barrier completes
            // exactly when every warp is done or has seen the flag.
            uint32_t itn = 0;
            for (;;) {
              while (itn < n_iter && !vm[9]) {
                const uint32_t base = (itn * kScanWarps + warp) * 32 * NB;
                ++itn;
                if (base < U) {
                    uint32_t id[NB];
    #pragma unroll
                    for (int nb = 0; nb < NB; ++nb) {
                        const uint32_t idx = base + nb * 32 + lane;
                        id[nb] = idx < U ? __ldg(uq + idx) : kIdNone;
                    }
                    uint4 rw[NB][G];
    #pragma unroll
                    for (int nb = 0; nb < NB; ++nb)
    #pragma unroll
                        for (int t = 0; t < G; ++t) {
                            uint32_t rid = G == 1 ? id[nb] : __shfl_sync(0xffffffffu, id[nb], (lane & ~(G - 1)) | t);
                            if (rid == kIdNone) rid = 0;
                            rw[nb][t] = ldg_nc_16(p.codes + (uint64_t)rid * ROWB + q * 16);
                        }
                    const unsigned long long tau = *reinterpret_cast<volatile unsigned long long *>(tau_p);
    #pragma unroll
                    for (int nb = 0; nb < NB; ++nb) {
                        float mine = 0.f;
    #pragma unroll
                        for (int t = 0; t < G; ++t) {
                            float s = adc16<G>(rw[nb][t], lutb, Bw, sel, swap1, swap2);
                            if (G >= 2) s += __shfl_xor_sync(0xffffffffu, s, 1);
                            if (G == 4) s += __shfl_xor_sync(0xffffffffu, s, 2);
                            if (q == (uint32_t)t) mine = s;
                        }
                        const unsigned long long key = ((unsigned long long)__float_as_uint(mine) << 32) | id[nb];
                        const bool keep = id[nb] != kIdNone && key < tau;
                        const uint32_t bal = __ballot_sync(0xffffffffu, keep);
                        if (bal) {
                            uint32_t pos = 0;
                            if (lane == 0) pos = atomicAdd(&misc[0], (uint32_t)__popc(bal));
                            pos = __shfl_sync(0xffffffffu, pos, 0);
                            if (keep) buf[pos + __popc(bal & lt_mask)] = key;
                        }
                    }
                    if (lane == 0 && vm[0] > limit) vm[9] = 1;
                }
              }
              if (!__syncthreads_or(vm[9] != 0)) break;
              prune<KPT>(buf, misc, samp, rank, p.k, p.cap, limit);
            }

        }

        // exact top-k of what is left
        uint32_t n = vm[0];
        if constexpr (LM) {                                    // list-major experiment: sorted and free of repeats
            prune_exact(buf, misc, rank, p.k, p.cap);
            n = vm[0];
        } else {
            if (n > 2 * p.k && n >= 1024) {
                prune<KPT>(buf, misc, samp, rank, p.k, p.cap, limit);
                n = vm[0];
            }
            uint32_t P = 32;
            while (P < n) P <<= 1;
            for (uint32_t i = n + tid; i < P; i += kScanThreads) buf[i] = kKeyMax;
            __syncthreads();
            bitonic_sort_smem(buf, P, 2);
        }
        const uint32_t cnt = n < p.k ? n : p.k;
        if (p.parts > 1) {                                     // partial result: the slice's k smallest keys, padded
            unsigned long long *pk = p.part_keys + ((size_t)b * p.parts + part) * p.k;
            for (uint32_t i = tid; i < p.k; i += kScanThreads) pk[i] = i < cnt ? buf[i] : kKeyMax;
            continue;
        }
        for (uint32_t i = tid; i < p.k; i += kScanThreads) {
            const bool pad = i >= cnt;
            const unsigned long long key = pad ? kKeyMax : buf[i];
            p.out_ids[(size_t)b * p.k + i] = pad ? kIdNone : (uint32_t)key;
            p.out_dists[(size_t)b * p.k + i] = pad ? __int_as_float(0x7f800000) : __uint_as_float((uint32_t)(key >> 32));
        }
        if (tid == 0) {
            if (p.out_counts) p.out_counts[b] = cnt;
            if (p.out_uniq) p.out_uniq[b] = U;
        }
    }
}

// Small batches: scan_kernel ran `parts` CTAs per query (a power of two), each on a slice
// of the query's distinct list; the slices are disjoint, so the query's top-k is the k smallest of the parts' keys.
// Every part's keys arrive sorted.  One CTA per query, K2 = power of two >= k, all keys in shared memory.
//   Selection first (parts >= 4): with m = ceil(k / parts), T = the largest of the parts' m-th keys bounds the
//   k-th smallest key of all from above (every part has m keys <= T, parts * m >= k), so only each part's prefix
//   of keys <= T can be in the result -- about 1.3 k keys instead of parts * k; they are gathered and sorted.
//   Otherwise (2 parts, a part with fewer than m keys, or prefixes longer than kMergeSelect keys): pairwise merge --
//   of two ascending lists a, b of K2 keys, min(a[i], b[K2-1-i]) are the K2 smallest of both as a bitonic
//   sequence, which log2(K2) compare-exchange steps sort; log2(parts) such rounds, all pairs of a round side by side.
constexpr int kMergeThreads = 512;
constexpr uint32_t kMergeSelect = 4096;              // most keys the selection path sorts (8 per thread)
__global__ void __launch_bounds__(kMergeThreads) merge_parts_kernel(const unsigned long long *__restrict__ part_keys,
                                                                    const uint32_t *__restrict__ uniq_counts, uint32_t q_begin,
                                                                    uint32_t parts, uint32_t k, uint32_t K2, uint32_t *out_ids,
                                                                    float *out_dists, uint32_t *out_counts, uint32_t *out_uniq)
{
    extern __shared__ __align__(16) unsigned char smem[];
    unsigned long long *buf = reinterpret_cast<unsigned long long *>(smem);   // [parts][K2]
    __shared__ unsigned long long s_bound;
    __shared__ uint32_t s_off[17];
    const uint32_t b = q_begin + blockIdx.x, tid = threadIdx.x;
    const uint32_t lg = 31u - (uint32_t)__clz(K2);
    const unsigned long long *src = part_keys + (size_t)b * parts * k;
    if (tid == 0) s_bound = 0ull;
    for (uint32_t i0 = tid; i0 < parts * K2; i0 += 8 * kMergeThreads) {     // eight independent loads in flight per thread
        unsigned long long r[8];
#pragma unroll
        for (uint32_t e = 0; e < 8; ++e) {
            const uint32_t i = i0 + e * kMergeThreads, pt = i >> lg, j = i & (K2 - 1);
            r[e] = (i < parts * K2 && j < k) ? __ldg(src + (size_t)pt * k + j) : kKeyMax;
        }
#pragma unroll
        for (uint32_t e = 0; e < 8; ++e) {
            const uint32_t i = i0 + e * kMergeThreads;
            if (i < parts * K2) buf[i] = r[e];
        }
    }
    __syncthreads();
    bool selected = false;
    if (parts >= 4) {
        const uint32_t m = (k + parts - 1) / parts;
        if (tid < parts) atomicMax(&s_bound, buf[((size_t)tid << lg) + m - 1]);
        __syncthreads();
        const unsigned long long T = s_bound;
        if (T != kKeyMax) {                                    // every part has at least m keys
            if (tid < parts) {                                 // keys <= T of part tid: a prefix of its sorted list
                const unsigned long long *a = buf + ((size_t)tid << lg);
                uint32_t lo = 0, hi = K2;
                while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (a[mid] <= T) lo = mid + 1; else hi = mid; }
                s_off[tid + 1] = lo;
            }
            if (tid == 0) s_off[0] = 0;
            __syncthreads();
            if (tid == 0) for (uint32_t q = 0; q < parts; ++q) s_off[q + 1] += s_off[q];
            __syncthreads();
            const uint32_t total = s_off[parts];
            if (total <= kMergeSelect) {                       // uniform: gather the prefixes (through registers: in place)
                unsigned long long r[kMergeSelect / kMergeThreads];
#pragma unroll
                for (uint32_t e = 0; e < kMergeSelect / kMergeThreads; ++e) {
                    const uint32_t i = tid + e * kMergeThreads;
                    r[e] = kKeyMax;
                    if (i < total) {
                        uint32_t q = 0;
                        while (s_off[q + 1] <= i) ++q;
                        r[e] = buf[((size_t)q << lg) + (i - s_off[q])];
                    }
                }
                __syncthreads();
                uint32_t P = 32;
                while (P < total) P <<= 1;
#pragma unroll
                for (uint32_t e = 0; e < kMergeSelect / kMergeThreads; ++e) {
                    const uint32_t i = tid + e * kMergeThreads;
                    if (i < P) buf[i] = r[e];
                }
                __syncthreads();
                bitonic_sort_smem(buf, P, 2);
                selected = true;
            }
        }
    }
    if (!selected) {
        for (uint32_t width = 1; width < parts; width <<= 1) {
            const uint32_t pairs = parts / (2 * width);
            for (uint32_t i = tid; i < pairs * K2; i += kMergeThreads) {   // the K2 smallest of each pair, into its first list
                const uint32_t pr = i >> lg, j = i & (K2 - 1);
                unsigned long long *a = buf + (size_t)pr * 2 * width * K2, *c = a + (size_t)width * K2;
                const unsigned long long x = a[j], y = c[K2 - 1 - j];
                a[j] = x < y ? x : y;
            }
            __syncthreads();
            for (uint32_t stride = K2 >> 1; stride > 0; stride >>= 1) {    // bitonic -> ascending
                for (uint32_t i = tid; i < pairs * (K2 >> 1); i += kMergeThreads) {
                    const uint32_t pr = i >> (lg - 1), j = i & ((K2 >> 1) - 1);
                    unsigned long long *a = buf + (size_t)pr * 2 * width * K2;
                    const uint32_t lo = 2 * j - (j & (stride - 1)), hi = lo + stride;
                    const unsigned long long x = a[lo], y = a[hi];
                    if (x > y) { a[lo] = y; a[hi] = x; }
                }
                __syncthreads();
            }
        }
    }
    const uint32_t U = uniq_counts[b], cnt = U < k ? U : k;
    for (uint32_t i = tid; i < k; i += kMergeThreads) {
        const bool pad = i >= cnt;
        const unsigned long long key = buf[i];
        out_ids[(size_t)b * k + i] = pad ? kIdNone : (uint32_t)key;
        out_dists[(size_t)b * k + i] = pad ? __int_as_float(0x7f800000) : __uint_as_float((uint32_t)(key >> 32));
    }
    if (tid == 0) {
        if (out_counts) out_counts[b] = cnt;
        if (out_uniq) out_uniq[b] = U;
    }
}

}  // namespace fann
