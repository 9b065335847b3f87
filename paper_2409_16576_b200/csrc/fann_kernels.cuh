// fann_kernels.cuh -- device code of the FusionANNS GPU stage for sm_100a.
//
// Kernels (section 3, steps (1)(5)(6)(7)):
//   repack_rows_kernel   fann_load_codes: pad rows of M bytes to a 16-byte multiple
//   build_lut_kernel     (1) lut[b][m][j] = sum_t (q - c)^2
//   plan_kernel          split each query into S_b hash partitions that fit one SM's table
//   scan_kernel          (5) shared-memory hash dedup  (6) code gather + Eq. 1 ADC
//                        (7) per-partition top-k, all fused, persistent CTAs
//   merge_kernel         (7) merge the S_b partial top-k lists of a query, write outputs
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fann {

constexpr uint32_t kIdNone = 0xFFFFFFFFu;
constexpr uint32_t kEmpty = 0xFFFFFFFFu;             // empty hash slot (never a valid id: id < N < 2^32-1)
constexpr unsigned long long kKeyMax = ~0ull;        // padding key, sorts last
constexpr int kScanThreads = 1024;
constexpr int kWarpQueue = 64;                       // winners staged per warp before scoring
constexpr uint32_t kStatusTableFull = 1u;
constexpr uint32_t kStatusPlanOverflow = 2u;

struct WsHeader {                                    // first 256 bytes of the workspace
    uint32_t work_counter;                           // next work item (scan kernel)
    uint32_t n_items;                                // work items of this batch
    uint32_t status;                                 // kStatus* bits
    uint32_t pad;
};

struct ScanParams {
    const uint8_t *codes;                            // [N][row_bytes], library copy
    uint64_t N;
    uint32_t row_bytes;
    const float *lut;                                // [B][M][256]
    uint32_t M;
    const long long *cand_offsets;                   // [B+1]
    const uint32_t *cand_ids;
    uint32_t k, KP, capbuf, ipt, nslots;
    WsHeader *hdr;
    const uint32_t *S;                               // [B] partitions per query
    const uint2 *items;                              // [n_items] (query, partition)
    uint32_t *part_count;                            // [n_items]
    uint32_t *part_uniq;                             // [n_items]
    unsigned long long *part_keys;                   // [n_items][KP]
    uint32_t *uniq_ids;                              // dump mode: [total_cands]
    uint32_t *uniq_counts;                           // dump mode: [B]
};

// ---------------------------------------------------------------- helpers

__device__ __forceinline__ uint32_t mix32(uint32_t x)
{
    x *= 0x85EBCA6Bu;
    x ^= x >> 15;
    x *= 0xC2B2AE35u;
    x ^= x >> 16;
    return x;
}

__device__ __forceinline__ uint4 ldg_nc_16(const void *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// Block-wide bitonic sort (ascending) of n = 2^p keys in shared memory,
// starting from sorted runs of length `run` (run = 1: full sort; run = n/2 with
// the second half stored descending: a single merge).
__device__ __forceinline__ void bitonic_sort_smem(unsigned long long *a, uint32_t n, uint32_t first_size)
{
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

// One thread = 4 consecutive centroids j of one (query, sub-space).
__global__ void build_lut_kernel(const float *__restrict__ queries, const float *__restrict__ codebooks,
                                 float *__restrict__ lut, uint32_t B, uint32_t M, uint32_t dsub)
{
    uint64_t u = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t per_q = (uint64_t)M * 64;
    if (u >= (uint64_t)B * per_q) return;
    uint32_t b = (uint32_t)(u / per_q);
    uint32_t rem = (uint32_t)(u % per_q);
    uint32_t m = rem >> 6, j0 = (rem & 63) << 2;
    const float *q = queries + (size_t)b * M * dsub + (size_t)m * dsub;
    const float *c = codebooks + ((size_t)m * 256 + j0) * dsub;
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    for (uint32_t t = 0; t < dsub; ++t) {
        float qv = __ldg(q + t);
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
            float dlt = qv - __ldg(c + jj * dsub + t);
            s[jj] = fmaf(dlt, dlt, s[jj]);
        }
    }
    *reinterpret_cast<float4 *>(lut + ((size_t)b * M + m) * 256 + j0) = make_float4(s[0], s[1], s[2], s[3]);
}

// ---------------------------------------------------------------- plan

// Single CTA.  S_b = ceil(C_b / cap_c) hash partitions per query, so that the
// IDs one partition can receive fit the per-CTA table at <= 80 % load even if
// none repeats.  Writes item_start[B+1], items[], n_items; resets the counters.
__global__ void plan_kernel(const long long *__restrict__ cand_offsets, uint32_t B, uint32_t cap_c,
                            uint32_t max_items, WsHeader *hdr, uint32_t *S, uint32_t *item_start,
                            uint2 *items, uint32_t *uniq_counts)
{
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t running;
    if (threadIdx.x == 0) running = 0;
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (uint32_t base = 0; base < B; base += blockDim.x) {
        uint32_t b = base + threadIdx.x;
        uint32_t s = 0;
        if (b < B) {
            long long c = cand_offsets[b + 1] - cand_offsets[b];
            if (c < 0) c = 0;
            s = (uint32_t)((c + cap_c - 1) / cap_c);
            if (s == 0) s = 1;
            S[b] = s;
            if (uniq_counts) uniq_counts[b] = 0;
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
                if (start + p < max_items) items[start + p] = make_uint2(b, p);
        }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) running = start + s;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        item_start[B] = running;
        hdr->work_counter = 0;
        hdr->status = (running > max_items) ? kStatusPlanOverflow : 0u;
        hdr->n_items = (running > max_items) ? 0u : running;
    }
}

// ---------------------------------------------------------------- (5)(6)(7) fused scan

// Shared-memory map of one scan CTA (byte offsets), see scan_smem_bytes().
//   [0, 64)            misc: item, buffer count, uniq count, tau
//   [64, +capbuf*8)    top-k candidate buffer, 64-bit keys (dist bits << 32 | id)
//   [.., +8 KB)        per-warp queues of dedup winners waiting to be scored
//   [.., +row_bytes KB) lookup table of the query, [row_bytes][256] fp32 (rows >= M are zero)
//   [.., +nslots*4)    dedup hash table (open addressing, linear probing)
__host__ __device__ inline size_t scan_smem_bytes(uint32_t capbuf, uint32_t row_bytes, uint32_t nslots)
{
    return 64 + (size_t)capbuf * 8 + (size_t)(kScanThreads / 32) * kWarpQueue * 4 +
           (size_t)row_bytes * 1024 + (size_t)nslots * 4;
}

// Eq. 1 for one row held in registers: one table read per code byte.
template <int NCHUNK>
__device__ __forceinline__ float adc_row(const uint4 (&r)[NCHUNK], const float *lut)
{
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < NCHUNK; ++c) {
        const uint32_t w[4] = {r[c].x, r[c].y, r[c].z, r[c].w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
#pragma unroll
            for (int by = 0; by < 4; ++by) {
                uint32_t code = (w[i] >> (8 * by)) & 0xFFu;
                acc += lut[(c * 16 + i * 4 + by) * 256 + code];
            }
        }
    }
    return acc;
}

template <int NCHUNK, bool DUMP>
__global__ void __launch_bounds__(kScanThreads, 1) scan_kernel(const ScanParams p)
{
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t *misc = reinterpret_cast<uint32_t *>(smem);
    unsigned long long *tau_p = reinterpret_cast<unsigned long long *>(smem + 16);
    unsigned long long *buf = reinterpret_cast<unsigned long long *>(smem + 64);
    uint32_t *wq = reinterpret_cast<uint32_t *>(smem + 64 + (size_t)p.capbuf * 8);
    float *lut = reinterpret_cast<float *>(wq + (kScanThreads / 32) * kWarpQueue);
    uint32_t *table = reinterpret_cast<uint32_t *>(lut + (size_t)p.row_bytes * 256);

    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t nslots = p.nslots;
    const uint32_t n_items = p.hdr->n_items;
    const uint32_t prune_thresh = p.capbuf - kScanThreads * (p.ipt + 1);
    uint32_t *myq = wq + warp * kWarpQueue;

    for (;;) {
        __syncthreads();                                       // previous item fully done
        if (tid == 0) misc[0] = atomicAdd(&p.hdr->work_counter, 1u);
        __syncthreads();
        const uint32_t item = misc[0];
        if (item >= n_items) break;
        const uint2 it = p.items[item];
        const uint32_t b = it.x, part = it.y, S = p.S[b];
        const long long off0 = p.cand_offsets[b];
        const long long C = p.cand_offsets[b + 1] - off0;

        {   // clear the table, stage the lookup table
            uint4 *t4 = reinterpret_cast<uint4 *>(table);
            const uint4 e4 = make_uint4(kEmpty, kEmpty, kEmpty, kEmpty);
            for (uint32_t i = tid; i < (nslots >> 2); i += kScanThreads) t4[i] = e4;
            if (!DUMP) {
                const float4 *g4 = reinterpret_cast<const float4 *>(p.lut + (size_t)b * p.M * 256);
                float4 *l4 = reinterpret_cast<float4 *>(lut);
                const uint32_t n_real = p.M * 64, n_all = p.row_bytes * 64;
                for (uint32_t i = tid; i < n_all; i += kScanThreads)
                    l4[i] = (i < n_real) ? __ldg(g4 + i) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
            if (tid == 0) { misc[1] = 0; misc[2] = 0; *tau_p = kKeyMax; }
        }
        __syncthreads();

        uint32_t qn = 0;                                       // entries in this warp's queue (warp-uniform)
        uint32_t n_won = 0;                                    // winners seen by this warp (lane 0 counts)

        // score the ids in myq[0 .. n), n <= 32: gather the code row, Eq. 1, threshold, append
        auto score = [&](uint32_t n) {
            const bool act = lane < n;
            unsigned long long key = kKeyMax;
            if (act) {
                const uint32_t id = myq[lane];
                const uint4 *row = reinterpret_cast<const uint4 *>(p.codes + (uint64_t)id * p.row_bytes);
                uint4 r[NCHUNK];
#pragma unroll
                for (int c = 0; c < NCHUNK; ++c) r[c] = ldg_nc_16(row + c);
                const float d = adc_row<NCHUNK>(r, lut);
                key = ((unsigned long long)__float_as_uint(d) << 32) | id;
            }
            const bool keep = act && key < *tau_p;
            const uint32_t bal = __ballot_sync(0xffffffffu, keep);
            if (bal) {
                uint32_t basep = 0;
                if (lane == 0) basep = atomicAdd(&misc[1], (uint32_t)__popc(bal));
                basep = __shfl_sync(0xffffffffu, basep, 0);
                if (keep) buf[basep + __popc(bal & lt_mask)] = key;
            }
        };

        for (long long base = 0; base < C; base += (long long)kScanThreads * p.ipt) {
            for (uint32_t i = 0; i < p.ipt; ++i) {
                const long long idx = base + (long long)i * kScanThreads + tid;
                bool won = false;
                uint32_t id = kIdNone;
                if (idx < C) {
                    id = __ldg(p.cand_ids + off0 + idx);
                    if (id != kIdNone && (uint64_t)id < p.N) {
                        const unsigned long long pr = (unsigned long long)mix32(id) * S;
                        if ((uint32_t)(pr >> 32) == part) {
                            uint32_t slot = __umulhi((uint32_t)pr, nslots);
                            for (uint32_t probes = 0;; ++probes) {
                                const uint32_t cur = *reinterpret_cast<volatile uint32_t *>(table + slot);
                                if (cur == id) break;
                                if (cur == kEmpty) {
                                    const uint32_t old = atomicCAS(table + slot, kEmpty, id);
                                    if (old == kEmpty) { won = true; break; }
                                    if (old == id) break;
                                }
                                slot = (slot + 1 == nslots) ? 0u : slot + 1;
                                if (probes >= nslots) { atomicOr(&p.hdr->status, kStatusTableFull); break; }
                            }
                        }
                    }
                }
                const uint32_t bal = __ballot_sync(0xffffffffu, won);
                if (bal) {
                    if (lane == 0) n_won += __popc(bal);
                    if (DUMP) {
                        uint32_t basep = 0;
                        if (lane == 0) basep = atomicAdd(p.uniq_counts + b, (uint32_t)__popc(bal));
                        basep = __shfl_sync(0xffffffffu, basep, 0);
                        if (won) p.uniq_ids[off0 + basep + __popc(bal & lt_mask)] = id;
                    } else {
                        if (won) myq[qn + __popc(bal & lt_mask)] = id;
                        qn += __popc(bal);
                        __syncwarp();
                        if (qn >= 32) {
                            score(32);
                            const uint32_t rem = qn - 32;
                            const uint32_t v = (lane < rem) ? myq[32 + lane] : 0u;
                            __syncwarp();
                            if (lane < rem) myq[lane] = v;
                            __syncwarp();
                            qn = rem;
                        }
                    }
                }
            }
            if (!DUMP) {
                if (__syncthreads_or(misc[1] > prune_thresh)) {
                    const uint32_t cnt = misc[1];
                    for (uint32_t i = cnt + tid; i < p.capbuf; i += kScanThreads) buf[i] = kKeyMax;
                    __syncthreads();
                    bitonic_sort_smem(buf, p.capbuf, 2);
                    if (tid == 0) {
                        misc[1] = cnt < p.k ? cnt : p.k;
                        *tau_p = cnt >= p.k ? buf[p.k - 1] : kKeyMax;
                    }
                    __syncthreads();
                }
            }
        }
        if (!DUMP && qn > 0) score(qn);
        if (lane == 0 && n_won) atomicAdd(&misc[2], n_won);
        __syncthreads();
        if (tid == 0) p.part_uniq[item] = misc[2];
        if (!DUMP) {
            const uint32_t cnt = misc[1];
            for (uint32_t i = cnt + tid; i < p.capbuf; i += kScanThreads) buf[i] = kKeyMax;
            __syncthreads();
            bitonic_sort_smem(buf, p.capbuf, 2);
            const uint32_t keep = cnt < p.k ? cnt : p.k;
            unsigned long long *out = p.part_keys + (size_t)item * p.KP;
            for (uint32_t i = tid; i < p.KP; i += kScanThreads) out[i] = (i < keep) ? buf[i] : kKeyMax;
            if (tid == 0) p.part_count[item] = keep;
        }
    }
}

// ---------------------------------------------------------------- (7) merge + outputs

// One CTA per query: merges the S_b ascending partial lists (KP keys each,
// padded with kKeyMax) with bitonic merges in shared memory, writes
// out_ids / out_dists (ascending, padded with (NONE, +inf)), counts, uniq.
__global__ void merge_kernel(uint32_t k, uint32_t KP, const WsHeader *hdr, const uint32_t *S,
                             const uint32_t *item_start, const uint32_t *part_uniq,
                             const unsigned long long *part_keys, uint32_t *out_ids, float *out_dists,
                             uint32_t *out_counts, uint32_t *out_uniq)
{
    extern __shared__ __align__(16) unsigned char smem[];
    unsigned long long *keys = reinterpret_cast<unsigned long long *>(smem);
    __shared__ uint32_t s_cnt;
    const uint32_t b = blockIdx.x, tid = threadIdx.x;
    const bool bad = (hdr->status & kStatusPlanOverflow) != 0;
    const uint32_t first = bad ? 0 : item_start[b], Sb = bad ? 0 : S[b];
    if (tid == 0) s_cnt = 0;
    for (uint32_t i = tid; i < KP; i += blockDim.x)
        keys[i] = Sb ? part_keys[(size_t)first * KP + i] : kKeyMax;
    __syncthreads();
    for (uint32_t s = 1; s < Sb; ++s) {
        for (uint32_t i = tid; i < KP; i += blockDim.x)
            keys[2 * KP - 1 - i] = part_keys[(size_t)(first + s) * KP + i];
        __syncthreads();
        bitonic_sort_smem(keys, 2 * KP, 2 * KP);               // ascending + descending halves: one merge
    }
    uint32_t local = 0;
    for (uint32_t i = tid; i < k; i += blockDim.x) {
        const unsigned long long key = keys[i];
        const bool pad = key == kKeyMax;
        out_ids[(size_t)b * k + i] = pad ? kIdNone : (uint32_t)key;
        out_dists[(size_t)b * k + i] = pad ? __int_as_float(0x7f800000) : __uint_as_float((uint32_t)(key >> 32));
        local += pad ? 0u : 1u;
    }
    if (local) atomicAdd(&s_cnt, local);
    __syncthreads();
    if (tid == 0) {
        if (out_counts) out_counts[b] = s_cnt;
        if (out_uniq) {
            uint32_t u = 0;
            for (uint32_t s = 0; s < Sb; ++s) u += part_uniq[first + s];
            out_uniq[b] = u;
        }
    }
}

}  // namespace fann
