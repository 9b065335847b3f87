// fann_next.cuh -- device code of the steps around the hot path:
//   lists_count_kernel / lists_scan_kernel / lists_expand_kernel
//                        step (3) on the GPU: posting-list metadata resident in HBM, candidate lists built
//                        from probed list indices
//   rerank_kernel<E>     step (8): heuristic re-ranking, Algorithm 1 / Eq. 3
//   page_reads_kernel    intra- / inter-mini-batch I/O dedup at page level, Fig. 8
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "fann_kernels.cuh"

namespace fann {

// ---------------------------------------------------------------- (3) candidate lists from resident metadata

struct ListsHeader {                                  // first 64 bytes of a fann_search_lists workspace
    unsigned long long total;                         // sum of the probed lists' lengths of the batch
    unsigned long long capacity;                      // max_total_cands of the call
    uint32_t overflow;                                // 1: total > capacity, nothing was expanded
    uint32_t pad[11];
};

// One warp per query: C_b = sum of the lengths of its probed lists.  A probe equal to 0xFFFFFFFF is padding and a
// probe >= n_lists names no list (R21).
__global__ void lists_count_kernel(const long long *__restrict__ list_offsets, uint64_t n_lists,
                                   const uint32_t *__restrict__ probes, uint32_t B, uint32_t nprobe,
                                   unsigned long long *__restrict__ per_query)
{
    const uint32_t b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (b >= B) return;
    unsigned long long s = 0;
    for (uint32_t j = lane; j < nprobe; j += 32) {
        const uint32_t l = __ldg(probes + (size_t)b * nprobe + j);
        if ((uint64_t)l < n_lists) s += (unsigned long long)(__ldg(list_offsets + l + 1) - __ldg(list_offsets + l));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) per_query[b] = s;
}

// Single CTA: cand_offsets[b] = exclusive prefix sum of per_query (in place: per_query and cand_offsets may be the
// same array of B + 1 entries), total and the capacity check into the header.
__global__ void lists_scan_kernel(const unsigned long long *per_query, uint32_t B, long long *cand_offsets,
                                  ListsHeader *hdr, unsigned long long capacity)
{
    __shared__ unsigned long long warp_sums[32];
    __shared__ unsigned long long running;
    if (threadIdx.x == 0) running = 0;
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (uint32_t base = 0; base < B; base += blockDim.x) {
        const uint32_t b = base + threadIdx.x;
        const unsigned long long v = b < B ? per_query[b] : 0ull;
        unsigned long long incl = v;
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long u = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += u;
        }
        if (lane == 31) warp_sums[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const unsigned long long w = warp_sums[lane];
            unsigned long long wi = w;
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned long long u = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += u;
            }
            warp_sums[lane] = wi - w;
        }
        __syncthreads();
        const unsigned long long start = running + warp_sums[warp] + incl - v;
        if (b < B) cand_offsets[b] = (long long)start;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) running = start + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        cand_offsets[B] = (long long)running;
        hdr->total = running;
        hdr->capacity = capacity;
        hdr->overflow = running > capacity ? 1u : 0u;
    }
}

constexpr int kExpandThreads = 256;

// One CTA per query (or several, for small batches): its probed lists' IDs concatenated in probe order at cand_ids + cand_offsets[b]
// (PAPER.md:L125 step (3)).  Dynamic shared memory: nprobe + 1 start positions.
__global__ void __launch_bounds__(kExpandThreads) lists_expand_kernel(const long long *__restrict__ list_offsets,
                                                                      const uint32_t *__restrict__ list_ids, uint64_t n_lists,
                                                                      const uint32_t *__restrict__ probes, uint32_t nprobe,
                                                                      const long long *__restrict__ cand_offsets,
                                                                      uint32_t *__restrict__ cand_ids, const ListsHeader *hdr,
                                                                      uint32_t ctas_per_query, uint32_t write_rows)
{
    extern __shared__ uint32_t start[];                           // [nprobe + 1] positions inside the query's list
    __shared__ uint32_t carry;
    if (hdr->overflow) return;                                    // the workspace cannot hold the batch: write nothing
    // small batches: several CTAs per query share its lists (CTA `sub` copies lists sub * 8 + warp, + 8 * ctas, ...)
    const uint32_t b = blockIdx.x / ctas_per_query, sub = blockIdx.x - b * ctas_per_query;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t *pr = probes + (size_t)b * nprobe;
    if (tid == 0) carry = 0;
    __syncthreads();
    __shared__ uint32_t wsum[kExpandThreads / 32];
    for (uint32_t base = 0; base < nprobe; base += kExpandThreads) {   // block exclusive scan of the list lengths
        const uint32_t j = base + tid;
        uint32_t len = 0;
        if (j < nprobe) {
            const uint32_t l = __ldg(pr + j);
            if ((uint64_t)l < n_lists) len = (uint32_t)(__ldg(list_offsets + l + 1) - __ldg(list_offsets + l));
        }
        uint32_t incl = len;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += u;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t woff = 0;
        for (uint32_t w = 0; w < warp; ++w) woff += wsum[w];
        if (j < nprobe) start[j] = carry + woff + incl - len;
        __syncthreads();
        if (tid == kExpandThreads - 1) carry += woff + incl;
        __syncthreads();
    }
    if (tid == 0) start[nprobe] = carry;
    __syncthreads();
    uint32_t *out = cand_ids + cand_offsets[b];
    for (uint32_t j = sub * (kExpandThreads / 32) + warp; j < nprobe; j += ctas_per_query * (kExpandThreads / 32)) {
        const uint32_t len = start[j + 1] - start[j];
        if (!len) continue;
        const long long l0 = __ldg(list_offsets + __ldg(pr + j));
        const uint32_t *src = list_ids + l0;
        uint32_t *dst = out + start[j];
        if (write_rows) {
            // list-major experiment: (the entry's position in list_ids = the row of the list-major code copy, its vector-ID)
            uint2 *dst2 = reinterpret_cast<uint2 *>(cand_ids) + cand_offsets[b] + start[j];
            for (uint32_t e = lane; e < len; e += 32) dst2[e] = make_uint2((uint32_t)l0 + e, __ldg(src + e));
            continue;
        }
        for (uint32_t e = lane; e < len; e += 32) dst[e] = __ldg(src + e);
    }
}

// ---------------------------------------------------------------- lists-direct: sorted lists + grid

constexpr uint32_t kSortMaxList = 8192;               // longest list lists_sort_grid_kernel sorts (in shared memory)

// fann_load_lists: one CTA per posting list.  Sorts the list's IDs ascending in place (set semantics: the order of a
// list's IDs carries no meaning) and writes its grid: grid[l][g] = position of the first ID >=
// grid_start(N, g), g = 0 .. kGridCells (the last entry = number of valid IDs; IDs >= N and padding sort behind it).
// A list longer than kSortMaxList is left as it is and *unsorted is raised (the direct path is then not used).
__global__ void __launch_bounds__(256) lists_sort_grid_kernel(const long long *__restrict__ list_offsets, uint32_t *list_ids,
                                                              uint64_t N, uint16_t *__restrict__ grid, uint32_t *unsorted)
{
    extern __shared__ uint32_t sm_ids[];
    const uint32_t l = blockIdx.x, tid = threadIdx.x;
    const long long o0 = list_offsets[l];
    const long long Lll = list_offsets[l + 1] - o0;
    uint16_t *g = grid + (size_t)l * (kGridCells + 1);
    if (Lll < 0 || Lll > (long long)kSortMaxList) {
        if (tid == 0) atomicExch(unsorted, 1u);
        if (tid <= kGridCells) g[tid] = 0;
        return;
    }
    const uint32_t L = (uint32_t)Lll;
    uint32_t P = 32;
    while (P < L) P <<= 1;
    for (uint32_t i = tid; i < P; i += 256) sm_ids[i] = i < L ? list_ids[o0 + i] : 0xFFFFFFFFu;
    __syncthreads();
    for (uint32_t size = 2; size <= P; size <<= 1)
        for (uint32_t stride = size >> 1; stride > 0; stride >>= 1) {
            for (uint32_t i = tid; i < (P >> 1); i += 256) {
                const uint32_t lo = 2 * i - (i & (stride - 1)), hi = lo + stride;
                const bool asc = (lo & size) == 0;
                const uint32_t x = sm_ids[lo], y = sm_ids[hi];
                if ((x > y) == asc) { sm_ids[lo] = y; sm_ids[hi] = x; }
            }
            __syncthreads();
        }
    for (uint32_t i = tid; i < L; i += 256) list_ids[o0 + i] = sm_ids[i];
    if (tid <= kGridCells) {
        const uint64_t bound = tid == kGridCells ? N : (uint64_t)grid_start(N, tid);
        uint32_t lo = 0, hi = L;                              // first position with id >= bound
        while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if ((uint64_t)sm_ids[mid] < bound) lo = mid + 1; else hi = mid; }
        g[tid] = (uint16_t)lo;
    }
}

// Lists-direct, one CTA per query, after plan_kernel fixed S_b (a power of two): the exact number of IDs of every
// ID-range class, from the grids of the probed lists.  Ordered placement if every class fits a dedup table even if
// none of its IDs repeats, else hash classes (which read whole lists).  bucket_cnt[item] = the class's ID count.
__global__ void __launch_bounds__(256) lists_classes_kernel(const uint16_t *__restrict__ grid, uint64_t n_lists, uint64_t N,
                                                            const uint32_t *__restrict__ probes, uint32_t nprobe,
                                                            const uint32_t *__restrict__ S, const uint32_t *__restrict__ item_start,
                                                            uint32_t class_max, uint32_t force, uint32_t *__restrict__ mode,
                                                            uint32_t *__restrict__ bucket_cnt)
{
    __shared__ uint32_t tot[kGridCells];
    const uint32_t b = blockIdx.x, tid = threadIdx.x, Sb = S[b];
    if (tid < kGridCells) tot[tid] = 0;
    __syncthreads();
    const bool can_order = Sb >= 1 && Sb <= kGridCells && (Sb & (Sb - 1)) == 0 && N >= 4096 && force != kModeHashed;
    if (can_order) {
        const uint32_t w = kGridCells / Sb;
        for (uint32_t j = tid; j < nprobe; j += 256) {
            const uint32_t l = __ldg(probes + (size_t)b * nprobe + j);
            if ((uint64_t)l >= n_lists) continue;
            const uint16_t *g = grid + (size_t)l * (kGridCells + 1);
            uint32_t prev = __ldg(g);
            for (uint32_t c = 0; c < Sb; ++c) {
                const uint32_t nxt = __ldg(g + (c + 1) * w);
                if (nxt > prev) atomicAdd(&tot[c], nxt - prev);
                prev = nxt;
            }
        }
    }
    __syncthreads();
    bool big = false;
    if (can_order && tid < Sb) {
        big = tot[tid] > class_max;
        bucket_cnt[item_start[b] + tid] = tot[tid];
    }
    big = __syncthreads_or(big);
    if (tid == 0) mode[b] = (can_order && (!big || force == kModeOrdered)) ? kModeOrdered : kModeHashed;
}

// List-major experiment: row e of the copy = the code row of the vector list entry e names (zero if it names none).
__global__ void list_codes_kernel(const uint8_t *__restrict__ codes, uint64_t N, uint32_t row_bytes,
                                  const uint32_t *__restrict__ list_ids, uint64_t e0, uint64_t n, uint8_t *__restrict__ dst)
{
    const uint32_t chunks = row_bytes >> 4;
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n * chunks) return;
    const uint64_t e = e0 + t / chunks;
    const uint32_t c = (uint32_t)(t % chunks);
    const uint32_t id = __ldg(list_ids + e);
    uint4 v = make_uint4(0, 0, 0, 0);
    if ((uint64_t)id < N) v = __ldg(reinterpret_cast<const uint4 *>(codes + (uint64_t)id * row_bytes) + c);
    reinterpret_cast<uint4 *>(dst + e * row_bytes)[c] = v;
}

// ---------------------------------------------------------------- (8) heuristic re-ranking, Algorithm 1

constexpr int kRerankThreads = 256;
constexpr uint32_t kRerankMaxK = 1024, kRerankMaxBatch = 1024, kRerankMaxTasks = 2048, kRerankMaxDim = 2048;

enum : int { kElemF32 = 0, kElemU8 = 1, kElemI8 = 2 };

template <int E> struct ElemT;
template <> struct ElemT<kElemF32> { using type = float; };
template <> struct ElemT<kElemU8> { using type = uint8_t; };
template <> struct ElemT<kElemI8> { using type = int8_t; };

struct RerankParams {
    const void *vectors;                              // [N][d] raw vectors, element type E
    uint64_t N;
    uint32_t d;
    const float *queries;                             // [B][d]
    const uint32_t *tasks;                            // [B][n] candidate IDs in ascending PQ order, 0xFFFFFFFF padded
    uint32_t n, batch_size, k, beta;
    float eps;
    uint32_t *out_ids;                                // [B][k]
    float *out_dists;                                 // [B][k]
    uint32_t *out_counts, *out_batches, *out_reads;   // [B] each; the last two may be NULL
};

// Exact squared L2 between the query (shared memory) and one raw vector, by one warp, fp32 (PAPER.md:L172
// "calculate the distances between the query vector and vectors within this mini-batch").
template <int E>
__device__ __forceinline__ float warp_sqdist(const float *q, const typename ElemT<E>::type *v, uint32_t d, uint32_t lane)
{
    float acc = 0.f;
    if ((d & 3u) == 0 && (reinterpret_cast<uintptr_t>(v) & (E == kElemF32 ? 15 : 3)) == 0) {
        for (uint32_t c = lane; c < (d >> 2); c += 32) {
            float x[4];
            if (E == kElemF32) {
                const float4 t = __ldg(reinterpret_cast<const float4 *>(v) + c);
                x[0] = t.x; x[1] = t.y; x[2] = t.z; x[3] = t.w;
            } else {
                const uint32_t t = __ldg(reinterpret_cast<const uint32_t *>(v) + c);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const uint32_t byte = (t >> (8 * i)) & 0xFFu;
                    x[i] = E == kElemU8 ? (float)byte : (float)(int)(int8_t)byte;
                }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) { const float dl = q[4 * c + i] - x[i]; acc = fmaf(dl, dl, acc); }
        }
    } else {
        for (uint32_t t = lane; t < d; t += 32) { const float dl = q[t] - (float)v[t]; acc = fmaf(dl, dl, acc); }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    return acc;
}

// One CTA per query.  Q of Algorithm 1 is kept as a sorted array of 64-bit keys (distance bits << 32 | position in
// Tasks): at all times the k smallest keys of the tasks seen so far, which is what the paper's max-heap with a
// strict "<" on insertion holds (R24).  A mini-batch: the warps compute the exact distances, then every
// old and new key finds its rank in the union by counting smaller keys, the k smallest are written in rank order,
// Delta = (new keys among them) / k (Eq. 3: members of S_n that are not in S_{n-1} are exactly those), and thread 0
// advances the StabilityCounter.  Mini-batches after the stop are never read -- the point of the heuristic.
// Shared memory: query d floats | tasks n | Q two buffers of k keys | new keys batch_size.
template <int E>
__global__ void __launch_bounds__(kRerankThreads) rerank_kernel(const RerankParams p)
{
    using T = typename ElemT<E>::type;
    extern __shared__ __align__(16) unsigned char smem[];
    float *q = reinterpret_cast<float *>(smem);
    uint32_t *tasks = reinterpret_cast<uint32_t *>(q + ((p.d + 3u) & ~3u));
    unsigned long long *Qa = reinterpret_cast<unsigned long long *>(tasks + ((p.n + 3u) & ~3u));
    unsigned long long *Qb = Qa + p.k;
    unsigned long long *fresh = Qb + p.k;
    __shared__ uint32_t s_ntasks, s_changed, s_reads, s_stop, s_valid;
    const uint32_t b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) { s_ntasks = p.n; s_reads = 0; s_stop = 0; }
    __syncthreads();
    for (uint32_t t = tid; t < p.d; t += kRerankThreads) q[t] = p.queries[(size_t)b * p.d + t];
    for (uint32_t j = tid; j < p.n; j += kRerankThreads) {
        const uint32_t id = p.tasks[(size_t)b * p.n + j];
        tasks[j] = id;
        if (id == kIdNone) atomicMin(&s_ntasks, j);                // padding ends the task list
    }
    __syncthreads();
    const uint32_t n_tasks = s_ntasks;
    const T *vec = reinterpret_cast<const T *>(p.vectors);
    uint32_t cur = 0, stability = 0, batches = 0;                  // |Q|; uniform across the CTA
    unsigned long long *Q = Qa, *Qn = Qb;
    for (uint32_t i = 0; i < n_tasks; i += p.batch_size) {         // Algorithm 1 line 3
        const uint32_t m = min(p.batch_size, n_tasks - i);
        if (tid == 0) { s_changed = 0; s_valid = 0; }
        __syncthreads();
        for (uint32_t jj = warp; jj < m; jj += kRerankThreads / 32) {   // lines 5-6: GetDistance
            const uint32_t id = tasks[i + jj];
            unsigned long long key = kKeyMax;
            if ((uint64_t)id < p.N) {
                const float dist = warp_sqdist<E>(q, vec + (size_t)id * p.d, p.d, lane);
                key = ((unsigned long long)__float_as_uint(dist) << 32) | (i + jj);
            }
            if (lane == 0) {
                fresh[jj] = key;
                if (key != kKeyMax) atomicAdd(&s_valid, 1u);
            }
        }
        __syncthreads();
        // line 7, all insertions of the mini-batch at once: rank of every key in Q + fresh
        for (uint32_t t = tid; t < cur + m; t += kRerankThreads) {
            const bool is_new = t >= cur;
            const unsigned long long key = is_new ? fresh[t - cur] : Q[t];
            if (key == kKeyMax) continue;
            uint32_t rank = is_new ? 0u : t;
            if (is_new) for (uint32_t s = 0; s < cur; ++s) rank += Q[s] < key ? 1u : 0u;
            for (uint32_t s = 0; s < m; ++s) rank += fresh[s] < key ? 1u : 0u;
            if (rank < p.k) {
                Qn[rank] = key;
                if (is_new) atomicAdd(&s_changed, 1u);
            }
        }
        __syncthreads();
        cur = min(p.k, cur + s_valid);
        { unsigned long long *t = Q; Q = Qn; Qn = t; }
        ++batches;
        if (tid == 0) {                                            // lines 9-18
            s_reads += s_valid;
            const double delta = (double)s_changed / (double)p.k;
            if (delta < (double)p.eps) { if (++stability >= p.beta) s_stop = 1; }
            else stability = 0;
        }
        __syncthreads();
        if (s_stop) break;
    }
    for (uint32_t s = tid; s < p.k; s += kRerankThreads) {         // line 20: return Q (ascending)
        const bool have = s < cur;
        const unsigned long long key = have ? Q[s] : kKeyMax;
        p.out_ids[(size_t)b * p.k + s] = have ? tasks[(uint32_t)key] : kIdNone;
        p.out_dists[(size_t)b * p.k + s] = have ? __uint_as_float((uint32_t)(key >> 32)) : __int_as_float(0x7f800000);
    }
    if (tid == 0) {
        p.out_counts[b] = cur;
        if (p.out_batches) p.out_batches[b] = batches;
        if (p.out_reads) p.out_reads[b] = s_reads;
    }
}

// ---------------------------------------------------------------- page-level I/O dedup, Fig. 8

constexpr int kPageThreads = 256;
constexpr uint32_t kPageMaxTasks = 4096;

struct PageParams {
    const uint32_t *page_of;                          // [N] vector -> SSD page
    uint64_t N, n_pages;
    const uint32_t *tasks;                            // [B][n]
    uint32_t n, batch_size, n_batches;                // n_batches = ceil(n / batch_size)
    const uint32_t *batches_run;                      // [B] mini-batches Algorithm 1 executed (0 = all), or NULL
    const uint32_t *resident;                         // bitmap over pages already in the DRAM buffer, or NULL
    uint32_t *out_pages;                              // [B][n] pages to read, mini-batch after mini-batch, 0xFFFFFFFF padded
    uint32_t *out_batch_reads;                        // [B][n_batches]
    uint32_t *out_total;                              // [B]
};

// One CTA per query; mini-batches in order.  The DRAM buffer of the query is a shared-memory hash
// set of page numbers that persists across its mini-batches: the thread whose compare-and-swap installs a page is
// the one that reads it, so a page is read once per query whatever the number of tasks that need it ("merging I/Os
// mapped to the same SSD page within a mini-batch" and "the DRAM buffer ... in subsequent mini-batches").
// Dynamic shared memory: slots (power of two >= 2 n) words.
__global__ void __launch_bounds__(kPageThreads) page_reads_kernel(const PageParams p, uint32_t slots)
{
    extern __shared__ uint32_t set[];
    __shared__ uint32_t s_ntasks, s_count;
    const uint32_t b = blockIdx.x, tid = threadIdx.x;
    for (uint32_t s = tid; s < slots; s += kPageThreads) set[s] = kEmpty;
    if (tid == 0) { s_ntasks = p.n; s_count = 0; }
    __syncthreads();
    const uint32_t *tasks = p.tasks + (size_t)b * p.n;
    for (uint32_t j = tid; j < p.n; j += kPageThreads)
        if (__ldg(tasks + j) == kIdNone) atomicMin(&s_ntasks, j);
    __syncthreads();
    const uint32_t n_tasks = s_ntasks;
    const uint32_t limit = p.batches_run ? p.batches_run[b] : 0u;
    uint32_t *out = p.out_pages + (size_t)b * p.n;
    uint32_t prev = 0;
    for (uint32_t t = 0; t < p.n_batches; ++t) {
        const uint32_t i = t * p.batch_size;
        const bool run = i < n_tasks && (limit == 0 || t < limit);
        if (run) {
            const uint32_t m = min(p.batch_size, n_tasks - i);
            for (uint32_t jj = tid; jj < m; jj += kPageThreads) {
                const uint32_t id = __ldg(tasks + i + jj);
                if ((uint64_t)id >= p.N) continue;
                const uint32_t pg = __ldg(p.page_of + id);
                if (p.resident && (uint64_t)pg < p.n_pages && ((__ldg(p.resident + (pg >> 5)) >> (pg & 31)) & 1u)) continue;
                uint32_t h = pg * 0x9E3779B1u;
                uint32_t slot = (h ^ (h >> 15)) & (slots - 1);
                for (;;) {
                    const uint32_t old = atomicCAS(&set[slot], kEmpty, pg);
                    if (old == kEmpty) { out[atomicAdd(&s_count, 1u)] = pg; break; }   // this thread reads the page
                    if (old == pg) break;                          // already read (this mini-batch or an earlier one)
                    slot = (slot + 1) & (slots - 1);
                }
            }
        }
        __syncthreads();
        if (tid == 0) { p.out_batch_reads[(size_t)b * p.n_batches + t] = s_count - prev; }
        prev = s_count;
        __syncthreads();
    }
    const uint32_t total = s_count;
    for (uint32_t s = total + tid; s < p.n; s += kPageThreads) out[s] = kIdNone;
    if (tid == 0) p.out_total[b] = total;
}

}  // namespace fann
