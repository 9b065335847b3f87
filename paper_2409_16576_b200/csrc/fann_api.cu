// fann_api.cu -- the C ABI of include/fann.h: argument checks, workspace
// layout, launch geometry, kernel launches.  No compute happens on the host.
#include "../../include/fann.h"
#include "fann_kernels.cuh"
#include "fann_next.cuh"

#include <atomic>
#include <condition_variable>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

using namespace fann;

// What one call needs besides the caller's stream: a second stream and events for the transfer / partition overlap.
// Calls take one from the index's pool and give it back on return, so concurrent calls on one handle (different
// host threads, streams and workspaces; "each CPU thread handles an individual query") never share
// an event between a record and its wait.
struct CallCtx {
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_done[kMaxChunks] = {};
};

struct fann_index {
    int device = 0;
    uint64_t N = 0;
    uint32_t M = 0, row_bytes = 0;
    uint8_t *codes = nullptr;              // [N][row_bytes]
    uint8_t *bounce = nullptr;             // staging for host-sourced code chunks
    size_t bounce_bytes = 0;
    // posting-list metadata, raw vectors and the vector -> page table, each optional
    long long *list_offsets = nullptr;     // [n_lists + 1]
    uint32_t *list_ids = nullptr;          // [list_entries]
    uint64_t n_lists = 0, list_entries = 0;
    void *vectors = nullptr;               // [vec_N][vec_d] of vec_elem
    uint64_t vec_N = 0;
    uint32_t vec_d = 0;
    int vec_elem = 0;
    uint16_t *list_grid = nullptr;         // [n_lists][kGridCells + 1]: sorted lists' positions of the ID-range cells
    bool lists_sorted = false;             // every list was sorted and indexed at load (lists-direct path possible)
    bool lists_direct = true;              // FANN_LISTS_DIRECT=0: always expand + split (the path of unsorted lists)
    uint8_t *lm_codes = nullptr;           // list-major experiment: [list_entries][row_bytes], row e = code of list_ids[e]
    uint32_t *page_of = nullptr;           // [page_N]
    uint64_t page_N = 0, n_pages = 0;
    int num_sms = 0;
    int smem_optin = 0;                    // max dynamic shared memory per block
    uint32_t chunks = 1;                   // batch chunks (FANN_CHUNKS): partition of chunk i+1 runs beside the scan of chunk i
    uint32_t force_mode = 2;               // dedup placement: 0 ordered, 1 hashed, 2 decided per query (FANN_DEDUP_MODE)
    uint32_t scan_ring = 3;                // scan kernel: stages of the per-warp code-row ring, 0 = rows through registers (FANN_SCAN_RING)
    bool partition = true;                 // split lists into their dedup classes first (FANN_PARTITION=0: filter per pass)
    bool host_direct = true;               // host entries: kernels write results straight into pinned host output arrays (FANN_HOST_DIRECT=0: staged + copied)
    bool split_scan = true;                // several scan CTAs per query when the batch is smaller than the machine (FANN_SPLIT_SCAN=0: one)
    uint32_t dedup_smem = 0;               // dynamic shared memory of a dedup CTA
    uint32_t dedup_smem_half = 0;          // same for two CTAs per SM
    uint32_t dedup_threads = 0;            // 0: chosen per call (geometry()); 1024 or 512: forced (FANN_DEDUP_THREADS)
    void *static_ws = nullptr;             // device address of g_static_ws on this device (fann_dedup_scan_topk_static), resolved in fann_create
    cudaError_t static_ws_err = cudaSuccess;
    std::atomic<uint64_t> launches{0};
    std::atomic<uint32_t> generation{0};   // bumped by the loaders: captured graphs (fann_pool) hold the arrays' addresses
    // everything below is shared by concurrent callers and guarded by `mu`
    std::mutex mu;
    std::vector<CallCtx *> ctx_pool;       // idle call contexts
    // geometry of the last launches (fann_get_info)
    uint32_t last_dedup_threads = 1024, last_dedup_smem = 0, last_dedup_ctas = 0, last_scan_ctas = 0, last_scan_smem = 0, last_cap = 0, last_slots = 0, last_chunks = 0;
    // optional per-kernel timing (benchmarks; timed calls are serialised by `timing_mu`)
    std::mutex timing_mu;
    std::atomic<bool> timing{false};
    cudaEvent_t ev_lut[2] = {}, ev_plan[2] = {}, ev_part[2] = {}, ev_dedup[kMaxChunks][2] = {}, ev_scan[kMaxChunks][2] = {};
    bool have_lut = false, have_scan = false, have_part = false;
    uint32_t timed_chunks = 0;
    bool timed_scan = false;
};

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                      \
    do {                                                                                    \
        cudaError_t e__ = (expr);                                                           \
        if (e__ != cudaSuccess)                                                             \
            return fail(e__ == cudaErrorMemoryAllocation ? FANN_ENOMEM : FANN_ECUDA,        \
                        "%s: %s", #expr, cudaGetErrorString(e__));                          \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static void destroy_ctx(CallCtx *c)
{
    if (!c) return;
    if (c->side) cudaStreamDestroy(c->side);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    for (auto &e : c->ev_done) if (e) cudaEventDestroy(e);
    delete c;
}

// RAII: a call context from the index's pool (created on first use), returned on scope exit.
struct CtxLease {
    fann_index *ix;
    CallCtx *c = nullptr;
    explicit CtxLease(fann_index *ix_) : ix(ix_)       // ix_ == NULL: the call needs no second stream
    {
        if (!ix) return;
        {
            std::lock_guard<std::mutex> g(ix->mu);
            if (!ix->ctx_pool.empty()) { c = ix->ctx_pool.back(); ix->ctx_pool.pop_back(); }
        }
        if (c) return;
        c = new CallCtx();
        bool ok = cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) == cudaSuccess;
        for (auto &e : c->ev_done) ok = ok && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
        if (!ok) { destroy_ctx(c); c = nullptr; }
    }
    ~CtxLease()
    {
        if (!c) return;
        std::lock_guard<std::mutex> g(ix->mu);
        ix->ctx_pool.push_back(c);
    }
};

// ---------------------------------------------------------------- the no-allocation entry's workspace

// fann_dedup_scan_topk_static: the workspace of the path as a file-scope device array (fann.h).  In host code the
// name g_static_ws is a host-side stand-in of the symbol, NOT a device address: the address the kernels get comes
// from cudaGetSymbolAddress, asked once per device with that device current (fann_create) and kept here.
static __device__ __align__(256) unsigned char g_static_ws[FANN_STATIC_WS_BYTES];

constexpr int kMaxDevices = 64;
static std::mutex g_static_mu;
static void *g_static_ptr[kMaxDevices] = {};

// The calling thread's current device must be `device`.
static cudaError_t static_ws_resolve(int device, void **out)
{
    *out = nullptr;
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[device]) {
        void *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_static_ws);
        if (e != cudaSuccess) return e;
        g_static_ptr[device] = ptr;
    }
    *out = g_static_ptr[device];
    return cudaSuccess;
}

// ---------------------------------------------------------------- geometry + workspace layout

struct Geom {
    uint32_t nslots_max, cap_c, dedup_smem, dedup_threads;   // dedup: table slots per CTA, candidates per partition, CTA shape
    uint32_t cap, scan_smem, ring;                   // scan: candidate-buffer keys, shared memory per CTA, ring depth
    uint32_t parts, k;                               // scan CTAs per query (> 1 for batches smaller than the machine), k
    uint32_t part_ctas;                              // partition CTAs per query (> 1 for small batches)
    uint32_t min_classes;                            // lists-direct: at least this many ID-range classes per query (small batches)
};

// Dedup CTA shape: one 1024-thread CTA per SM with the whole shared memory as its table, or -- when the mean candidate
// list needs two or more partitions anyway -- two 512-thread CTAs per SM with half the table each, so that one computes
// while the other waits at a barrier (partition_kernel makes the number of partitions free: each ID is read once).
static void geometry(const fann_index *ix, uint32_t k, uint32_t B, uint64_t total_cands, Geom *g, uint32_t shape = 0,
                     bool allow_split = true, bool ld = false)
{
    const uint32_t ldb = ld ? dedup_ld_bytes() : 0u;           // lists-direct: the segment table sits before the dedup table
    g->dedup_threads = 1024; g->dedup_smem = ix->dedup_smem;
    g->nslots_max = ((g->dedup_smem - dedup_table_off(1024) - ldb) / 4) & ~3u;
    g->cap_c = (uint32_t)((uint64_t)g->nslots_max * 3 / 4);      // <= 75 % load even with no repeats
    const uint64_t mean_c = total_cands / (B ? B : 1);
    const bool split = shape ? shape == 512
                             : (ix->dedup_threads == 512 || (ix->dedup_threads == 0 && (ix->partition || ld) && mean_c > g->cap_c));
    if (split && ix->dedup_smem_half >= 32768) {
        g->dedup_threads = 512; g->dedup_smem = ix->dedup_smem_half;
        g->nslots_max = ((g->dedup_smem - dedup_table_off(512) - ldb) / 4) & ~3u;
        g->cap_c = (uint32_t)((uint64_t)g->nslots_max * 3 / 4);
    }
    g->ring = ix->scan_ring;
    // a batch of fewer queries than half the SMs: several scan CTAs per query, each on a slice of the query's
    // distinct list, merged by merge_parts_kernel (at most 16 parts: 16 k keys fit the merge CTA's shared memory)
    g->k = k;
    g->parts = 1;
    if (ix->split_scan && allow_split && 2 * B <= (uint32_t)ix->num_sms) {
        const uint32_t fit = (uint32_t)ix->num_sms / B;
        g->parts = fit >= 16 ? 16u : fit >= 8 ? 8u : fit >= 4 ? 4u : 2u;   // a power of two (pairwise merge)
    }
    g->part_ctas = 1;
    if (ix->split_scan && allow_split)
        while (g->part_ctas < 16 && 2 * g->part_ctas * B <= (uint32_t)ix->num_sms) g->part_ctas <<= 1;
    // lists-direct, small batch: more (smaller) ID-range classes per query than its size asks for, so that one query's
    // dedup spreads over the machine like its scan does (a class is a run of the 64 grid cells: a power of two)
    g->min_classes = 1;
    if (ld && ix->split_scan && allow_split)
        while (g->min_classes < 32 && g->min_classes * B <= (uint32_t)ix->num_sms) g->min_classes <<= 1;
    g->cap = (k <= 256 || g->ring) ? 4096u : 8192u;            // the ring takes the shared memory of the larger buffer
    g->scan_smem = (uint32_t)scan_smem_bytes(g->cap, g->ring);
}

struct WsLayout {
    size_t hdr, S, mode, item_start, items, uniq_counts, part_ok, part_aux, bucket_cnt, part_keys, part_ids, uniq_ids, total;
    uint32_t max_items;
};

static void ws_layout(uint32_t B, uint64_t total_cands, const Geom &g, bool with_uniq, WsLayout *w)
{
    const uint64_t max_items = 2 * ((uint64_t)B + total_cands / g.cap_c + 1) +  // x2: the lists-direct path rounds S_b up to a power of two
                               (uint64_t)B * (g.min_classes > 1 ? g.min_classes : 0u);
    w->max_items = (uint32_t)(max_items > 0xFFFFFFF0ull ? 0xFFFFFFF0ull : max_items);
    size_t o = 0;
    w->hdr = o;         o = align_up(o + 256, 256);
    w->S = o;           o = align_up(o + (size_t)B * 4, 256);
    w->mode = o;        o = align_up(o + (size_t)B * 4, 256);
    w->item_start = o;  o = align_up(o + ((size_t)B + 1) * 4, 256);
    w->items = o;       o = align_up(o + (size_t)w->max_items * 8, 256);
    w->uniq_counts = o; o = align_up(o + (size_t)B * 4, 256);
    w->part_ok = o;     o = align_up(o + (size_t)B * 4, 256);
    w->part_aux = o;    o = align_up(o + (size_t)B * 8, 256);        // partition_multi_kernel: arrivals, failure flag
    w->bucket_cnt = o;  o = align_up(o + (size_t)w->max_items * 4, 256);
    w->part_keys = o;   if (g.parts > 1) o = align_up(o + (size_t)B * g.parts * g.k * 8, 256);   // partial top-k of the scan parts
    w->part_ids = o;    o = align_up(o + (size_t)total_cands * 8 + 16, 256);      // class buckets, 2 C_b per query
    w->uniq_ids = o;    if (with_uniq) o = align_up(o + (size_t)total_cands * 4 + 16, 256);
    w->total = o;
}

// ---------------------------------------------------------------- lifecycle

extern "C" const char *fann_last_error(void) { return g_err; }
extern "C" const char *fann_version(void) { return "fann 0.3 sm_100a"; }

template <int G, int NB, int D, bool LM = false>
static cudaError_t set_scan_attr(int smem)
{
    return cudaFuncSetAttribute(scan_kernel<G, NB, D, LM>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
}

extern "C" int fann_create(fann_index **out, int device)
{
    if (!out) return fail(FANN_EINVAL, "fann_create: out is NULL");
    *out = nullptr;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0)
        return fail(FANN_ECUDA, "fann_create: no CUDA device (%s); there is no CPU fallback",
                    e != cudaSuccess ? cudaGetErrorString(e) : "count 0");
    if (device < 0 || device >= n) return fail(FANN_EINVAL, "fann_create: device %d of %d", device, n);
    DeviceGuard guard(device);
    int num_sms = 0, smem_optin = 0;
    CUDA_TRY(cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, device));
    CUDA_TRY(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device));
    const int scan_max = (int)scan_smem_bytes(8192);
    if (scan_max > smem_optin)
        return fail(FANN_EUNSUPPORTED, "fann_create: device offers %d bytes of shared memory per block, %d needed",
                    smem_optin, scan_max);
    CUDA_TRY((cudaFuncSetAttribute(dedup_kernel<1024, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)));
    CUDA_TRY((cudaFuncSetAttribute(dedup_kernel<512, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)));
    CUDA_TRY((cudaFuncSetAttribute(dedup_kernel<1024, 8, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)));
    CUDA_TRY((cudaFuncSetAttribute(dedup_kernel<512, 8, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)));
    const int ring_max = (int)scan_smem_bytes(4096, 3);
    if (ring_max > smem_optin)
        return fail(FANN_EUNSUPPORTED, "fann_create: device offers %d bytes of shared memory per block, %d needed",
                    smem_optin, ring_max);
    CUDA_TRY((set_scan_attr<1, 4, 0>(scan_max)));
    CUDA_TRY((set_scan_attr<2, 4, 0>(scan_max)));
    CUDA_TRY((set_scan_attr<4, 2, 0>(scan_max)));
    CUDA_TRY((set_scan_attr<1, 4, 3>(ring_max)));
    CUDA_TRY((set_scan_attr<2, 4, 3>(ring_max)));
    CUDA_TRY((set_scan_attr<4, 2, 3>(ring_max)));
    CUDA_TRY((set_scan_attr<1, 4, 3, true>(ring_max)));
    CUDA_TRY((set_scan_attr<2, 4, 3, true>(ring_max)));
    CUDA_TRY((set_scan_attr<4, 2, 3, true>(ring_max)));
    CUDA_TRY(cudaFuncSetAttribute(merge_parts_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 16384 * 8));
    int per_sm = 0;
    CUDA_TRY(cudaDeviceGetAttribute(&per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, device));
    fann_index *ix = new fann_index();
    ix->device = device; ix->num_sms = num_sms; ix->smem_optin = smem_optin;
    ix->static_ws_err = static_ws_resolve(device, &ix->static_ws);     // `device` is current (guard above)
    if (ix->static_ws_err != cudaSuccess) cudaGetLastError();          // only fann_dedup_scan_topk_static needs it: it reports
    ix->dedup_smem = (uint32_t)smem_optin;
    // two dedup CTAs per SM: each gets half of the SM's shared memory less the 1 KB the driver reserves per CTA
    ix->dedup_smem_half = (uint32_t)((per_sm / 2 - 1024) & ~255);
    // A/B knobs (DESIGN.md 6.4 "Knobs"); the defaults are the product, tests run every alternative
    if (const char *s = getenv("FANN_CHUNKS")) { int v = atoi(s); if (v >= 1 && v <= kMaxChunks) ix->chunks = (uint32_t)v; }
    if (const char *s = getenv("FANN_DEDUP_MODE")) { int v = atoi(s); if (v == 0 || v == 1) ix->force_mode = (uint32_t)v; }
    if (const char *s = getenv("FANN_PARTITION")) ix->partition = atoi(s) != 0;
    if (const char *s = getenv("FANN_SPLIT_SCAN")) ix->split_scan = atoi(s) != 0;
    if (const char *s = getenv("FANN_HOST_DIRECT")) ix->host_direct = atoi(s) != 0;
    if (const char *s = getenv("FANN_LISTS_DIRECT")) ix->lists_direct = atoi(s) != 0;
    if (const char *s = getenv("FANN_SCAN_RING")) { int v = atoi(s); if (v == 0 || v == 3) ix->scan_ring = (uint32_t)v; }
    if (const char *s = getenv("FANN_DEDUP_THREADS")) { int v = atoi(s); if (v == 512 || v == 1024) ix->dedup_threads = (uint32_t)v; }
    *out = ix;
    return FANN_OK;
}

extern "C" void fann_destroy(fann_index *ix)
{
    if (!ix) return;
    DeviceGuard guard(ix->device);
    cudaDeviceSynchronize();
    if (ix->codes) cudaFree(ix->codes);
    if (ix->bounce) cudaFree(ix->bounce);
    if (ix->list_offsets) cudaFree(ix->list_offsets);
    if (ix->list_ids) cudaFree(ix->list_ids);
    if (ix->vectors) cudaFree(ix->vectors);
    if (ix->page_of) cudaFree(ix->page_of);
    if (ix->lm_codes) cudaFree(ix->lm_codes);
    if (ix->list_grid) cudaFree(ix->list_grid);
    for (CallCtx *c : ix->ctx_pool) destroy_ctx(c);
    for (auto &e : ix->ev_lut) if (e) cudaEventDestroy(e);
    for (auto &e : ix->ev_plan) if (e) cudaEventDestroy(e);
    for (auto &e : ix->ev_part) if (e) cudaEventDestroy(e);
    for (auto &c : ix->ev_dedup) for (auto &e : c) if (e) cudaEventDestroy(e);
    for (auto &c : ix->ev_scan) for (auto &e : c) if (e) cudaEventDestroy(e);
    delete ix;
}

extern "C" int fann_get_info(const fann_index *ix, fann_info *out)
{
    if (!ix || !out) return fail(FANN_EINVAL, "fann_get_info: NULL argument");
    std::lock_guard<std::mutex> g(const_cast<fann_index *>(ix)->mu);
    out->codes_device_ptr = (uint64_t)(uintptr_t)ix->codes;
    out->reserved = 0;
    out->N = ix->N; out->M = ix->M; out->row_bytes = ix->row_bytes;
    out->num_sms = (uint32_t)ix->num_sms;
    out->dedup_threads = ix->last_dedup_threads; out->dedup_ctas = ix->last_dedup_ctas;
    out->dedup_smem_bytes = ix->last_dedup_smem; out->table_slots = ix->last_slots;
    out->scan_threads = kScanThreads; out->scan_ctas = ix->last_scan_ctas;
    out->scan_smem_bytes = ix->last_scan_smem; out->scan_buffer_keys = ix->last_cap;
    out->chunks = ix->last_chunks;
    out->kernel_launches = ix->launches.load();
    return FANN_OK;
}

// ---------------------------------------------------------------- fann_load_codes

static uint32_t stored_row_bytes(uint32_t M) { return M <= 16 ? 16u : (M <= 32 ? 32u : 64u); }

extern "C" int fann_load_codes(fann_index *ix, const uint8_t *codes, uint64_t first, uint64_t n,
                               uint64_t N_total, uint32_t M, int src_is_device, void *stream_)
{
    if (!ix || !codes) return fail(FANN_EINVAL, "fann_load_codes: NULL argument");
    if (M == 0 || N_total == 0) return fail(FANN_EINVAL, "fann_load_codes: M and N_total must be > 0");
    if (M > FANN_MAX_M) return fail(FANN_EUNSUPPORTED, "fann_load_codes: M=%u > %u", M, FANN_MAX_M);
    if (N_total >= 0xFFFFFFFFull) return fail(FANN_EUNSUPPORTED, "fann_load_codes: N_total must be < 2^32-1");
    if (first > N_total || n > N_total - first) return fail(FANN_EINVAL, "fann_load_codes: rows [%llu,+%llu) outside N_total=%llu",
                                                            (unsigned long long)first, (unsigned long long)n, (unsigned long long)N_total);
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    ix->generation++;
    if (!ix->codes) {
        ix->N = N_total; ix->M = M; ix->row_bytes = stored_row_bytes(M);
        cudaError_t e = cudaMalloc(&ix->codes, (size_t)N_total * ix->row_bytes);
        if (e != cudaSuccess) {
            ix->codes = nullptr; ix->N = 0; ix->M = 0;
            return fail(FANN_ENOMEM, "fann_load_codes: cudaMalloc(%zu): %s", (size_t)N_total * ix->row_bytes, cudaGetErrorString(e));
        }
    } else if (N_total != ix->N || M != ix->M) {
        return fail(FANN_EINVAL, "fann_load_codes: (N_total, M) = (%llu, %u) differs from the first call (%llu, %u)",
                    (unsigned long long)N_total, M, (unsigned long long)ix->N, ix->M);
    }
    if (n == 0) return FANN_OK;
    uint8_t *dst = ix->codes + (size_t)first * ix->row_bytes;
    const uint32_t chunks = ix->row_bytes >> 4;
    if (src_is_device) {
        if (M == ix->row_bytes) {
            CUDA_TRY(cudaMemcpyAsync(dst, codes, (size_t)n * M, cudaMemcpyDeviceToDevice, stream));
        } else {
            const uint64_t rows_per_launch = 1ull << 26;
            for (uint64_t r0 = 0; r0 < n; r0 += rows_per_launch) {
                uint64_t nr = n - r0 < rows_per_launch ? n - r0 : rows_per_launch;
                uint64_t threads = nr * chunks;
                repack_rows_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, stream>>>(
                    codes + r0 * M, dst + r0 * ix->row_bytes, nr, M, ix->row_bytes);
                ix->launches++;
            }
            CUDA_TRY(cudaGetLastError());
        }
        return FANN_OK;
    }
    // host source: through a device bounce buffer, chunk by chunk
    if (M == ix->row_bytes) {
        CUDA_TRY(cudaMemcpyAsync(dst, codes, (size_t)n * M, cudaMemcpyHostToDevice, stream));
        CUDA_TRY(cudaStreamSynchronize(stream));
        return FANN_OK;
    }
    const size_t want = 64u << 20;
    if (!ix->bounce) {
        CUDA_TRY(cudaMalloc(&ix->bounce, want));
        ix->bounce_bytes = want;
    }
    const uint64_t rows_per = ix->bounce_bytes / M;
    for (uint64_t r0 = 0; r0 < n; r0 += rows_per) {
        uint64_t nr = n - r0 < rows_per ? n - r0 : rows_per;
        CUDA_TRY(cudaMemcpyAsync(ix->bounce, codes + r0 * M, (size_t)nr * M, cudaMemcpyHostToDevice, stream));
        uint64_t threads = nr * chunks;
        repack_rows_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, stream>>>(
            ix->bounce, dst + r0 * ix->row_bytes, nr, M, ix->row_bytes);
        ix->launches++;
        CUDA_TRY(cudaGetLastError());
        CUDA_TRY(cudaStreamSynchronize(stream));
    }
    return FANN_OK;
}

// ---------------------------------------------------------------- (1) fann_build_lut

extern "C" int fann_build_lut(fann_index *ix, const float *queries, uint32_t B,
                              const float *codebooks, uint32_t dsub, float *lut, void *stream_)
{
    if (!ix || !queries || !codebooks || !lut) return fail(FANN_EINVAL, "fann_build_lut: NULL argument");
    if (!ix->codes) return fail(FANN_EINVAL, "fann_build_lut: load codes first (M is unknown)");
    if (B == 0) return fail(FANN_EINVAL, "fann_build_lut: B == 0");
    if (dsub == 0 || dsub > 64) return fail(FANN_EUNSUPPORTED, "fann_build_lut: dsub=%u not in 1..64", dsub);
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    const uint64_t blocks = (uint64_t)B * ((ix->M + 3) / 4);
    if (blocks > 0x7FFFFFFFull) return fail(FANN_EUNSUPPORTED, "fann_build_lut: B=%u too large for one launch", B);
    if (((uintptr_t)lut & 15) != 0) return fail(FANN_EINVAL, "fann_build_lut: lut must be 16-byte aligned");
    if ((((uintptr_t)queries | (uintptr_t)codebooks) & 3) != 0)
        return fail(FANN_EINVAL, "fann_build_lut: queries and codebooks must be 4-byte aligned");
    const bool vec = (((uintptr_t)codebooks | (uintptr_t)queries) & 15) == 0;   // float4 reads of the codebook
    const bool timing = ix->timing.load();
    std::unique_lock<std::mutex> tl(ix->timing_mu, std::defer_lock);
    if (timing) tl.lock();
    if (timing) cudaEventRecord(ix->ev_lut[0], stream);
    if (vec && dsub == 2) build_lut_kernel<2><<<(unsigned)blocks, 256, 0, stream>>>(queries, codebooks, lut, ix->M, dsub);
    else if (vec && dsub == 4) build_lut_kernel<4><<<(unsigned)blocks, 256, 0, stream>>>(queries, codebooks, lut, ix->M, dsub);
    else if (vec && dsub == 8) build_lut_kernel<8><<<(unsigned)blocks, 256, 0, stream>>>(queries, codebooks, lut, ix->M, dsub);
    else build_lut_kernel<0><<<(unsigned)blocks, 256, 0, stream>>>(queries, codebooks, lut, ix->M, dsub);
    if (timing) { cudaEventRecord(ix->ev_lut[1], stream); ix->have_lut = true; }
    ix->launches++;
    CUDA_TRY(cudaGetLastError());
    return FANN_OK;
}

// ---------------------------------------------------------------- (5)(6)(7)

extern "C" size_t fann_workspace_bytes(const fann_index *ix, uint32_t B, uint64_t total_cands, uint32_t k)
{
    if (!ix || !ix->codes) { fail(FANN_EINVAL, "fann_workspace_bytes: index has no codes"); return 0; }
    if (B == 0 || k == 0 || k > FANN_MAX_K) { fail(FANN_EINVAL, "fann_workspace_bytes: B=%u k=%u", B, k); return 0; }
    Geom g;
    geometry(ix, k, B, total_cands, &g);
    WsLayout w;
    ws_layout(B, total_cands, g, true, &w);
    return w.total;
}

static cudaError_t launch_scan(const fann_index *ix, int grid, size_t smem, cudaStream_t stream, const ScanParams &p)
{
    if (p.key_src) {                                           // list-major experiment (ring only)
        switch (ix->row_bytes) {
        case 16: scan_kernel<1, 4, 3, true><<<grid, kScanThreads, smem, stream>>>(p); break;
        case 32: scan_kernel<2, 4, 3, true><<<grid, kScanThreads, smem, stream>>>(p); break;
        default: scan_kernel<4, 2, 3, true><<<grid, kScanThreads, smem, stream>>>(p); break;
        }
        return cudaGetLastError();
    }
    if (ix->scan_ring) switch (ix->row_bytes) {
    case 16: scan_kernel<1, 4, 3><<<grid, kScanThreads, smem, stream>>>(p); break;
    case 32: scan_kernel<2, 4, 3><<<grid, kScanThreads, smem, stream>>>(p); break;
    default: scan_kernel<4, 2, 3><<<grid, kScanThreads, smem, stream>>>(p); break;
    } else switch (ix->row_bytes) {
    case 16: scan_kernel<1, 4, 0><<<grid, kScanThreads, smem, stream>>>(p); break;
    case 32: scan_kernel<2, 4, 0><<<grid, kScanThreads, smem, stream>>>(p); break;
    default: scan_kernel<4, 2, 0><<<grid, kScanThreads, smem, stream>>>(p); break;
    }
    return cudaGetLastError();
}

static int scan_ctas_per_sm(const fann_index *ix, size_t smem)
{
    int n = 0;
    cudaError_t e;
    if (ix->scan_ring) switch (ix->row_bytes) {
    case 16: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, scan_kernel<1, 4, 3>, kScanThreads, smem); break;
    case 32: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, scan_kernel<2, 4, 3>, kScanThreads, smem); break;
    default: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, scan_kernel<4, 2, 3>, kScanThreads, smem); break;
    } else switch (ix->row_bytes) {
    case 16: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, scan_kernel<1, 4, 0>, kScanThreads, smem); break;
    case 32: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, scan_kernel<2, 4, 0>, kScanThreads, smem); break;
    default: e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, scan_kernel<4, 2, 0>, kScanThreads, smem); break;
    }
    return (e == cudaSuccess && n >= 1) ? n : 1;
}

// plan + mode + partition + dedup (+ scan unless dump), chunk of queries by chunk (one chunk by default).
// exact_total: the call covers the whole CSR (cand_offsets[0] == 0, cand_offsets[B] == total_cands); a chunk of a
// larger batch (fann_search_host) passes absolute offsets into the whole ID array instead.
static int run_path(fann_index *ix, bool dump, const float *lut, uint32_t B,
                    const int64_t *cand_offsets, const uint32_t *cand_ids, uint64_t total_cands,
                    uint32_t k, uint32_t *out_ids, float *out_dists, uint32_t *out_counts,
                    uint32_t *out_uniq, uint32_t *uniq_ids, uint32_t *uniq_counts,
                    void *workspace, size_t workspace_bytes, cudaStream_t stream,
                    uint32_t shape = 0, bool keep_status = false, bool exact_total = true, bool allow_split = true,
                    const uint32_t *probes = nullptr, uint32_t nprobe = 0)
{
    // probes != NULL: lists-direct (fann_search_lists on sorted posting lists): cand_ids is not read, the dedup kernel
    // takes every item's IDs straight from the probed lists
    const bool ld = probes != nullptr;
    Geom g;
    geometry(ix, k, B, total_cands, &g, shape, allow_split, ld);
    WsLayout w;
    ws_layout(B, total_cands, g, !dump, &w);
    if (!workspace || ((uintptr_t)workspace & 255) != 0)
        return fail(FANN_EWORKSPACE, "workspace is NULL or not 256-byte aligned");
    if (workspace_bytes < w.total)
        return fail(FANN_EWORKSPACE, "workspace has %zu bytes, %zu needed", workspace_bytes, w.total);
    if (((uintptr_t)cand_offsets & 7) != 0) return fail(FANN_EINVAL, "cand_offsets must be 8-byte aligned");
    if ((((uintptr_t)cand_ids | (uintptr_t)out_ids | (uintptr_t)out_dists | (uintptr_t)out_counts |
          (uintptr_t)out_uniq | (uintptr_t)uniq_ids | (uintptr_t)uniq_counts) & 3) != 0)
        return fail(FANN_EINVAL, "ID and output arrays must be 4-byte aligned");
    if (lut && ((uintptr_t)lut & 15) != 0) return fail(FANN_EINVAL, "lut must be 16-byte aligned");
    DeviceGuard guard(ix->device);
    char *ws = (char *)workspace;
    WsHeader *hdr = (WsHeader *)(ws + w.hdr);
    uint32_t *S = (uint32_t *)(ws + w.S);
    uint32_t *mode = (uint32_t *)(ws + w.mode);
    uint32_t *item_start = (uint32_t *)(ws + w.item_start);
    uint2 *items = (uint2 *)(ws + w.items);
    if (!dump) { uniq_counts = (uint32_t *)(ws + w.uniq_counts); uniq_ids = (uint32_t *)(ws + w.uniq_ids); }

    const bool timing = ix->timing.load();
    std::unique_lock<std::mutex> tl(ix->timing_mu, std::defer_lock);
    if (timing) tl.lock();
    if (timing) cudaEventRecord(ix->ev_plan[0], stream);
    plan_kernel<<<1, 1024, 0, stream>>>((const long long *)cand_offsets, B, g.cap_c, w.max_items, hdr, S,
                                        item_start, items, uniq_counts, keep_status ? 1u : 0u,
                                        (unsigned long long)total_cands, exact_total ? 1u : 0u,
                                        g.part_ctas > 1 && !ld ? (uint32_t *)(ws + w.bucket_cnt) : nullptr,
                                        g.part_ctas > 1 && !ld ? (uint32_t *)(ws + w.part_aux) : nullptr, ld ? g.min_classes : 0u);
    if (ld)
        lists_classes_kernel<<<B, 256, 0, stream>>>(ix->list_grid, ix->n_lists, ix->N, probes, nprobe, S, item_start,
                                                    (uint32_t)((uint64_t)g.nslots_max * 9 / 10), ix->force_mode, mode,
                                                    (uint32_t *)(ws + w.bucket_cnt));
    else
        mode_kernel<<<(B + 7) / 8, 256, 0, stream>>>((const long long *)cand_offsets, cand_ids, B, ix->N,
                                                      ix->force_mode, ix->partition ? 0u : g.cap_c, mode);
    if (timing) cudaEventRecord(ix->ev_plan[1], stream);
    ix->launches += 2;
    CUDA_TRY(cudaGetLastError());

    uint32_t chunks = (dump || ld) ? 1u : ix->chunks;
    if (chunks > B) chunks = B;
    const bool overlap = chunks > 1 && ix->partition;
    CtxLease lease(overlap ? ix : nullptr);                    // returned to the pool when the call returns
    CallCtx *cx = lease.c;
    if (overlap) {
        if (!cx) return fail(FANN_ECUDA, "could not create the second stream of the call");
        CUDA_TRY(cudaEventRecord(cx->ev_fork, stream));
        CUDA_TRY(cudaStreamWaitEvent(cx->side, cx->ev_fork, 0));
    }

    DedupParams dp;
    dp.cand_offsets = (const long long *)cand_offsets; dp.cand_ids = cand_ids; dp.N = ix->N;
    dp.nslots_max = g.nslots_max; dp.hdr = hdr; dp.S = S; dp.mode = mode; dp.item_start = item_start; dp.items = items;
    dp.uniq_ids = uniq_ids; dp.uniq_counts = uniq_counts;
    dp.part_ids = ix->partition ? (const uint32_t *)(ws + w.part_ids) : nullptr;
    dp.part_ok = (const uint32_t *)(ws + w.part_ok); dp.bucket_cnt = (const uint32_t *)(ws + w.bucket_cnt);
    dp.list_offsets = ix->list_offsets; dp.list_ids = ix->list_ids; dp.list_grid = ix->list_grid;
    dp.probes = probes; dp.nprobe = nprobe; dp.n_lists = ix->n_lists;
    PartParams pp;
    pp.cand_offsets = (const long long *)cand_offsets; pp.cand_ids = cand_ids; pp.N = ix->N;
    pp.S = S; pp.mode = mode; pp.item_start = item_start;
    pp.part_ids = (uint32_t *)(ws + w.part_ids); pp.part_ok = (uint32_t *)(ws + w.part_ok);
    pp.bucket_cnt = (uint32_t *)(ws + w.bucket_cnt);
    pp.class_max = (uint32_t)((uint64_t)g.nslots_max * 9 / 10);
    pp.ctas = g.part_ctas; pp.aux = (uint32_t *)(ws + w.part_aux);
    ScanParams sp;
    sp.codes = ix->codes; sp.M = ix->M; sp.lut = lut; sp.cand_offsets = (const long long *)cand_offsets;
    sp.uniq_ids = uniq_ids; sp.uniq_counts = uniq_counts; sp.k = k; sp.cap = g.cap;
    sp.out_ids = out_ids; sp.out_dists = out_dists; sp.out_counts = out_counts; sp.out_uniq = out_uniq;
    sp.parts = g.parts; sp.part_keys = (unsigned long long *)(ws + w.part_keys);
    sp.key_src = nullptr; sp.id_limit = 0xFFFFFFFFu;
    uint32_t merge_k2 = 32;                                    // a part's keys padded to a power of two
    while (merge_k2 < k) merge_k2 <<= 1;
    const int per_sm = dump ? 1 : scan_ctas_per_sm(ix, g.scan_smem);

    // With chunks > 1 the partition launches of all chunks go to the side stream at once: the partition kernel is
    // HBM-bound, light on registers and shared memory, and fits on an SM beside a scan CTA, so the split of chunk
    // c + 1 runs under the scan of chunk c.  Dedup and scan stay on `stream`, chunk by chunk.
    if (overlap) {
        for (uint32_t c = 0; c < chunks; ++c) {
            const uint32_t qb = (uint32_t)((uint64_t)B * c / chunks), qe = (uint32_t)((uint64_t)B * (c + 1) / chunks);
            pp.q_begin = qb;
            partition_kernel<<<qe - qb, kPartThreads, 0, cx->side>>>(pp);
            ix->launches++;
            CUDA_TRY(cudaGetLastError());
            CUDA_TRY(cudaEventRecord(cx->ev_done[c], cx->side));
        }
    }
    uint32_t scan_ctas = 0;
    for (uint32_t c = 0; c < chunks; ++c) {
        const uint32_t qb = (uint32_t)((uint64_t)B * c / chunks), qe = (uint32_t)((uint64_t)B * (c + 1) / chunks);
        if (overlap) CUDA_TRY(cudaStreamWaitEvent(stream, cx->ev_done[c], 0));
        if (!overlap && ix->partition && c == 0 && !ld) {
            pp.q_begin = 0;
            if (timing) cudaEventRecord(ix->ev_part[0], stream);
            if (g.part_ctas > 1) partition_multi_kernel<<<B * g.part_ctas, kPartThreads, 0, stream>>>(pp);
            else partition_kernel<<<B, kPartThreads, 0, stream>>>(pp);
            if (timing) { cudaEventRecord(ix->ev_part[1], stream); ix->have_part = true; }
            ix->launches++;
            CUDA_TRY(cudaGetLastError());
        }
        if (timing) cudaEventRecord(ix->ev_dedup[c][0], stream);
        dp.q_begin = qb; dp.q_end = qe; dp.counter = &hdr->dedup_counter[c];
        if (ld) {
            if (g.dedup_threads == 512) dedup_kernel<512, 8, true><<<2 * ix->num_sms, 512, g.dedup_smem, stream>>>(dp);
            else dedup_kernel<1024, 8, true><<<ix->num_sms, 1024, g.dedup_smem, stream>>>(dp);
        } else if (g.dedup_threads == 512) dedup_kernel<512, 8><<<2 * ix->num_sms, 512, g.dedup_smem, stream>>>(dp);
        else dedup_kernel<1024, 8><<<ix->num_sms, 1024, g.dedup_smem, stream>>>(dp);
        if (timing) cudaEventRecord(ix->ev_dedup[c][1], stream);
        ix->launches++;
        CUDA_TRY(cudaGetLastError());
        if (dump) continue;
        sp.q_begin = qb; sp.q_end = qe; sp.counter = &hdr->scan_counter[c];
        int grid = ix->num_sms * per_sm;
        if ((uint32_t)grid > (qe - qb) * g.parts) grid = (int)((qe - qb) * g.parts);
        if (timing) cudaEventRecord(ix->ev_scan[c][0], stream);
        cudaError_t e = launch_scan(ix, grid, g.scan_smem, stream, sp);
        if (e == cudaSuccess && g.parts > 1) {
            merge_parts_kernel<<<qe - qb, kMergeThreads, (size_t)g.parts * merge_k2 * 8, stream>>>(
                sp.part_keys, uniq_counts, qb, g.parts, k, merge_k2, out_ids, out_dists, out_counts, out_uniq);
            ix->launches++;
            e = cudaGetLastError();
        }
        if (timing) cudaEventRecord(ix->ev_scan[c][1], stream);
        ix->launches++;
        if (e != cudaSuccess) return fail(FANN_ECUDA, "scan kernel launch: %s", cudaGetErrorString(e));
        scan_ctas = (uint32_t)grid;
    }
    {
        std::lock_guard<std::mutex> lg(ix->mu);
        if (scan_ctas) ix->last_scan_ctas = scan_ctas;
        ix->last_dedup_threads = g.dedup_threads; ix->last_dedup_smem = g.dedup_smem;
        ix->last_dedup_ctas = (uint32_t)ix->num_sms * (1024u / g.dedup_threads); ix->last_slots = g.nslots_max; ix->last_chunks = chunks;
        ix->last_scan_smem = g.scan_smem; ix->last_cap = g.cap;
    }
    if (timing) {
        ix->timed_chunks = chunks;
        ix->timed_scan = !dump;
        ix->have_scan = true;
    }
    return FANN_OK;
}

extern "C" int fann_dedup_scan_topk(fann_index *ix, const float *lut, uint32_t B,
                                    const int64_t *cand_offsets, const uint32_t *cand_ids,
                                    uint64_t total_cands, uint32_t k,
                                    uint32_t *out_ids, float *out_dists,
                                    uint32_t *out_counts, uint32_t *out_uniq,
                                    void *workspace, size_t workspace_bytes, void *stream)
{
    if (!ix || !lut || !cand_offsets || !out_ids || !out_dists)
        return fail(FANN_EINVAL, "fann_dedup_scan_topk: NULL argument");
    if (!cand_ids && total_cands) return fail(FANN_EINVAL, "fann_dedup_scan_topk: cand_ids is NULL");
    if (!ix->codes) return fail(FANN_EINVAL, "fann_dedup_scan_topk: load codes first");
    if (B == 0) return fail(FANN_EINVAL, "fann_dedup_scan_topk: B == 0");
    if (k == 0 || k > FANN_MAX_K) return fail(FANN_EUNSUPPORTED, "fann_dedup_scan_topk: k=%u not in 1..%u", k, FANN_MAX_K);
    return run_path(ix, false, lut, B, cand_offsets, cand_ids, total_cands, k, out_ids, out_dists,
                    out_counts, out_uniq, nullptr, nullptr, workspace, workspace_bytes, (cudaStream_t)stream);
}

// The same path with its workspace in g_static_ws: allocates nothing (fann.h).  One array per device, shared by
// every call: overlapping calls race.
extern "C" int fann_dedup_scan_topk_static(fann_index *ix, const float *lut, uint32_t B,
                                           const int64_t *cand_offsets, const uint32_t *cand_ids,
                                           uint64_t total_cands, uint32_t k,
                                           uint32_t *out_ids, float *out_dists,
                                           uint32_t *out_counts, uint32_t *out_uniq,
                                           uint32_t *out_status, void *stream_)
{
    if (!ix || !lut || !cand_offsets || !out_ids || !out_dists)
        return fail(FANN_EINVAL, "fann_dedup_scan_topk_static: NULL argument");
    if (!cand_ids && total_cands) return fail(FANN_EINVAL, "fann_dedup_scan_topk_static: cand_ids is NULL");
    if (!ix->codes) return fail(FANN_EINVAL, "fann_dedup_scan_topk_static: load codes first");
    if (B == 0) return fail(FANN_EINVAL, "fann_dedup_scan_topk_static: B == 0");
    if (k == 0 || k > FANN_MAX_K)
        return fail(FANN_EUNSUPPORTED, "fann_dedup_scan_topk_static: k=%u not in 1..%u", k, FANN_MAX_K);
    if (((uintptr_t)out_status & 3) != 0) return fail(FANN_EINVAL, "fann_dedup_scan_topk_static: out_status must be 4-byte aligned");
    if (!ix->static_ws)
        return fail(FANN_ECUDA, "fann_dedup_scan_topk_static: cudaGetSymbolAddress of the static workspace failed in fann_create: %s",
                    cudaGetErrorString(ix->static_ws_err));
    if (ix->chunks != 1)
        return fail(FANN_EUNSUPPORTED, "fann_dedup_scan_topk_static: not with FANN_CHUNKS > 1 (the chunked path creates a stream)");
    Geom g;
    geometry(ix, k, B, total_cands, &g);                       // as run_path and fann_workspace_bytes compute it
    WsLayout w;
    ws_layout(B, total_cands, g, true, &w);
    if (w.total > (size_t)FANN_STATIC_WS_BYTES)
        return fail(FANN_EWORKSPACE, "fann_dedup_scan_topk_static: B=%u, total_cands=%llu, k=%u need %zu bytes of workspace, "
                    "the static array holds %u (FANN_STATIC_WS_BYTES); use fann_dedup_scan_topk with a workspace of your own",
                    B, (unsigned long long)total_cands, k, w.total, (unsigned)FANN_STATIC_WS_BYTES);
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    // the array keeps the last call's contents: the header (status word, work counters) starts at zero
    CUDA_TRY(cudaMemsetAsync((char *)ix->static_ws + w.hdr, 0, 256, stream));
    const int rc = run_path(ix, false, lut, B, cand_offsets, cand_ids, total_cands, k, out_ids, out_dists,
                            out_counts, out_uniq, nullptr, nullptr, ix->static_ws, (size_t)FANN_STATIC_WS_BYTES, stream);
    if (rc != FANN_OK) return rc;
    if (out_status)
        CUDA_TRY(cudaMemcpyAsync(out_status, (const char *)ix->static_ws + w.hdr, 4, cudaMemcpyDeviceToDevice, stream));
    return FANN_OK;
}

extern "C" int fann_dedup_only(fann_index *ix, uint32_t B, const int64_t *cand_offsets,
                               const uint32_t *cand_ids, uint64_t total_cands,
                               uint32_t *uniq_ids, uint32_t *uniq_counts,
                               void *workspace, size_t workspace_bytes, void *stream)
{
    if (!ix || !cand_offsets || !uniq_counts) return fail(FANN_EINVAL, "fann_dedup_only: NULL argument");
    if ((!cand_ids || !uniq_ids) && total_cands) return fail(FANN_EINVAL, "fann_dedup_only: NULL id array");
    if (!ix->codes) return fail(FANN_EINVAL, "fann_dedup_only: load codes first (N is unknown)");
    if (B == 0) return fail(FANN_EINVAL, "fann_dedup_only: B == 0");
    return run_path(ix, true, nullptr, B, cand_offsets, cand_ids, total_cands, 1, nullptr, nullptr,
                    nullptr, nullptr, uniq_ids, uniq_counts, workspace, workspace_bytes, (cudaStream_t)stream);
}

extern "C" int fann_workspace_status(fann_index *ix, const void *workspace, void *stream)
{
    if (!ix || !workspace) return fail(FANN_EINVAL, "fann_workspace_status: NULL argument");
    DeviceGuard guard(ix->device);
    WsHeader h;
    CUDA_TRY(cudaMemcpyAsync(&h, workspace, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
    if (h.status & kStatusPlanOverflow)
        return fail(FANN_EINVAL, "total_cands passed to the call was smaller than cand_offsets[B]");
    if (h.status & kStatusTableFull)
        return fail(FANN_EOVERFLOW, "a dedup hash table filled up (colliding candidate IDs)");
    return FANN_OK;
}

extern "C" int fann_workspace_modes(fann_index *ix, const void *workspace, uint32_t B, uint64_t total_cands, uint32_t k,
                                    uint32_t *n_ordered, uint32_t *n_hashed, void *stream)
{
    if (!ix || !workspace || B == 0) return fail(FANN_EINVAL, "fann_workspace_modes: bad argument");
    if (!ix->codes || k == 0 || k > FANN_MAX_K) return fail(FANN_EINVAL, "fann_workspace_modes: bad argument");
    DeviceGuard guard(ix->device);
    Geom g;
    geometry(ix, k, B, total_cands, &g);
    WsLayout w;
    ws_layout(B, total_cands, g, true, &w);
    std::vector<uint32_t> mode(B);
    CUDA_TRY(cudaMemcpyAsync(mode.data(), (const char *)workspace + w.mode, (size_t)B * 4, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
    uint32_t h = 0;
    for (uint32_t b = 0; b < B; ++b) h += mode[b] == kModeHashed ? 1u : 0u;
    if (n_ordered) *n_ordered = B - h;
    if (n_hashed) *n_hashed = h;
    return FANN_OK;
}

// ---------------------------------------------------------------- host-buffer entry

struct HostScratch {
    size_t queries, offsets, ids, lut, out_ids, out_dists, out_counts, ws, ws_bytes, total;
};

static void host_scratch_layout(const fann_index *ix, uint32_t B, uint32_t dsub, uint64_t total_cands,
                                uint32_t k, HostScratch *h)
{
    Geom g;
    geometry(ix, k, B, total_cands, &g);
    WsLayout w;
    ws_layout(B, total_cands, g, true, &w);
    size_t o = 0;
    h->queries = o;    o = align_up(o + (size_t)B * ix->M * dsub * 4, 256);
    h->offsets = o;    o = align_up(o + ((size_t)B + 1) * 8, 256);
    h->ids = o;        o = align_up(o + (size_t)total_cands * 4, 256);
    h->lut = o;        o = align_up(o + (size_t)B * ix->M * 1024, 256);
    h->out_ids = o;    o = align_up(o + (size_t)B * k * 4, 256);
    h->out_dists = o;  o = align_up(o + (size_t)B * k * 4, 256);
    h->out_counts = o; o = align_up(o + (size_t)B * 4, 256);
    h->ws = o;         h->ws_bytes = w.total; o += w.total;
    h->total = o;
}

extern "C" size_t fann_search_host_scratch_bytes(const fann_index *ix, uint32_t B, uint32_t dsub,
                                                 uint64_t total_cands, uint32_t k)
{
    if (!ix || !ix->codes || B == 0 || dsub == 0 || k == 0 || k > FANN_MAX_K) {
        fail(FANN_EINVAL, "fann_search_host_scratch_bytes: bad argument");
        return 0;
    }
    HostScratch h;
    host_scratch_layout(ix, B, dsub, total_cands, k, &h);
    return h.total;
}

// The device address of a page-locked host array (cudaHostAlloc / cudaHostRegister: what pinned torch tensors are),
// or NULL for pageable memory.  The host entries hand such output arrays to the kernels themselves: a query's results
// cross PCIe while the other queries are still being scanned, and no copy follows the last kernel.
static void *mapped_host_ptr(const void *host)
{
    if (!host) return nullptr;
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return a.type == cudaMemoryTypeHost ? a.devicePointer : nullptr;
}

extern "C" int fann_search_host(fann_index *ix, const float *queries_h, uint32_t B,
                                const float *codebooks_d, uint32_t dsub,
                                const int64_t *cand_offsets_h, const uint32_t *cand_ids_h,
                                uint32_t k, uint32_t *out_ids_h, float *out_dists_h, uint32_t *out_counts_h,
                                void *device_scratch, size_t scratch_bytes, void *stream_)
{
    if (!ix || !queries_h || !codebooks_d || !cand_offsets_h || !out_ids_h || !out_dists_h)
        return fail(FANN_EINVAL, "fann_search_host: NULL argument");
    if (!ix->codes) return fail(FANN_EINVAL, "fann_search_host: load codes first");
    if (B == 0 || dsub == 0) return fail(FANN_EINVAL, "fann_search_host: B or dsub is 0");
    if (k == 0 || k > FANN_MAX_K) return fail(FANN_EUNSUPPORTED, "fann_search_host: k=%u", k);
    const uint64_t total = (uint64_t)cand_offsets_h[B];
    if (!cand_ids_h && total) return fail(FANN_EINVAL, "fann_search_host: cand_ids_h is NULL");
    HostScratch h;
    host_scratch_layout(ix, B, dsub, total, k, &h);
    if (!device_scratch || ((uintptr_t)device_scratch & 255) != 0 || scratch_bytes < h.total)
        return fail(FANN_EWORKSPACE, "fann_search_host: scratch has %zu bytes, %zu needed (256-byte aligned)",
                    scratch_bytes, h.total);
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    char *s = (char *)device_scratch;
    CUDA_TRY(cudaMemcpyAsync(s + h.queries, queries_h, (size_t)B * ix->M * dsub * 4, cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(s + h.offsets, cand_offsets_h, ((size_t)B + 1) * 8, cudaMemcpyHostToDevice, stream));
    int rc = fann_build_lut(ix, (const float *)(s + h.queries), B, codebooks_d, dsub, (float *)(s + h.lut), stream);
    if (rc != FANN_OK) return rc;
    // The candidate IDs are the bulk of the transfer (PAPER.md:L125 step (4)).  They go up in chunks of queries
    // on the index's side stream, and the path runs chunk by chunk behind them: queries are independent, and
    // offsets stay absolute, so a chunk is the same call on a sub-range of the batch.
    Geom g;
    geometry(ix, k, B, total, &g);                             // one dedup CTA shape for all chunks: the layout depends on it
    const uint32_t nchunk = (B >= 64 && total >= (4u << 20) && ix->chunks == 1) ? 8u : 1u;   // 16 MB of IDs and up
    uint32_t *o_ids = (uint32_t *)(s + h.out_ids), *o_counts = (uint32_t *)(s + h.out_counts);
    float *o_dists = (float *)(s + h.out_dists);
    bool direct = false;
    if (ix->host_direct) {
        void *di = mapped_host_ptr(out_ids_h), *dd = mapped_host_ptr(out_dists_h), *dc = mapped_host_ptr(out_counts_h);
        if (di && dd && (dc || !out_counts_h)) {
            direct = true; o_ids = (uint32_t *)di; o_dists = (float *)dd;
            if (dc) o_counts = (uint32_t *)dc;
        }
    }
    CtxLease lease(ix);
    CallCtx *cx = lease.c;
    if (!cx) return fail(FANN_ECUDA, "fann_search_host: could not create the transfer stream");
    CUDA_TRY(cudaEventRecord(cx->ev_fork, stream));
    CUDA_TRY(cudaStreamWaitEvent(cx->side, cx->ev_fork, 0));   // the scratch may still be in use by earlier work on `stream`
    for (uint32_t c = 0; c < nchunk; ++c) {
        const uint32_t b0 = (uint32_t)((uint64_t)B * c / nchunk), b1 = (uint32_t)((uint64_t)B * (c + 1) / nchunk);
        const uint64_t e0 = (uint64_t)cand_offsets_h[b0], e1 = (uint64_t)cand_offsets_h[b1];
        if (e1 > e0)
            CUDA_TRY(cudaMemcpyAsync(s + h.ids + e0 * 4, cand_ids_h + e0, (size_t)(e1 - e0) * 4, cudaMemcpyHostToDevice, cx->side));
        CUDA_TRY(cudaEventRecord(cx->ev_done[c], cx->side));
        CUDA_TRY(cudaStreamWaitEvent(stream, cx->ev_done[c], 0));
        rc = run_path(ix, false, (const float *)(s + h.lut) + (size_t)b0 * ix->M * 256, b1 - b0,
                      (const int64_t *)(s + h.offsets) + b0, (const uint32_t *)(s + h.ids), total, k,
                      o_ids + (size_t)b0 * k, o_dists + (size_t)b0 * k, o_counts + b0, nullptr, nullptr, nullptr,
                      s + h.ws, h.ws_bytes, stream, g.dedup_threads, c > 0, nchunk == 1, nchunk == 1);
        if (rc != FANN_OK) return rc;
    }
    if (!direct) {
        CUDA_TRY(cudaMemcpyAsync(out_ids_h, s + h.out_ids, (size_t)B * k * 4, cudaMemcpyDeviceToHost, stream));
        CUDA_TRY(cudaMemcpyAsync(out_dists_h, s + h.out_dists, (size_t)B * k * 4, cudaMemcpyDeviceToHost, stream));
        if (out_counts_h)
            CUDA_TRY(cudaMemcpyAsync(out_counts_h, s + h.out_counts, (size_t)B * 4, cudaMemcpyDeviceToHost, stream));
    }
    CUDA_TRY(cudaStreamSynchronize(stream));
    return fann_workspace_status(ix, s + h.ws, stream);
}


// ---------------------------------------------------------------- NEXT-2: posting lists resident in HBM

extern "C" int fann_load_lists(fann_index *ix, const int64_t *list_offsets, const uint32_t *list_ids,
                               uint64_t n_lists, uint64_t n_entries, int src_is_device, void *stream_)
{
    if (!ix || !list_offsets) return fail(FANN_EINVAL, "fann_load_lists: NULL argument");
    if (!list_ids && n_entries) return fail(FANN_EINVAL, "fann_load_lists: list_ids is NULL");
    if (n_lists == 0 || n_lists >= 0xFFFFFFFFull) return fail(FANN_EINVAL, "fann_load_lists: n_lists must be in 1 .. 2^32-2");
    if (((uintptr_t)list_offsets & 7) != 0 || ((uintptr_t)list_ids & 3) != 0)
        return fail(FANN_EINVAL, "fann_load_lists: list_offsets must be 8-byte and list_ids 4-byte aligned");
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    ix->generation++;
    if (ix->list_offsets) { cudaFree(ix->list_offsets); ix->list_offsets = nullptr; }
    if (ix->list_ids) { cudaFree(ix->list_ids); ix->list_ids = nullptr; }
    if (ix->lm_codes) { cudaFree(ix->lm_codes); ix->lm_codes = nullptr; }      // built from the old lists
    ix->n_lists = 0; ix->list_entries = 0;
    cudaError_t e = cudaMalloc(&ix->list_offsets, (n_lists + 1) * 8);
    if (e == cudaSuccess) e = cudaMalloc(&ix->list_ids, (n_entries ? n_entries : 1) * 4);
    if (e != cudaSuccess) {
        if (ix->list_offsets) { cudaFree(ix->list_offsets); ix->list_offsets = nullptr; }
        return fail(FANN_ENOMEM, "fann_load_lists: cudaMalloc: %s", cudaGetErrorString(e));
    }
    const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CUDA_TRY(cudaMemcpyAsync(ix->list_offsets, list_offsets, (n_lists + 1) * 8, kind, stream));
    if (n_entries) CUDA_TRY(cudaMemcpyAsync(ix->list_ids, list_ids, n_entries * 4, kind, stream));
    long long ends[2] = {-1, -1};                              // offsets[0] and offsets[n_lists] bound every read of list_ids
    CUDA_TRY(cudaMemcpyAsync(&ends[0], ix->list_offsets, 8, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaMemcpyAsync(&ends[1], ix->list_offsets + n_lists, 8, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    if (ends[0] != 0 || ends[1] < 0 || (uint64_t)ends[1] != n_entries) {
        cudaFree(ix->list_offsets); cudaFree(ix->list_ids);
        ix->list_offsets = nullptr; ix->list_ids = nullptr;
        return fail(FANN_EINVAL, "fann_load_lists: list_offsets[0] = %lld, list_offsets[n_lists] = %lld, n_entries = %llu",
                    ends[0], ends[1], (unsigned long long)n_entries);
    }
    ix->n_lists = n_lists; ix->list_entries = n_entries;
    // Sort every list and index it by ID-range cell (needs N: load the codes first), so that fann_search_lists can
    // read a class's IDs straight from the lists.  The order of a list's IDs carries no meaning (L150).
    ix->lists_sorted = false;
    if (ix->list_grid) { cudaFree(ix->list_grid); ix->list_grid = nullptr; }
    if (ix->codes && ix->N && n_entries < 0xFFFFFFFFull) {
        uint32_t *flag = nullptr;
        if (cudaMalloc(&ix->list_grid, n_lists * (kGridCells + 1) * sizeof(uint16_t)) == cudaSuccess &&
            cudaMalloc(&flag, 4) == cudaSuccess) {
            CUDA_TRY(cudaMemsetAsync(flag, 0, 4, stream));
            lists_sort_grid_kernel<<<(unsigned)n_lists, 256, kSortMaxList * 4, stream>>>(ix->list_offsets, ix->list_ids, ix->N,
                                                                                       ix->list_grid, flag);
            ix->launches++;
            uint32_t unsorted = 1;
            cudaError_t e2 = cudaMemcpyAsync(&unsorted, flag, 4, cudaMemcpyDeviceToHost, stream);
            if (e2 == cudaSuccess) e2 = cudaStreamSynchronize(stream);
            cudaFree(flag);
            if (e2 != cudaSuccess) return fail(FANN_ECUDA, "fann_load_lists: sorting the lists: %s", cudaGetErrorString(e2));
            ix->lists_sorted = unsorted == 0;
        } else {
            if (ix->list_grid) { cudaFree(ix->list_grid); ix->list_grid = nullptr; }
            if (flag) cudaFree(flag);
            cudaGetLastError();
        }
    }
    return FANN_OK;
}

struct ListsLayout { size_t hdr, offsets, ids, ws, ws_bytes, total; };

static bool lists_direct_ok(const fann_index *ix, uint32_t nprobe)
{
    return ix->lists_direct && ix->lists_sorted && ix->list_grid && nprobe <= kLdMaxProbe;
}

static void lists_layout(const fann_index *ix, uint32_t B, uint64_t cap, uint32_t k, ListsLayout *l)
{
    Geom g;
    geometry(ix, k, B, cap, &g, 0, true, ix->lists_direct && ix->lists_sorted);   // the direct path's tables are a little smaller
    WsLayout w;
    ws_layout(B, cap, g, true, &w);
    size_t o = 0;
    l->hdr = o;     o = align_up(o + sizeof(ListsHeader), 256);
    l->offsets = o; o = align_up(o + ((size_t)B + 1) * 8, 256);
    l->ids = o;     o = align_up(o + (size_t)cap * 4 + 16, 256);
    l->ws = o;      l->ws_bytes = w.total; o += w.total;
    l->total = o;
}

extern "C" size_t fann_search_lists_workspace_bytes(const fann_index *ix, uint32_t B, uint64_t max_total_cands, uint32_t k)
{
    if (!ix || !ix->codes) { fail(FANN_EINVAL, "fann_search_lists_workspace_bytes: index has no codes"); return 0; }
    if (B == 0 || k == 0 || k > FANN_MAX_K) { fail(FANN_EINVAL, "fann_search_lists_workspace_bytes: B=%u k=%u", B, k); return 0; }
    ListsLayout l;
    lists_layout(ix, B, max_total_cands, k, &l);
    return l.total;
}

// Steps (3)(5)(6)(7) for B queries inside a workspace laid out by `l`.
static int search_lists_impl(fann_index *ix, const float *lut, uint32_t B, const uint32_t *probes, uint32_t nprobe,
                             uint64_t max_total_cands, uint32_t k, uint32_t *out_ids, float *out_dists,
                             uint32_t *out_counts, uint32_t *out_uniq, char *ws, const ListsLayout &l,
                             cudaStream_t stream)
{
    ListsHeader *hdr = (ListsHeader *)(ws + l.hdr);
    long long *offsets = (long long *)(ws + l.offsets);
    uint32_t *ids = (uint32_t *)(ws + l.ids);
    lists_count_kernel<<<(B + 7) / 8, 256, 0, stream>>>(ix->list_offsets, ix->n_lists, probes, B, nprobe,
                                                         (unsigned long long *)offsets);
    lists_scan_kernel<<<1, 1024, 0, stream>>>((const unsigned long long *)offsets, B, offsets, hdr,
                                              (unsigned long long)max_total_cands);
    if (lists_direct_ok(ix, nprobe)) {
        // sorted lists with a grid: no candidate array, no class split -- the dedup kernel reads every class's IDs
        // straight from the probed lists (cand_offsets only places the queries' distinct lists)
        ix->launches += 2;
        CUDA_TRY(cudaGetLastError());
        return run_path(ix, false, lut, B, (const int64_t *)offsets, ids, max_total_cands, k, out_ids, out_dists, out_counts,
                        out_uniq, nullptr, nullptr, ws + l.ws, l.ws_bytes, stream, 0, false, false, true, probes, nprobe);
    }
    uint32_t expand_ctas = 1;                                  // small batches: spread a query's lists over several CTAs
    while (expand_ctas < 16 && 2 * expand_ctas * B <= (uint32_t)ix->num_sms && 8 * expand_ctas < nprobe) expand_ctas <<= 1;
    lists_expand_kernel<<<B * expand_ctas, kExpandThreads, ((size_t)nprobe + 1) * 4, stream>>>(
        ix->list_offsets, ix->list_ids, ix->n_lists, probes, nprobe, offsets, ids, hdr, expand_ctas, 0u);
    ix->launches += 3;
    CUDA_TRY(cudaGetLastError());
    // a batch larger than the workspace was sized for leaves cand_offsets[B] > max_total_cands: the path refuses it
    return run_path(ix, false, lut, B, (const int64_t *)offsets, ids, max_total_cands, k, out_ids, out_dists, out_counts,
                    out_uniq, nullptr, nullptr, ws + l.ws, l.ws_bytes, stream, 0, false, false);
}

extern "C" int fann_search_lists(fann_index *ix, const float *lut, uint32_t B, const uint32_t *probes, uint32_t nprobe,
                                 uint64_t max_total_cands, uint32_t k, uint32_t *out_ids, float *out_dists,
                                 uint32_t *out_counts, uint32_t *out_uniq, void *workspace, size_t workspace_bytes,
                                 void *stream_)
{
    if (!ix || !lut || !probes || !out_ids || !out_dists) return fail(FANN_EINVAL, "fann_search_lists: NULL argument");
    if (!ix->codes) return fail(FANN_EINVAL, "fann_search_lists: load codes first");
    if (!ix->list_offsets) return fail(FANN_EINVAL, "fann_search_lists: load the posting lists first (fann_load_lists)");
    if (B == 0 || nprobe == 0) return fail(FANN_EINVAL, "fann_search_lists: B or nprobe is 0");
    if (nprobe > FANN_MAX_NPROBE) return fail(FANN_EUNSUPPORTED, "fann_search_lists: nprobe=%u > %u", nprobe, FANN_MAX_NPROBE);
    if (k == 0 || k > FANN_MAX_K) return fail(FANN_EUNSUPPORTED, "fann_search_lists: k=%u not in 1..%u", k, FANN_MAX_K);
    if (((uintptr_t)probes & 3) != 0) return fail(FANN_EINVAL, "fann_search_lists: probes must be 4-byte aligned");
    ListsLayout l;
    lists_layout(ix, B, max_total_cands, k, &l);
    if (!workspace || ((uintptr_t)workspace & 255) != 0) return fail(FANN_EWORKSPACE, "workspace is NULL or not 256-byte aligned");
    if (workspace_bytes < l.total) return fail(FANN_EWORKSPACE, "workspace has %zu bytes, %zu needed", workspace_bytes, l.total);
    DeviceGuard guard(ix->device);
    return search_lists_impl(ix, lut, B, probes, nprobe, max_total_cands, k, out_ids, out_dists, out_counts, out_uniq,
                             (char *)workspace, l, (cudaStream_t)stream_);
}

extern "C" int fann_search_lists_status(fann_index *ix, const void *workspace, uint32_t B, uint64_t max_total_cands,
                                        uint32_t k, uint64_t *total_cands, void *stream_)
{
    if (!ix || !workspace) return fail(FANN_EINVAL, "fann_search_lists_status: NULL argument");
    if (!ix->codes || B == 0 || k == 0 || k > FANN_MAX_K) return fail(FANN_EINVAL, "fann_search_lists_status: bad argument");
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    ListsHeader h;
    CUDA_TRY(cudaMemcpyAsync(&h, workspace, sizeof(h), cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    if (total_cands) *total_cands = h.total;
    if (h.overflow)
        return fail(FANN_EWORKSPACE, "the probed lists hold %llu candidate IDs, the workspace was sized for %llu (max_total_cands)",
                    h.total, h.capacity);
    ListsLayout l;
    lists_layout(ix, B, max_total_cands, k, &l);
    return fann_workspace_status(ix, (const char *)workspace + l.ws, stream);
}

struct ListsHostScratch { size_t queries, probes, lut, out_ids, out_dists, out_counts, ws, ws_bytes, total; };

static void lists_host_layout(const fann_index *ix, uint32_t B, uint32_t dsub, uint32_t nprobe, uint64_t cap, uint32_t k,
                              ListsHostScratch *h)
{
    ListsLayout l;
    lists_layout(ix, B, cap, k, &l);
    size_t o = 0;
    h->queries = o;    o = align_up(o + (size_t)B * ix->M * dsub * 4, 256);
    h->probes = o;     o = align_up(o + (size_t)B * nprobe * 4, 256);
    h->lut = o;        o = align_up(o + (size_t)B * ix->M * 1024, 256);
    h->out_ids = o;    o = align_up(o + (size_t)B * k * 4, 256);
    h->out_dists = o;  o = align_up(o + (size_t)B * k * 4, 256);
    h->out_counts = o; o = align_up(o + (size_t)B * 4, 256);
    h->ws = o;         h->ws_bytes = l.total; o += l.total;
    h->total = o;
}

extern "C" size_t fann_search_lists_host_scratch_bytes(const fann_index *ix, uint32_t B, uint32_t dsub, uint32_t nprobe,
                                                       uint64_t max_total_cands, uint32_t k)
{
    if (!ix || !ix->codes || B == 0 || dsub == 0 || nprobe == 0 || k == 0 || k > FANN_MAX_K) {
        fail(FANN_EINVAL, "fann_search_lists_host_scratch_bytes: bad argument");
        return 0;
    }
    ListsHostScratch h;
    lists_host_layout(ix, B, dsub, nprobe, max_total_cands, k, &h);
    return h.total;
}

extern "C" int fann_search_lists_host(fann_index *ix, const float *queries_h, uint32_t B, const float *codebooks_d,
                                      uint32_t dsub, const uint32_t *probes_h, uint32_t nprobe, uint64_t max_total_cands,
                                      uint32_t k, uint32_t *out_ids_h, float *out_dists_h, uint32_t *out_counts_h,
                                      void *device_scratch, size_t scratch_bytes, void *stream_)
{
    if (!ix || !queries_h || !codebooks_d || !probes_h || !out_ids_h || !out_dists_h)
        return fail(FANN_EINVAL, "fann_search_lists_host: NULL argument");
    if (!ix->codes || !ix->list_offsets) return fail(FANN_EINVAL, "fann_search_lists_host: load codes and posting lists first");
    if (B == 0 || dsub == 0 || nprobe == 0) return fail(FANN_EINVAL, "fann_search_lists_host: B, dsub or nprobe is 0");
    if (k == 0 || k > FANN_MAX_K) return fail(FANN_EUNSUPPORTED, "fann_search_lists_host: k=%u", k);
    ListsHostScratch h;
    lists_host_layout(ix, B, dsub, nprobe, max_total_cands, k, &h);
    if (!device_scratch || ((uintptr_t)device_scratch & 255) != 0 || scratch_bytes < h.total)
        return fail(FANN_EWORKSPACE, "fann_search_lists_host: scratch has %zu bytes, %zu needed (256-byte aligned)",
                    scratch_bytes, h.total);
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    char *s = (char *)device_scratch;
    // PAPER.md:L125 step (4) with the metadata on the GPU: only the query vectors and nprobe list indices per query go up
    CUDA_TRY(cudaMemcpyAsync(s + h.queries, queries_h, (size_t)B * ix->M * dsub * 4, cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(s + h.probes, probes_h, (size_t)B * nprobe * 4, cudaMemcpyHostToDevice, stream));
    int rc = fann_build_lut(ix, (const float *)(s + h.queries), B, codebooks_d, dsub, (float *)(s + h.lut), stream);
    if (rc != FANN_OK) return rc;
    // (Running the batch in chunks of queries, a chunk's results going down on a second stream while the next chunk
    // computes, was measured at u8_1b_m64 -- 80 MB of results, 1.4 ms of PCIe time: 4 chunks cost more in kernel
    // ramp-up and drain, 4.1 ms over the device path, than the overlap saves, 2.9 ms in one piece.)
    ListsLayout l;
    lists_layout(ix, B, max_total_cands, k, &l);
    uint32_t *o_ids = (uint32_t *)(s + h.out_ids), *o_counts = (uint32_t *)(s + h.out_counts);
    float *o_dists = (float *)(s + h.out_dists);
    bool direct = false;
    if (ix->host_direct) {                                     // pinned output arrays: the kernels write them (80 MB, 1.4 ms of copies at u8_1b_m64)
        void *di = mapped_host_ptr(out_ids_h), *dd = mapped_host_ptr(out_dists_h), *dc = mapped_host_ptr(out_counts_h);
        if (di && dd && (dc || !out_counts_h)) {
            direct = true; o_ids = (uint32_t *)di; o_dists = (float *)dd;
            if (dc) o_counts = (uint32_t *)dc;
        }
    }
    rc = search_lists_impl(ix, (const float *)(s + h.lut), B, (const uint32_t *)(s + h.probes), nprobe, max_total_cands, k,
                           o_ids, o_dists, o_counts, nullptr, s + h.ws, l, stream);
    if (rc != FANN_OK) return rc;
    if (!direct) {
        CUDA_TRY(cudaMemcpyAsync(out_ids_h, s + h.out_ids, (size_t)B * k * 4, cudaMemcpyDeviceToHost, stream));
        CUDA_TRY(cudaMemcpyAsync(out_dists_h, s + h.out_dists, (size_t)B * k * 4, cudaMemcpyDeviceToHost, stream));
        if (out_counts_h)
            CUDA_TRY(cudaMemcpyAsync(out_counts_h, s + h.out_counts, (size_t)B * 4, cudaMemcpyDeviceToHost, stream));
    }
    return fann_search_lists_status(ix, s + h.ws, B, max_total_cands, k, nullptr, stream);   // synchronises
}

// ---------------------------------------------------------------- EXPERIMENT: list-major code copy, streamed

// Not the paper's layout (its codes are indexed by vector-ID, L152, and the lists hold IDs only, L150): a second copy
// of the codes in posting-list order, replicas included, so that step (6) reads a probed list as one contiguous run
// instead of gathering rows.  Every candidate is scored, repeats included; they are removed where the top-k buffer is
// pruned (a vector in several probed lists has the same key each time).  See DESIGN.md 6.7.
extern "C" int fann_build_list_codes(fann_index *ix, void *stream_)
{
    if (!ix) return fail(FANN_EINVAL, "fann_build_list_codes: NULL index");
    if (!ix->codes || !ix->list_offsets) return fail(FANN_EINVAL, "fann_build_list_codes: load codes and posting lists first");
    if (ix->list_entries >= 0xFFFFFFFFull) return fail(FANN_EUNSUPPORTED, "fann_build_list_codes: more than 2^32-2 list entries");
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    if (ix->lm_codes) { cudaFree(ix->lm_codes); ix->lm_codes = nullptr; }
    const size_t bytes = (size_t)(ix->list_entries ? ix->list_entries : 1) * ix->row_bytes;
    cudaError_t e = cudaMalloc(&ix->lm_codes, bytes);
    if (e != cudaSuccess) { ix->lm_codes = nullptr; return fail(FANN_ENOMEM, "fann_build_list_codes: cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)); }
    const uint32_t chunks = ix->row_bytes >> 4;
    const uint64_t per_launch = 1ull << 26;
    for (uint64_t e0 = 0; e0 < ix->list_entries; e0 += per_launch) {
        const uint64_t n = ix->list_entries - e0 < per_launch ? ix->list_entries - e0 : per_launch;
        list_codes_kernel<<<(unsigned)((n * chunks + 255) / 256), 256, 0, stream>>>(ix->codes, ix->N, ix->row_bytes, ix->list_ids,
                                                                                  e0, n, ix->lm_codes);
        ix->launches++;
    }
    CUDA_TRY(cudaGetLastError());
    return FANN_OK;
}

struct StreamLayout { size_t hdr, counter, counts, offsets, rows, total; };

static void stream_layout(uint32_t B, uint64_t cap, StreamLayout *l)
{
    size_t o = 0;
    l->hdr = o;     o = align_up(o + sizeof(ListsHeader), 256);
    l->counter = o; o = align_up(o + 256, 256);
    l->counts = o;  o = align_up(o + (size_t)B * 4, 256);
    l->offsets = o; o = align_up(o + ((size_t)B + 1) * 8, 256);
    l->rows = o;    o = align_up(o + (size_t)cap * 8 + 16, 256);      // (row, vector-ID) per candidate
    l->total = o;
}

extern "C" size_t fann_search_lists_stream_workspace_bytes(const fann_index *ix, uint32_t B, uint64_t max_total_cands)
{
    if (!ix || B == 0) { fail(FANN_EINVAL, "fann_search_lists_stream_workspace_bytes: bad argument"); return 0; }
    StreamLayout l;
    stream_layout(B, max_total_cands, &l);
    return l.total;
}

__global__ void stream_counts_kernel(const long long *__restrict__ offsets, uint32_t B, uint32_t *__restrict__ counts,
                                     uint32_t *counter, const fann::ListsHeader *hdr)
{
    const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b == 0) *counter = 0;
    if (b < B) counts[b] = hdr->overflow ? 0u : (uint32_t)(offsets[b + 1] - offsets[b]);
}

extern "C" int fann_search_lists_stream(fann_index *ix, const float *lut, uint32_t B, const uint32_t *probes, uint32_t nprobe,
                                        uint64_t max_total_cands, uint32_t k, uint32_t *out_ids, float *out_dists,
                                        uint32_t *out_counts, void *workspace, size_t workspace_bytes, void *stream_)
{
    if (!ix || !lut || !probes || !out_ids || !out_dists) return fail(FANN_EINVAL, "fann_search_lists_stream: NULL argument");
    if (!ix->lm_codes) return fail(FANN_EINVAL, "fann_search_lists_stream: build the list-major copy first (fann_build_list_codes)");
    if (B == 0 || nprobe == 0) return fail(FANN_EINVAL, "fann_search_lists_stream: B or nprobe is 0");
    if (nprobe > FANN_MAX_NPROBE) return fail(FANN_EUNSUPPORTED, "fann_search_lists_stream: nprobe=%u > %u", nprobe, FANN_MAX_NPROBE);
    if (k == 0 || k > FANN_MAX_K) return fail(FANN_EUNSUPPORTED, "fann_search_lists_stream: k=%u not in 1..%u", k, FANN_MAX_K);
    if (!ix->scan_ring) return fail(FANN_EUNSUPPORTED, "fann_search_lists_stream: needs the ring scan (FANN_SCAN_RING=0 is set)");
    if (((uintptr_t)probes & 3) != 0 || ((uintptr_t)lut & 15) != 0) return fail(FANN_EINVAL, "fann_search_lists_stream: misaligned probes or lut");
    StreamLayout l;
    stream_layout(B, max_total_cands, &l);
    if (!workspace || ((uintptr_t)workspace & 255) != 0) return fail(FANN_EWORKSPACE, "workspace is NULL or not 256-byte aligned");
    if (workspace_bytes < l.total) return fail(FANN_EWORKSPACE, "workspace has %zu bytes, %zu needed", workspace_bytes, l.total);
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    char *ws = (char *)workspace;
    ListsHeader *hdr = (ListsHeader *)(ws + l.hdr);
    long long *offsets = (long long *)(ws + l.offsets);
    uint32_t *rows = (uint32_t *)(ws + l.rows), *counts = (uint32_t *)(ws + l.counts), *counter = (uint32_t *)(ws + l.counter);
    lists_count_kernel<<<(B + 7) / 8, 256, 0, stream>>>(ix->list_offsets, ix->n_lists, probes, B, nprobe,
                                                         (unsigned long long *)offsets);
    lists_scan_kernel<<<1, 1024, 0, stream>>>((const unsigned long long *)offsets, B, offsets, hdr,
                                              (unsigned long long)max_total_cands);
    lists_expand_kernel<<<B, kExpandThreads, ((size_t)nprobe + 1) * 4, stream>>>(
        ix->list_offsets, ix->list_ids, ix->n_lists, probes, nprobe, offsets, rows, hdr, 1u, 1u);
    stream_counts_kernel<<<(B + 255) / 256, 256, 0, stream>>>(offsets, B, counts, counter, hdr);
    ix->launches += 4;
    CUDA_TRY(cudaGetLastError());
    Geom g;
    geometry(ix, k, B, max_total_cands, &g, 0, false);
    ScanParams sp;
    sp.codes = ix->lm_codes; sp.M = ix->M; sp.lut = lut; sp.cand_offsets = offsets; sp.uniq_ids = rows; sp.uniq_counts = counts;
    sp.k = k; sp.cap = g.cap; sp.q_begin = 0; sp.q_end = B; sp.counter = counter;
    sp.out_ids = out_ids; sp.out_dists = out_dists; sp.out_counts = out_counts; sp.out_uniq = nullptr;
    sp.parts = 1; sp.part_keys = nullptr; sp.key_src = rows; sp.id_limit = (uint32_t)ix->N;
    int grid = ix->num_sms * scan_ctas_per_sm(ix, g.scan_smem);
    if ((uint32_t)grid > B) grid = (int)B;
    cudaError_t e = launch_scan(ix, grid, g.scan_smem, stream, sp);
    ix->launches++;
    if (e != cudaSuccess) return fail(FANN_ECUDA, "scan kernel launch: %s", cudaGetErrorString(e));
    return FANN_OK;
}

extern "C" int fann_search_lists_stream_status(fann_index *ix, const void *workspace, uint64_t *total_cands, void *stream_)
{
    if (!ix || !workspace) return fail(FANN_EINVAL, "fann_search_lists_stream_status: NULL argument");
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    ListsHeader h;
    CUDA_TRY(cudaMemcpyAsync(&h, workspace, sizeof(h), cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    if (total_cands) *total_cands = h.total;
    if (h.overflow)
        return fail(FANN_EWORKSPACE, "the probed lists hold %llu candidate IDs, the workspace was sized for %llu (max_total_cands)",
                    h.total, h.capacity);
    return FANN_OK;
}

// ---------------------------------------------------------------- NEXT-3: low-latency small-batch serving

// "the remaining HBM space is divided into multiple blocks ... each block is allocated to an
// individual query ... recycled".  A pool is one HBM allocation cut into fixed blocks; a call takes a free block
// (and the stream that belongs to it) and gives it back when its results are on the host.
struct fann_pool {
    fann_index *ix = nullptr;
    char *mem = nullptr;
    size_t block_bytes = 0;
    uint32_t n_blocks = 0, max_B = 0, k_max = 0, dsub = 0, max_nprobe = 0;
    uint64_t max_cands = 0;
    std::vector<cudaStream_t> streams;
    // CUDA graphs of the posting-list form (one per block and call shape): the ten kernel launches and five copies of
    // a call replayed by one cudaGraphLaunch from the block's pinned staging buffer
    struct Graph { uint32_t B, nprobe, k, generation; const float *codebooks; cudaGraphExec_t exec; };
    std::vector<std::vector<Graph>> graphs;        // per block; a block is used by one call at a time
    char *staging = nullptr;                       // pinned host memory, staging_bytes per block
    size_t staging_bytes = 0, st_queries = 0, st_probes = 0, st_ids = 0, st_dists = 0, st_counts = 0, st_hdr = 0;
    bool use_graphs = true;                        // FANN_SMALL_GRAPH=0: plain launches
    std::mutex mu;
    std::condition_variable cv;
    std::vector<uint32_t> free_blocks;
    uint32_t in_use = 0, high_water = 0;
    uint64_t calls = 0, waits = 0;
};

struct BlockLease {
    fann_pool *pool;
    uint32_t id;
    explicit BlockLease(fann_pool *p) : pool(p)
    {
        std::unique_lock<std::mutex> g(p->mu);
        if (p->free_blocks.empty()) { p->waits++; p->cv.wait(g, [&] { return !p->free_blocks.empty(); }); }
        id = p->free_blocks.back();
        p->free_blocks.pop_back();
        p->in_use++; p->calls++;
        if (p->in_use > p->high_water) p->high_water = p->in_use;
    }
    ~BlockLease()
    {
        { std::lock_guard<std::mutex> g(pool->mu); pool->free_blocks.push_back(id); pool->in_use--; }
        pool->cv.notify_one();
    }
    char *mem() const { return pool->mem + (size_t)id * pool->block_bytes; }
    char *staging() const { return pool->staging + (size_t)id * pool->staging_bytes; }
    cudaStream_t stream() const { return pool->streams[id]; }
};

extern "C" int fann_pool_create(fann_index *ix, uint32_t n_blocks, uint32_t max_B, uint64_t max_cands, uint32_t dsub,
                                uint32_t max_nprobe, uint32_t k_max, fann_pool **out)
{
    if (!ix || !out) return fail(FANN_EINVAL, "fann_pool_create: NULL argument");
    *out = nullptr;
    if (!ix->codes) return fail(FANN_EINVAL, "fann_pool_create: load codes first");
    if (n_blocks == 0 || n_blocks > 4096 || max_B == 0 || dsub == 0 || k_max == 0 || k_max > FANN_MAX_K)
        return fail(FANN_EINVAL, "fann_pool_create: n_blocks=%u max_B=%u dsub=%u k_max=%u", n_blocks, max_B, dsub, k_max);
    if (max_nprobe > FANN_MAX_NPROBE) return fail(FANN_EUNSUPPORTED, "fann_pool_create: max_nprobe=%u > %u", max_nprobe, FANN_MAX_NPROBE);
    DeviceGuard guard(ix->device);
    HostScratch h;
    host_scratch_layout(ix, max_B, dsub, max_cands, k_max, &h);
    size_t need = h.total;
    if (max_nprobe) {
        ListsHostScratch lh;
        lists_host_layout(ix, max_B, dsub, max_nprobe, max_cands, k_max, &lh);
        if (lh.total > need) need = lh.total;
    }
    // what depends on the batch size of the call and is not largest at max_B: the partial top-k of the scan parts (at
    // most num_sms x k keys) and the extra dedup items of a small lists-direct batch (at most 2 num_sms, 12 bytes each)
    need = align_up(need + (size_t)ix->num_sms * k_max * 8 + (size_t)2 * ix->num_sms * 12 + 8192, 256);
    fann_pool *p = new fann_pool();
    p->ix = ix; p->block_bytes = need; p->n_blocks = n_blocks; p->max_B = max_B; p->k_max = k_max; p->dsub = dsub;
    p->max_nprobe = max_nprobe; p->max_cands = max_cands;
    cudaError_t e = cudaMalloc(&p->mem, need * n_blocks);
    if (e != cudaSuccess) {
        delete p;
        return fail(FANN_ENOMEM, "fann_pool_create: cudaMalloc(%zu x %u): %s", need, n_blocks, cudaGetErrorString(e));
    }
    for (uint32_t i = 0; i < n_blocks; ++i) {
        cudaStream_t st = nullptr;
        if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess) {
            for (auto s2 : p->streams) cudaStreamDestroy(s2);
            cudaFree(p->mem);
            delete p;
            return fail(FANN_ECUDA, "fann_pool_create: could not create stream %u", i);
        }
        p->streams.push_back(st);
        p->free_blocks.push_back(n_blocks - 1 - i);
    }
    p->graphs.resize(n_blocks);
    if (const char *sg = getenv("FANN_SMALL_GRAPH")) p->use_graphs = atoi(sg) != 0;
    if (max_nprobe && p->use_graphs) {                         // staging for the graph replays of the posting-list form
        size_t o = 0;
        p->st_queries = o; o = align_up(o + (size_t)max_B * ix->M * dsub * 4, 256);
        p->st_probes = o;  o = align_up(o + (size_t)max_B * max_nprobe * 4, 256);
        p->st_ids = o;     o = align_up(o + (size_t)max_B * k_max * 4, 256);
        p->st_dists = o;   o = align_up(o + (size_t)max_B * k_max * 4, 256);
        p->st_counts = o;  o = align_up(o + (size_t)max_B * 4, 256);
        p->st_hdr = o;     o = align_up(o + sizeof(ListsHeader) + sizeof(WsHeader), 256);
        p->staging_bytes = o;
        if (cudaHostAlloc(&p->staging, o * n_blocks, cudaHostAllocDefault) != cudaSuccess) {
            p->staging = nullptr; p->use_graphs = false;       // no pinned memory: plain launches
            cudaGetLastError();
        }
    } else {
        p->use_graphs = false;
    }
    *out = p;
    return FANN_OK;
}

extern "C" void fann_pool_destroy(fann_pool *p)
{
    if (!p) return;
    DeviceGuard guard(p->ix->device);
    for (auto st : p->streams) { cudaStreamSynchronize(st); cudaStreamDestroy(st); }
    for (auto &blk : p->graphs) for (auto &g : blk) cudaGraphExecDestroy(g.exec);
    if (p->staging) cudaFreeHost(p->staging);
    if (p->mem) cudaFree(p->mem);
    delete p;
}

extern "C" int fann_pool_stats(fann_pool *p, fann_pool_info *out)
{
    if (!p || !out) return fail(FANN_EINVAL, "fann_pool_stats: NULL argument");
    std::lock_guard<std::mutex> g(p->mu);
    out->block_bytes = p->block_bytes; out->calls = p->calls; out->waits = p->waits;
    out->n_blocks = p->n_blocks; out->in_use = p->in_use; out->high_water = p->high_water; out->reserved = 0;
    return FANN_OK;
}

extern "C" int fann_search_small(fann_index *ix, fann_pool *pool, const float *queries_h, uint32_t B,
                                 const float *codebooks_d, uint32_t dsub, const int64_t *cand_offsets_h,
                                 const uint32_t *cand_ids_h, uint32_t k, uint32_t *out_ids_h, float *out_dists_h,
                                 uint32_t *out_counts_h)
{
    if (!ix || !pool || pool->ix != ix) return fail(FANN_EINVAL, "fann_search_small: NULL index or a pool of another index");
    if (B == 0 || B > pool->max_B || k == 0 || k > pool->k_max || dsub != pool->dsub)
        return fail(FANN_EINVAL, "fann_search_small: B=%u (pool: %u), k=%u (pool: %u), dsub=%u (pool: %u)", B, pool->max_B, k,
                    pool->k_max, dsub, pool->dsub);
    if (cand_offsets_h && (cand_offsets_h[B] < 0 || (uint64_t)cand_offsets_h[B] > pool->max_cands))
        return fail(FANN_EWORKSPACE, "fann_search_small: %lld candidate IDs, the pool's blocks hold %llu",
                    (long long)cand_offsets_h[B], (unsigned long long)pool->max_cands);
    BlockLease lease(pool);                                    // waits while every block is in use
    return fann_search_host(ix, queries_h, B, codebooks_d, dsub, cand_offsets_h, cand_ids_h, k, out_ids_h, out_dists_h,
                            out_counts_h, lease.mem(), pool->block_bytes, lease.stream());
}

extern "C" int fann_search_small_lists(fann_index *ix, fann_pool *pool, const float *queries_h, uint32_t B,
                                       const float *codebooks_d, uint32_t dsub, const uint32_t *probes_h, uint32_t nprobe,
                                       uint32_t k, uint32_t *out_ids_h, float *out_dists_h, uint32_t *out_counts_h)
{
    if (!ix || !pool || pool->ix != ix) return fail(FANN_EINVAL, "fann_search_small_lists: NULL index or a pool of another index");
    if (B == 0 || B > pool->max_B || k == 0 || k > pool->k_max || dsub != pool->dsub || nprobe == 0 || nprobe > pool->max_nprobe)
        return fail(FANN_EINVAL, "fann_search_small_lists: B=%u (pool: %u), k=%u (pool: %u), dsub=%u (pool: %u), nprobe=%u (pool: %u)",
                    B, pool->max_B, k, pool->k_max, dsub, pool->dsub, nprobe, pool->max_nprobe);
    BlockLease lease(pool);
    if (!pool->use_graphs)
        return fann_search_lists_host(ix, queries_h, B, codebooks_d, dsub, probes_h, nprobe, pool->max_cands, k, out_ids_h,
                                      out_dists_h, out_counts_h, lease.mem(), pool->block_bytes, lease.stream());
    // One cudaGraphLaunch per call: the block's graph for this call shape copies queries and probes up from the
    // block's pinned staging buffer, runs the path and copies results and the two status headers back.
    if (!queries_h || !codebooks_d || !probes_h || !out_ids_h || !out_dists_h)
        return fail(FANN_EINVAL, "fann_search_small_lists: NULL argument");
    if (!ix->codes || !ix->list_offsets) return fail(FANN_EINVAL, "fann_search_small_lists: load codes and posting lists first");
    DeviceGuard guard(ix->device);
    cudaStream_t stream = lease.stream();
    char *st = lease.staging(), *s = lease.mem();
    const size_t qbytes = (size_t)B * ix->M * dsub * 4, pbytes = (size_t)B * nprobe * 4, obytes = (size_t)B * k * 4;
    memcpy(st + pool->st_queries, queries_h, qbytes);
    memcpy(st + pool->st_probes, probes_h, pbytes);
    ListsHostScratch h;
    lists_host_layout(ix, B, dsub, nprobe, pool->max_cands, k, &h);
    if (h.total > pool->block_bytes)
        return fail(FANN_EWORKSPACE, "fann_search_small_lists: the call needs %zu bytes, a block of the pool has %zu", h.total, pool->block_bytes);
    ListsLayout l;
    lists_layout(ix, B, pool->max_cands, k, &l);
    cudaGraphExec_t exec = nullptr;
    const uint32_t gen = ix->generation.load();
    auto &cache = pool->graphs[lease.id];
    for (size_t i = 0; i < cache.size();) {                    // graphs captured before codes or lists were reloaded are stale
        if (cache[i].generation != gen) { cudaGraphExecDestroy(cache[i].exec); cache.erase(cache.begin() + i); }
        else ++i;
    }
    for (auto &g : cache)
        if (g.B == B && g.nprobe == nprobe && g.k == k && g.codebooks == codebooks_d) exec = g.exec;
    if (!exec) {
        // results: written by the kernels straight into the block's pinned staging buffer (its device address)
        char *o = ix->host_direct ? (char *)mapped_host_ptr(st) : nullptr;
        const bool direct = o != nullptr;
        CUDA_TRY(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal));
        int rc = FANN_OK;
        cudaError_t ce = cudaMemcpyAsync(s + h.queries, st + pool->st_queries, qbytes, cudaMemcpyHostToDevice, stream);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(s + h.probes, st + pool->st_probes, pbytes, cudaMemcpyHostToDevice, stream);
        if (ce == cudaSuccess) rc = fann_build_lut(ix, (const float *)(s + h.queries), B, codebooks_d, dsub, (float *)(s + h.lut), stream);
        if (ce == cudaSuccess && rc == FANN_OK)
            rc = search_lists_impl(ix, (const float *)(s + h.lut), B, (const uint32_t *)(s + h.probes), nprobe, pool->max_cands, k,
                                   direct ? (uint32_t *)(o + pool->st_ids) : (uint32_t *)(s + h.out_ids),
                                   direct ? (float *)(o + pool->st_dists) : (float *)(s + h.out_dists),
                                   direct ? (uint32_t *)(o + pool->st_counts) : (uint32_t *)(s + h.out_counts), nullptr,
                                   s + h.ws, l, stream);
        if (!direct) {
            if (ce == cudaSuccess) ce = cudaMemcpyAsync(st + pool->st_ids, s + h.out_ids, obytes, cudaMemcpyDeviceToHost, stream);
            if (ce == cudaSuccess) ce = cudaMemcpyAsync(st + pool->st_dists, s + h.out_dists, obytes, cudaMemcpyDeviceToHost, stream);
            if (ce == cudaSuccess) ce = cudaMemcpyAsync(st + pool->st_counts, s + h.out_counts, (size_t)B * 4, cudaMemcpyDeviceToHost, stream);
        }
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(st + pool->st_hdr, s + h.ws + l.hdr, sizeof(ListsHeader), cudaMemcpyDeviceToHost, stream);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(st + pool->st_hdr + sizeof(ListsHeader), s + h.ws + l.ws, sizeof(WsHeader), cudaMemcpyDeviceToHost, stream);
        cudaGraph_t graph = nullptr;
        cudaError_t ee = cudaStreamEndCapture(stream, &graph);
        if (rc != FANN_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (ce != cudaSuccess || ee != cudaSuccess || !graph) {
            if (graph) cudaGraphDestroy(graph);
            return fail(FANN_ECUDA, "fann_search_small_lists: graph capture: %s", cudaGetErrorString(ce != cudaSuccess ? ce : ee));
        }
        ce = cudaGraphInstantiate(&exec, graph, 0);
        cudaGraphDestroy(graph);
        if (ce != cudaSuccess) return fail(FANN_ECUDA, "fann_search_small_lists: cudaGraphInstantiate: %s", cudaGetErrorString(ce));
        cache.push_back({B, nprobe, k, gen, codebooks_d, exec});
    }
    CUDA_TRY(cudaGraphLaunch(exec, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    const ListsHeader *lh = (const ListsHeader *)(st + pool->st_hdr);
    const WsHeader *wh = (const WsHeader *)(st + pool->st_hdr + sizeof(ListsHeader));
    if (lh->overflow)
        return fail(FANN_EWORKSPACE, "the probed lists hold %llu candidate IDs, the pool's blocks hold %llu", lh->total, lh->capacity);
    if (wh->status & kStatusPlanOverflow) return fail(FANN_EINVAL, "total_cands passed to the call was smaller than cand_offsets[B]");
    if (wh->status & kStatusTableFull) return fail(FANN_EOVERFLOW, "a dedup hash table filled up (colliding candidate IDs)");
    memcpy(out_ids_h, st + pool->st_ids, obytes);
    memcpy(out_dists_h, st + pool->st_dists, obytes);
    if (out_counts_h) memcpy(out_counts_h, st + pool->st_counts, (size_t)B * 4);
    return FANN_OK;
}

// ---------------------------------------------------------------- NEXT-1: heuristic re-ranking

extern "C" int fann_load_vectors(fann_index *ix, const void *vectors, uint64_t first, uint64_t n, uint64_t N_total,
                                 uint32_t d, int elem_type, int src_is_device, void *stream_)
{
    if (!ix || !vectors) return fail(FANN_EINVAL, "fann_load_vectors: NULL argument");
    if (d == 0 || N_total == 0) return fail(FANN_EINVAL, "fann_load_vectors: d and N_total must be > 0");
    if (d > kRerankMaxDim) return fail(FANN_EUNSUPPORTED, "fann_load_vectors: d=%u > %u", d, kRerankMaxDim);
    if (elem_type != FANN_ELEM_F32 && elem_type != FANN_ELEM_U8 && elem_type != FANN_ELEM_I8)
        return fail(FANN_EUNSUPPORTED, "fann_load_vectors: elem_type %d", elem_type);
    if (N_total >= 0xFFFFFFFFull) return fail(FANN_EUNSUPPORTED, "fann_load_vectors: N_total must be < 2^32-1");
    if (first > N_total || n > N_total - first) return fail(FANN_EINVAL, "fann_load_vectors: rows outside N_total");
    const size_t es = elem_type == FANN_ELEM_F32 ? 4 : 1;
    if (((uintptr_t)vectors & (es - 1)) != 0) return fail(FANN_EINVAL, "fann_load_vectors: misaligned source");
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    if (!ix->vectors) {
        cudaError_t e = cudaMalloc(&ix->vectors, (size_t)N_total * d * es);
        if (e != cudaSuccess) { ix->vectors = nullptr; return fail(FANN_ENOMEM, "fann_load_vectors: cudaMalloc: %s", cudaGetErrorString(e)); }
        ix->vec_N = N_total; ix->vec_d = d; ix->vec_elem = elem_type;
    } else if (N_total != ix->vec_N || d != ix->vec_d || elem_type != ix->vec_elem) {
        return fail(FANN_EINVAL, "fann_load_vectors: (N_total, d, elem_type) differ from the first call");
    }
    if (n == 0) return FANN_OK;
    CUDA_TRY(cudaMemcpyAsync((char *)ix->vectors + (size_t)first * d * es, vectors, (size_t)n * d * es,
                             src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, stream));
    if (!src_is_device) CUDA_TRY(cudaStreamSynchronize(stream));
    return FANN_OK;
}

extern "C" int fann_rerank(fann_index *ix, const float *queries, uint32_t B, const uint32_t *task_ids, uint32_t n,
                           uint32_t batch_size, uint32_t k, float eps, uint32_t beta, uint32_t *out_ids, float *out_dists,
                           uint32_t *out_counts, uint32_t *out_batches, uint32_t *out_reads, void *stream_)
{
    if (!ix || !queries || !task_ids || !out_ids || !out_dists || !out_counts)
        return fail(FANN_EINVAL, "fann_rerank: NULL argument");
    if (!ix->vectors) return fail(FANN_EINVAL, "fann_rerank: load the raw vectors first (fann_load_vectors)");
    if (B == 0 || n == 0 || batch_size == 0 || k == 0 || beta == 0)
        return fail(FANN_EINVAL, "fann_rerank: B, n, batch_size, k and beta must be > 0");
    if (k > kRerankMaxK || n > kRerankMaxTasks)
        return fail(FANN_EUNSUPPORTED, "fann_rerank: k=%u (max %u), n=%u (max %u)", k, kRerankMaxK, n, kRerankMaxTasks);
    if (!(eps >= 0.f)) return fail(FANN_EINVAL, "fann_rerank: eps must be >= 0");
    if ((((uintptr_t)queries | (uintptr_t)task_ids | (uintptr_t)out_ids | (uintptr_t)out_dists | (uintptr_t)out_counts |
          (uintptr_t)out_batches | (uintptr_t)out_reads) & 3) != 0)
        return fail(FANN_EINVAL, "fann_rerank: arrays must be 4-byte aligned");
    if (batch_size > kRerankMaxBatch) batch_size = kRerankMaxBatch > n ? n : kRerankMaxBatch;
    if (batch_size > n) batch_size = n;                         // one mini-batch holds every task
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    RerankParams p;
    p.vectors = ix->vectors; p.N = ix->vec_N; p.d = ix->vec_d; p.queries = queries; p.tasks = task_ids;
    p.n = n; p.batch_size = batch_size; p.k = k; p.beta = beta; p.eps = eps;
    p.out_ids = out_ids; p.out_dists = out_dists; p.out_counts = out_counts; p.out_batches = out_batches; p.out_reads = out_reads;
    const size_t smem = (size_t)((p.d + 3u) & ~3u) * 4 + (size_t)((n + 3u) & ~3u) * 4 + ((size_t)2 * k + batch_size) * 8;
    switch (ix->vec_elem) {
    case FANN_ELEM_F32: rerank_kernel<kElemF32><<<B, kRerankThreads, smem, stream>>>(p); break;
    case FANN_ELEM_U8:  rerank_kernel<kElemU8><<<B, kRerankThreads, smem, stream>>>(p); break;
    default:            rerank_kernel<kElemI8><<<B, kRerankThreads, smem, stream>>>(p); break;
    }
    ix->launches++;
    CUDA_TRY(cudaGetLastError());
    return FANN_OK;
}

// ---------------------------------------------------------------- NEXT-4: page-level I/O dedup

extern "C" int fann_load_page_table(fann_index *ix, const uint32_t *page_of, uint64_t N, uint64_t n_pages,
                                    int src_is_device, void *stream_)
{
    if (!ix || !page_of) return fail(FANN_EINVAL, "fann_load_page_table: NULL argument");
    if (N == 0 || N >= 0xFFFFFFFFull || n_pages == 0 || n_pages >= 0xFFFFFFFFull)
        return fail(FANN_EINVAL, "fann_load_page_table: N and n_pages must be in 1 .. 2^32-2");
    if (((uintptr_t)page_of & 3) != 0) return fail(FANN_EINVAL, "fann_load_page_table: page_of must be 4-byte aligned");
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    if (ix->page_of) { cudaFree(ix->page_of); ix->page_of = nullptr; ix->page_N = 0; }
    cudaError_t e = cudaMalloc(&ix->page_of, N * 4);
    if (e != cudaSuccess) { ix->page_of = nullptr; return fail(FANN_ENOMEM, "fann_load_page_table: cudaMalloc: %s", cudaGetErrorString(e)); }
    CUDA_TRY(cudaMemcpyAsync(ix->page_of, page_of, N * 4, src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, stream));
    if (!src_is_device) CUDA_TRY(cudaStreamSynchronize(stream));
    ix->page_N = N; ix->n_pages = n_pages;
    return FANN_OK;
}

extern "C" int fann_page_reads(fann_index *ix, const uint32_t *task_ids, uint32_t B, uint32_t n, uint32_t batch_size,
                               const uint32_t *batches_run, const uint32_t *resident_bits, uint32_t *out_pages,
                               uint32_t *out_batch_reads, uint32_t *out_total, void *stream_)
{
    if (!ix || !task_ids || !out_pages || !out_batch_reads || !out_total)
        return fail(FANN_EINVAL, "fann_page_reads: NULL argument");
    if (!ix->page_of) return fail(FANN_EINVAL, "fann_page_reads: load the vector -> page table first (fann_load_page_table)");
    if (B == 0 || n == 0 || batch_size == 0) return fail(FANN_EINVAL, "fann_page_reads: B, n and batch_size must be > 0");
    if (n > kPageMaxTasks) return fail(FANN_EUNSUPPORTED, "fann_page_reads: n=%u > %u", n, kPageMaxTasks);
    if ((((uintptr_t)task_ids | (uintptr_t)batches_run | (uintptr_t)resident_bits | (uintptr_t)out_pages |
          (uintptr_t)out_batch_reads | (uintptr_t)out_total) & 3) != 0)
        return fail(FANN_EINVAL, "fann_page_reads: arrays must be 4-byte aligned");
    if (batch_size > n) batch_size = n;
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    PageParams p;
    p.page_of = ix->page_of; p.N = ix->page_N; p.n_pages = ix->n_pages; p.tasks = task_ids; p.n = n;
    p.batch_size = batch_size; p.n_batches = (n + batch_size - 1) / batch_size; p.batches_run = batches_run;
    p.resident = resident_bits; p.out_pages = out_pages; p.out_batch_reads = out_batch_reads; p.out_total = out_total;
    uint32_t slots = 64;
    while (slots < 2 * n) slots <<= 1;
    page_reads_kernel<<<B, kPageThreads, (size_t)slots * 4, stream>>>(p, slots);
    ix->launches++;
    CUDA_TRY(cudaGetLastError());
    return FANN_OK;
}

// ---------------------------------------------------------------- measurement

extern "C" int fann_set_timing(fann_index *ix, int enable)
{
    if (!ix) return fail(FANN_EINVAL, "fann_set_timing: NULL index");
    DeviceGuard guard(ix->device);
    std::lock_guard<std::mutex> tl(ix->timing_mu);
    if (enable) {
        for (auto &e : ix->ev_lut) if (!e) CUDA_TRY(cudaEventCreate(&e));
        for (auto &e : ix->ev_plan) if (!e) CUDA_TRY(cudaEventCreate(&e));
        for (auto &e : ix->ev_part) if (!e) CUDA_TRY(cudaEventCreate(&e));
        for (auto &c : ix->ev_dedup) for (auto &e : c) if (!e) CUDA_TRY(cudaEventCreate(&e));
        for (auto &c : ix->ev_scan) for (auto &e : c) if (!e) CUDA_TRY(cudaEventCreate(&e));
    }
    ix->timing.store(enable != 0);
    ix->have_lut = ix->have_scan = ix->have_part = false;
    ix->timed_chunks = 0; ix->timed_scan = false;
    return FANN_OK;
}

extern "C" int fann_last_timing(fann_index *ix, float *lut_ms, float *plan_ms, float *partition_ms, float *dedup_ms,
                                float *scan_ms)
{
    if (!ix) return fail(FANN_EINVAL, "fann_last_timing: NULL index");
    DeviceGuard guard(ix->device);
    std::lock_guard<std::mutex> tl(ix->timing_mu);
    float v[5] = {-1.f, -1.f, -1.f, -1.f, -1.f};
    if (ix->have_lut) { CUDA_TRY(cudaEventSynchronize(ix->ev_lut[1])); CUDA_TRY(cudaEventElapsedTime(&v[0], ix->ev_lut[0], ix->ev_lut[1])); }
    if (ix->have_part) { CUDA_TRY(cudaEventSynchronize(ix->ev_part[1])); CUDA_TRY(cudaEventElapsedTime(&v[4], ix->ev_part[0], ix->ev_part[1])); }
    if (ix->have_scan && ix->timed_chunks) {
        CUDA_TRY(cudaEventSynchronize(ix->ev_plan[1]));
        CUDA_TRY(cudaEventElapsedTime(&v[1], ix->ev_plan[0], ix->ev_plan[1]));
        v[2] = 0.f;
        for (uint32_t c = 0; c < ix->timed_chunks; ++c) {
            float t = 0.f;
            CUDA_TRY(cudaEventSynchronize(ix->ev_dedup[c][1]));
            CUDA_TRY(cudaEventElapsedTime(&t, ix->ev_dedup[c][0], ix->ev_dedup[c][1]));
            v[2] += t;
        }
        if (ix->timed_scan) {
            v[3] = 0.f;
            for (uint32_t c = 0; c < ix->timed_chunks; ++c) {
                float t = 0.f;
                CUDA_TRY(cudaEventSynchronize(ix->ev_scan[c][1]));
                CUDA_TRY(cudaEventElapsedTime(&t, ix->ev_scan[c][0], ix->ev_scan[c][1]));
                v[3] += t;
            }
        }
    }
    if (lut_ms) *lut_ms = v[0];
    if (plan_ms) *plan_ms = v[1];
    if (partition_ms) *partition_ms = v[4];
    if (dedup_ms) *dedup_ms = v[2];
    if (scan_ms) *scan_ms = v[3];
    return FANN_OK;
}
