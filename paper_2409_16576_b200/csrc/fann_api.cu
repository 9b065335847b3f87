// fann_api.cu -- the C ABI of include/fann.h: argument checks, workspace
// layout, launch geometry, kernel launches.  No compute happens on the host.
#include "../../include/fann.h"
#include "fann_kernels.cuh"

#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>

using namespace fann;

struct fann_index {
    int device = 0;
    uint64_t N = 0;
    uint32_t M = 0, row_bytes = 0;
    uint8_t *codes = nullptr;              // [N][row_bytes]
    uint8_t *bounce = nullptr;             // staging for host-sourced code chunks
    size_t bounce_bytes = 0;
    int num_sms = 0;
    int smem_optin = 0;                    // max dynamic shared memory per block
    uint32_t ipt = 2;                      // candidate IDs per thread per block-synchronous step
    uint64_t launches = 0;
    // geometry of the last scan launch (fann_get_info)
    uint32_t last_ctas = 0, last_smem = 0, last_slots = 0;
    // optional per-kernel timing: events 0/1 lut, 2/3 plan, 3/4 scan, 4/5 merge
    bool timing = false;
    cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    bool ev_lut = false, ev_scan = false, ev_merge = false;
};

static inline void rec(fann_index *ix, int i, cudaStream_t s) { if (ix->timing) cudaEventRecord(ix->ev[i], s); }

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

static uint32_t next_pow2(uint32_t v)
{
    uint32_t p = 1;
    while (p < v) p <<= 1;
    return p;
}

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ---------------------------------------------------------------- geometry + workspace layout

struct ScanGeom {
    uint32_t KP, capbuf, ipt, nslots, cap_c, smem_bytes;
};

static int scan_geometry(const fann_index *ix, uint32_t k, ScanGeom *g)
{
    g->ipt = ix->ipt;
    g->KP = next_pow2(k < 32 ? 32 : k);
    g->capbuf = next_pow2(k + kScanThreads * (g->ipt + 1));
    const size_t fixed = scan_smem_bytes(g->capbuf, ix->row_bytes, 0);
    if (fixed + 4096 * 4 > (size_t)ix->smem_optin)
        return fail(FANN_EUNSUPPORTED, "shared memory: %zu bytes fixed + table > %d", fixed, ix->smem_optin);
    g->nslots = (uint32_t)(((size_t)ix->smem_optin - fixed) / 4) & ~3u;
    g->cap_c = (uint32_t)((uint64_t)g->nslots * 4 / 5);          // <= 80 % load even with no repeats
    g->smem_bytes = (uint32_t)scan_smem_bytes(g->capbuf, ix->row_bytes, g->nslots);
    return FANN_OK;
}

struct WsLayout {
    size_t hdr, S, item_start, items, part_count, part_uniq, part_keys, total;
    uint32_t max_items;
};

static void ws_layout(uint32_t B, uint64_t total_cands, const ScanGeom &g, WsLayout *w)
{
    const uint64_t max_items = (uint64_t)B + total_cands / g.cap_c + 1;
    w->max_items = (uint32_t)(max_items > 0xFFFFFFF0ull ? 0xFFFFFFF0ull : max_items);
    size_t o = 0;
    w->hdr = o;        o = align_up(o + 256, 256);
    w->S = o;          o = align_up(o + (size_t)B * 4, 256);
    w->item_start = o; o = align_up(o + ((size_t)B + 1) * 4, 256);
    w->items = o;      o = align_up(o + (size_t)w->max_items * 8, 256);
    w->part_count = o; o = align_up(o + (size_t)w->max_items * 4, 256);
    w->part_uniq = o;  o = align_up(o + (size_t)w->max_items * 4, 256);
    w->part_keys = o;  o = align_up(o + (size_t)w->max_items * g.KP * 8, 256);
    w->total = o;
}

// ---------------------------------------------------------------- lifecycle

extern "C" const char *fann_last_error(void) { return g_err; }
extern "C" const char *fann_version(void) { return "fann 0.1 sm_100a"; }

template <int NCHUNK>
static cudaError_t set_scan_attrs(int smem)
{
    cudaError_t e = cudaFuncSetAttribute(scan_kernel<NCHUNK, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(scan_kernel<NCHUNK, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
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
    CUDA_TRY(set_scan_attrs<1>(smem_optin));
    CUDA_TRY(set_scan_attrs<2>(smem_optin));
    CUDA_TRY(set_scan_attrs<3>(smem_optin));
    CUDA_TRY(set_scan_attrs<4>(smem_optin));
    fann_index *ix = new fann_index();
    ix->device = device; ix->num_sms = num_sms; ix->smem_optin = smem_optin;
    if (const char *s = getenv("FANN_IPT")) { int v = atoi(s); if (v >= 1 && v <= 4) ix->ipt = (uint32_t)v; }
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
    for (auto &e : ix->ev) if (e) cudaEventDestroy(e);
    delete ix;
}

extern "C" int fann_get_info(const fann_index *ix, fann_info *out)
{
    if (!ix || !out) return fail(FANN_EINVAL, "fann_get_info: NULL argument");
    out->N = ix->N; out->M = ix->M; out->row_bytes = ix->row_bytes;
    out->num_sms = (uint32_t)ix->num_sms; out->scan_threads = kScanThreads;
    out->scan_ctas = ix->last_ctas; out->scan_smem_bytes = ix->last_smem; out->table_slots = ix->last_slots;
    out->kernel_launches = ix->launches;
    return FANN_OK;
}

// ---------------------------------------------------------------- fann_load_codes

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
    if (!ix->codes) {
        ix->N = N_total; ix->M = M; ix->row_bytes = (M + 15u) & ~15u;
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
    const uint64_t units = (uint64_t)B * ix->M * 64;
    rec(ix, 0, (cudaStream_t)stream_);
    build_lut_kernel<<<(unsigned)((units + 255) / 256), 256, 0, (cudaStream_t)stream_>>>(
        queries, codebooks, lut, B, ix->M, dsub);
    rec(ix, 1, (cudaStream_t)stream_);
    ix->ev_lut = ix->timing;
    ix->launches++;
    CUDA_TRY(cudaGetLastError());
    return FANN_OK;
}

// ---------------------------------------------------------------- (5)(6)(7)

extern "C" size_t fann_workspace_bytes(const fann_index *ix, uint32_t B, uint64_t total_cands, uint32_t k)
{
    if (!ix || !ix->codes) { fail(FANN_EINVAL, "fann_workspace_bytes: index has no codes"); return 0; }
    if (B == 0 || k == 0 || k > FANN_MAX_K) { fail(FANN_EINVAL, "fann_workspace_bytes: B=%u k=%u", B, k); return 0; }
    ScanGeom g;
    if (scan_geometry(ix, k, &g) != FANN_OK) return 0;
    WsLayout w;
    ws_layout(B, total_cands, g, &w);
    return w.total;
}

template <bool DUMP>
static cudaError_t launch_scan(uint32_t nchunk, int grid, size_t smem, cudaStream_t stream, const ScanParams &p)
{
    switch (nchunk) {
    case 1: scan_kernel<1, DUMP><<<grid, kScanThreads, smem, stream>>>(p); break;
    case 2: scan_kernel<2, DUMP><<<grid, kScanThreads, smem, stream>>>(p); break;
    case 3: scan_kernel<3, DUMP><<<grid, kScanThreads, smem, stream>>>(p); break;
    default: scan_kernel<4, DUMP><<<grid, kScanThreads, smem, stream>>>(p); break;
    }
    return cudaGetLastError();
}

static int run_scan(fann_index *ix, bool dump, const float *lut, uint32_t B,
                    const int64_t *cand_offsets, const uint32_t *cand_ids, uint64_t total_cands,
                    uint32_t k, uint32_t *out_ids, float *out_dists, uint32_t *out_counts,
                    uint32_t *out_uniq, uint32_t *uniq_ids, uint32_t *uniq_counts,
                    void *workspace, size_t workspace_bytes, cudaStream_t stream)
{
    ScanGeom g;
    int rc = scan_geometry(ix, k, &g);
    if (rc != FANN_OK) return rc;
    WsLayout w;
    ws_layout(B, total_cands, g, &w);
    if (!workspace || ((uintptr_t)workspace & 255) != 0)
        return fail(FANN_EWORKSPACE, "workspace is NULL or not 256-byte aligned");
    if (workspace_bytes < w.total)
        return fail(FANN_EWORKSPACE, "workspace has %zu bytes, %zu needed", workspace_bytes, w.total);
    DeviceGuard guard(ix->device);
    char *ws = (char *)workspace;
    WsHeader *hdr = (WsHeader *)(ws + w.hdr);
    uint32_t *S = (uint32_t *)(ws + w.S);
    uint32_t *item_start = (uint32_t *)(ws + w.item_start);
    uint2 *items = (uint2 *)(ws + w.items);

    rec(ix, 2, stream);
    plan_kernel<<<1, 1024, 0, stream>>>((const long long *)cand_offsets, B, g.cap_c, w.max_items, hdr, S,
                                        item_start, items, dump ? uniq_counts : nullptr);
    ix->launches++;
    CUDA_TRY(cudaGetLastError());

    ScanParams p;
    p.codes = ix->codes; p.N = ix->N; p.row_bytes = ix->row_bytes; p.lut = lut; p.M = ix->M;
    p.cand_offsets = (const long long *)cand_offsets; p.cand_ids = cand_ids;
    p.k = k; p.KP = g.KP; p.capbuf = g.capbuf; p.ipt = g.ipt; p.nslots = g.nslots;
    p.hdr = hdr; p.S = S; p.items = items;
    p.part_count = (uint32_t *)(ws + w.part_count);
    p.part_uniq = (uint32_t *)(ws + w.part_uniq);
    p.part_keys = (unsigned long long *)(ws + w.part_keys);
    p.uniq_ids = uniq_ids; p.uniq_counts = uniq_counts;
    const int grid = ix->num_sms;                                   // persistent: one CTA per SM
    rec(ix, 3, stream);
    cudaError_t e = dump ? launch_scan<true>(ix->row_bytes >> 4, grid, g.smem_bytes, stream, p)
                         : launch_scan<false>(ix->row_bytes >> 4, grid, g.smem_bytes, stream, p);
    ix->launches++;
    if (e != cudaSuccess) return fail(FANN_ECUDA, "scan kernel launch: %s", cudaGetErrorString(e));
    ix->last_ctas = (uint32_t)grid; ix->last_smem = g.smem_bytes; ix->last_slots = g.nslots;
    rec(ix, 4, stream);
    ix->ev_scan = ix->timing; ix->ev_merge = false;
    if (!dump) {
        merge_kernel<<<B, 256, (size_t)2 * g.KP * 8, stream>>>(k, g.KP, hdr, S, item_start, p.part_uniq,
                                                               p.part_keys, out_ids, out_dists, out_counts, out_uniq);
        rec(ix, 5, stream);
        ix->ev_merge = ix->timing;
        ix->launches++;
        CUDA_TRY(cudaGetLastError());
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
    return run_scan(ix, false, lut, B, cand_offsets, cand_ids, total_cands, k, out_ids, out_dists,
                    out_counts, out_uniq, nullptr, nullptr, workspace, workspace_bytes, (cudaStream_t)stream);
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
    return run_scan(ix, true, nullptr, B, cand_offsets, cand_ids, total_cands, 1, nullptr, nullptr,
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

// ---------------------------------------------------------------- host-buffer entry

struct HostScratch {
    size_t queries, offsets, ids, lut, out_ids, out_dists, out_counts, ws, ws_bytes, total;
};

static int host_scratch_layout(const fann_index *ix, uint32_t B, uint32_t dsub, uint64_t total_cands,
                               uint32_t k, HostScratch *h)
{
    ScanGeom g;
    int rc = scan_geometry(ix, k, &g);
    if (rc != FANN_OK) return rc;
    WsLayout w;
    ws_layout(B, total_cands, g, &w);
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
    return FANN_OK;
}

extern "C" size_t fann_search_host_scratch_bytes(const fann_index *ix, uint32_t B, uint32_t dsub,
                                                 uint64_t total_cands, uint32_t k)
{
    if (!ix || !ix->codes || B == 0 || dsub == 0 || k == 0 || k > FANN_MAX_K) {
        fail(FANN_EINVAL, "fann_search_host_scratch_bytes: bad argument");
        return 0;
    }
    HostScratch h;
    if (host_scratch_layout(ix, B, dsub, total_cands, k, &h) != FANN_OK) return 0;
    return h.total;
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
    int rc = host_scratch_layout(ix, B, dsub, total, k, &h);
    if (rc != FANN_OK) return rc;
    if (!device_scratch || ((uintptr_t)device_scratch & 255) != 0 || scratch_bytes < h.total)
        return fail(FANN_EWORKSPACE, "fann_search_host: scratch has %zu bytes, %zu needed (256-byte aligned)",
                    scratch_bytes, h.total);
    DeviceGuard guard(ix->device);
    cudaStream_t stream = (cudaStream_t)stream_;
    char *s = (char *)device_scratch;
    CUDA_TRY(cudaMemcpyAsync(s + h.queries, queries_h, (size_t)B * ix->M * dsub * 4, cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(s + h.offsets, cand_offsets_h, ((size_t)B + 1) * 8, cudaMemcpyHostToDevice, stream));
    if (total)
        CUDA_TRY(cudaMemcpyAsync(s + h.ids, cand_ids_h, (size_t)total * 4, cudaMemcpyHostToDevice, stream));
    rc = fann_build_lut(ix, (const float *)(s + h.queries), B, codebooks_d, dsub, (float *)(s + h.lut), stream);
    if (rc != FANN_OK) return rc;
    rc = fann_dedup_scan_topk(ix, (const float *)(s + h.lut), B, (const int64_t *)(s + h.offsets),
                              (const uint32_t *)(s + h.ids), total, k, (uint32_t *)(s + h.out_ids),
                              (float *)(s + h.out_dists), (uint32_t *)(s + h.out_counts), nullptr,
                              s + h.ws, h.ws_bytes, stream);
    if (rc != FANN_OK) return rc;
    CUDA_TRY(cudaMemcpyAsync(out_ids_h, s + h.out_ids, (size_t)B * k * 4, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaMemcpyAsync(out_dists_h, s + h.out_dists, (size_t)B * k * 4, cudaMemcpyDeviceToHost, stream));
    if (out_counts_h)
        CUDA_TRY(cudaMemcpyAsync(out_counts_h, s + h.out_counts, (size_t)B * 4, cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    return fann_workspace_status(ix, s + h.ws, stream);
}

// ---------------------------------------------------------------- timing

extern "C" int fann_set_timing(fann_index *ix, int enable)
{
    if (!ix) return fail(FANN_EINVAL, "fann_set_timing: NULL index");
    DeviceGuard guard(ix->device);
    if (enable)
        for (auto &e : ix->ev)
            if (!e) CUDA_TRY(cudaEventCreate(&e));
    ix->timing = enable != 0;
    ix->ev_lut = ix->ev_scan = ix->ev_merge = false;
    return FANN_OK;
}

extern "C" int fann_last_timing(fann_index *ix, float *lut_ms, float *plan_ms, float *scan_ms, float *merge_ms)
{
    if (!ix) return fail(FANN_EINVAL, "fann_last_timing: NULL index");
    DeviceGuard guard(ix->device);
    float v[4] = {-1.f, -1.f, -1.f, -1.f};
    if (ix->ev_lut) { CUDA_TRY(cudaEventSynchronize(ix->ev[1])); CUDA_TRY(cudaEventElapsedTime(&v[0], ix->ev[0], ix->ev[1])); }
    if (ix->ev_scan) {
        CUDA_TRY(cudaEventSynchronize(ix->ev[4]));
        CUDA_TRY(cudaEventElapsedTime(&v[1], ix->ev[2], ix->ev[3]));
        CUDA_TRY(cudaEventElapsedTime(&v[2], ix->ev[3], ix->ev[4]));
    }
    if (ix->ev_merge) { CUDA_TRY(cudaEventSynchronize(ix->ev[5])); CUDA_TRY(cudaEventElapsedTime(&v[3], ix->ev[4], ix->ev[5])); }
    if (lut_ms) *lut_ms = v[0];
    if (plan_ms) *plan_ms = v[1];
    if (scan_ms) *scan_ms = v[2];
    if (merge_ms) *merge_ms = v[3];
    return FANN_OK;
}
