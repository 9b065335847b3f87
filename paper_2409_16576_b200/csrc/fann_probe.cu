// fann_probe.cu -- MEASUREMENT ONLY (include/fann_probe.h).  Built by bench.py into libfann_probe.so; the
// product library libfann.so holds none of this.  Kernels that read code rows by ID and do nothing else:
// the row-gather ceiling of step (6), with five ways of issuing the reads.
#include "../../include/fann_probe.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>

namespace {

constexpr int kThreads = 512, kWarps = kThreads / 32;
constexpr int kRingDepth = 3, kStageBytes = 2048;

thread_local char g_err[256] = "";
int fail(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return -1;
}

__device__ __forceinline__ uint4 lds_u128(uint32_t addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}

// ---------------------------------------------------------------- rows through registers

template <int G, int NB, bool L2_64>
__global__ void __launch_bounds__(kThreads) probe_ldg16_kernel(const uint8_t *__restrict__ codes,
                                                               const uint32_t *__restrict__ ids, uint64_t n,
                                                               uint64_t N, uint32_t *sink)
{
    constexpr int ROWB = 16 * G;
    const uint32_t lane = threadIdx.x & 31, q = lane & (G - 1);
    const uint64_t warp_global = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint64_t nwarps = ((uint64_t)gridDim.x * blockDim.x) >> 5;
    uint32_t acc = 0;
    for (uint64_t base = warp_global * 32 * NB; base < n; base += nwarps * 32 * NB) {
        uint32_t id[NB];
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) {
            const uint64_t idx = base + nb * 32 + lane;
            id[nb] = idx < n ? __ldg(ids + idx) : 0u;
            if ((uint64_t)id[nb] >= N) id[nb] = 0;
        }
        uint4 rw[NB][G];
#pragma unroll
        for (int nb = 0; nb < NB; ++nb)
#pragma unroll
            for (int t = 0; t < G; ++t) {
                const uint32_t rid = G == 1 ? id[nb] : __shfl_sync(0xffffffffu, id[nb], (lane & ~(G - 1)) | t);
                const void *p = codes + (uint64_t)rid * ROWB + q * 16;
                uint4 &r = rw[nb][t];
                if (L2_64)
                    asm volatile("ld.global.nc.L1::no_allocate.L2::64B.v4.u32 {%0,%1,%2,%3}, [%4];"
                                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
                else
                    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
            }
#pragma unroll
        for (int nb = 0; nb < NB; ++nb)
#pragma unroll
            for (int t = 0; t < G; ++t) acc ^= rw[nb][t].x ^ rw[nb][t].y ^ rw[nb][t].z ^ rw[nb][t].w;
    }
    if (acc == 0x9E3779B9u) sink[0] = acc;                      // keeps the loads alive; practically never true
}

template <int H, int NB>
__global__ void __launch_bounds__(kThreads) probe_ldg32_kernel(const uint8_t *__restrict__ codes,
                                                               const uint32_t *__restrict__ ids, uint64_t n,
                                                               uint64_t N, uint32_t *sink)
{
    constexpr int ROWB = 32 * H;
    const uint32_t lane = threadIdx.x & 31, q = lane & (H - 1);
    const uint64_t warp_global = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint64_t nwarps = ((uint64_t)gridDim.x * blockDim.x) >> 5;
    uint32_t acc = 0;
    for (uint64_t base = warp_global * 32 * NB; base < n; base += nwarps * 32 * NB) {
        uint32_t id[NB];
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) {
            const uint64_t idx = base + nb * 32 + lane;
            id[nb] = idx < n ? __ldg(ids + idx) : 0u;
            if ((uint64_t)id[nb] >= N) id[nb] = 0;
        }
        uint32_t rw[NB][H][8];
#pragma unroll
        for (int nb = 0; nb < NB; ++nb)
#pragma unroll
            for (int t = 0; t < H; ++t) {
                const uint32_t rid = H == 1 ? id[nb] : __shfl_sync(0xffffffffu, id[nb], (lane & ~(H - 1)) | t);
                const void *p = codes + (uint64_t)rid * ROWB + q * 32;
                uint32_t *r = rw[nb][t];
                asm volatile("ld.global.nc.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                             : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "l"(p));
            }
#pragma unroll
        for (int nb = 0; nb < NB; ++nb)
#pragma unroll
            for (int t = 0; t < H; ++t)
#pragma unroll
                for (int e = 0; e < 8; ++e) acc ^= rw[nb][t][e];
    }
    if (acc == 0x9E3779B9u) sink[0] = acc;
}

// ---------------------------------------------------------------- rows through a per-warp shared-memory ring

// Stage st of a warp covers the IDs [ (st * nwarps + warp_global) * RPS, +RPS ), RPS = 2048 / ROWB rows.
template <int G>
__global__ void __launch_bounds__(kThreads) probe_cpasync_kernel(const uint8_t *__restrict__ codes,
                                                                 const uint32_t *__restrict__ ids, uint64_t n,
                                                                 uint64_t N, uint32_t *sink)
{
    constexpr int ROWB = 16 * G, IPL = 4 / G, RPS = 32 * IPL, D = kRingDepth;
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5, q = lane & (G - 1), r = lane / G;
    const uint64_t warp_global = (uint64_t)blockIdx.x * kWarps + warp, nwarps = (uint64_t)gridDim.x * kWarps;
    const uint32_t ring = (uint32_t)__cvta_generic_to_shared(smem) + warp * (D * kStageBytes);
    const uint64_t n_st = (n + nwarps * RPS - 1) / (nwarps * RPS);
    auto issue = [&](uint64_t st) {
        const uint64_t base = (st * nwarps + warp_global) * RPS;
        if (st < n_st && base < n) {
            const uint32_t sa = ring + (uint32_t)(st % D) * kStageBytes;
#pragma unroll
            for (int nb = 0; nb < IPL; ++nb) {
                const uint64_t idx = base + nb * 32 + lane;
                uint32_t id = idx < n ? __ldg(ids + idx) : 0u;
                if ((uint64_t)id >= N) id = 0;
#pragma unroll
                for (int t = 0; t < G; ++t) {
                    const uint32_t rid = G == 1 ? id : __shfl_sync(0xffffffffu, id, (lane & ~(G - 1)) | t);
                    asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;"
                                 :: "r"(sa + (nb * 32 + t * (32 / G) + r) * ROWB + q * 16),
                                    "l"(codes + (uint64_t)rid * ROWB + q * 16) : "memory");
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    uint32_t acc = 0;
#pragma unroll
    for (int d = 0; d < D - 1; ++d) issue(d);
    for (uint64_t st = 0; st < n_st; ++st) {
        issue(st + D - 1);
        asm volatile("cp.async.wait_group %0;" :: "n"(D - 1) : "memory");
        __syncwarp();
        if ((st * nwarps + warp_global) * RPS < n) {
            const uint32_t sa = ring + (uint32_t)(st % D) * kStageBytes + lane * 64;
#pragma unroll
            for (int i = 0; i < 4; ++i) { const uint4 v = lds_u128(sa + i * 16); acc ^= v.x ^ v.y ^ v.z ^ v.w; }
        }
        __syncwarp();
    }
    if (acc == 0x9E3779B9u) sink[0] = acc;
}

// sm_100 cp.async.bulk.tensor.2d ... tile::gather4: four arbitrary rows of a 2-D tensor per instruction.  The
// tensor is [N][ROWB] bytes with a box of one row; lane j of a warp issues the copy of rows 4j .. 4j+3 of the
// stage.  One mbarrier per stage counts the bytes (complete_tx).
template <int ROWB>
__global__ void __launch_bounds__(kThreads) probe_tma_gather4_kernel(const __grid_constant__ CUtensorMap tmap,
                                                                     const uint32_t *__restrict__ ids, uint64_t n,
                                                                     uint64_t N, uint32_t *sink)
{
    constexpr int IPL = 64 / ROWB, RPS = 32 * IPL, NI = RPS / 4, D = kRingDepth;   // IPL 1/2/4, NI 8/16/32
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint64_t warp_global = (uint64_t)blockIdx.x * kWarps + warp, nwarps = (uint64_t)gridDim.x * kWarps;
    const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t ring = smem0 + warp * (D * kStageBytes);
    const uint32_t bars = smem0 + kWarps * D * kStageBytes + warp * (D * 8);
    if (lane < D) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(bars + lane * 8) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    const uint64_t n_st = (n + nwarps * RPS - 1) / (nwarps * RPS);
    auto issue = [&](uint64_t st) {
        const uint64_t base = (st * nwarps + warp_global) * RPS;
        if (st >= n_st || base >= n) return;
        const uint32_t s = (uint32_t)(st % D);
        const uint32_t sa = ring + s * kStageBytes, bar = bars + s * 8;
        uint32_t id[IPL];
#pragma unroll
        for (int nb = 0; nb < IPL; ++nb) {
            const uint64_t idx = base + nb * 32 + lane;
            id[nb] = idx < n ? __ldg(ids + idx) : 0u;
            if ((uint64_t)id[nb] >= N) id[nb] = 0;
        }
        if (lane == 0)
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "n"(kStageBytes) : "memory");
        __syncwarp();
        int32_t rows[4];
#pragma unroll
        for (int rr = 0; rr < 4; ++rr) {
            uint32_t v = 0;
#pragma unroll
            for (int nb = 0; nb < IPL; ++nb) {
                const uint32_t t = __shfl_sync(0xffffffffu, id[nb], (4 * lane + rr) & 31);
                if ((uint32_t)nb == ((4 * lane) >> 5)) v = t;
            }
            rows[rr] = (int32_t)v;
        }
        if (lane < NI)
            asm volatile("cp.async.bulk.tensor.2d.shared::cta.global.tile::gather4.mbarrier::complete_tx::bytes "
                         "[%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
                         :: "r"(sa + lane * 4 * ROWB), "l"(&tmap), "r"(0), "r"(rows[0]), "r"(rows[1]), "r"(rows[2]),
                            "r"(rows[3]), "r"(bar) : "memory");
    };
    uint32_t acc = 0;
#pragma unroll
    for (int d = 0; d < D - 1; ++d) issue(d);
    for (uint64_t st = 0; st < n_st; ++st) {
        issue(st + D - 1);
        if ((st * nwarps + warp_global) * RPS < n) {
            const uint32_t s = (uint32_t)(st % D), parity = (uint32_t)(st / D) & 1u;
            asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                         "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                         "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                         :: "r"(bars + s * 8), "r"(parity) : "memory");
            const uint32_t sa = ring + s * kStageBytes + lane * 64;
#pragma unroll
            for (int i = 0; i < 4; ++i) { const uint4 v = lds_u128(sa + i * 16); acc ^= v.x ^ v.y ^ v.z ^ v.w; }
        }
        __syncwarp();                                          // every lane has read the stage before it is refilled
    }
    if (acc == 0x9E3779B9u) sink[0] = acc;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_row_map(CUtensorMap *map, const uint8_t *codes, uint32_t row_bytes, uint64_t N)
{
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
        return fail("cuTensorMapEncodeTiled is not available: %s", cudaGetErrorString(e));
    const cuuint64_t gdim[2] = {row_bytes, N};
    const cuuint64_t gstride[1] = {row_bytes};
    const cuuint32_t box[2] = {row_bytes, 1};                   // gather4: one row per box, four boxes per instruction
    const cuuint32_t estride[2] = {1, 1};
    CUresult r = ((EncodeTiledFn)fn)(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, (void *)codes, gdim, gstride, box, estride,
                                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                     CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail("cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return 0;
}

}  // namespace

extern "C" const char *fann_probe_last_error(void) { return g_err; }

extern "C" int fann_probe_gather(const uint8_t *codes, uint32_t row_bytes, uint64_t N, const uint32_t *ids, uint64_t n,
                                 uint32_t *sink, uint32_t flavor, uint32_t ctas_per_sm, void *stream_)
{
    if (!codes || !ids || !sink) return fail("fann_probe_gather: NULL argument");
    if (row_bytes != 16 && row_bytes != 32 && row_bytes != 64) return fail("fann_probe_gather: row_bytes %u", row_bytes);
    if (flavor > FANN_PROBE_TMA_GATHER4) return fail("fann_probe_gather: flavor %u", flavor);
    if (flavor == FANN_PROBE_LDG32 && row_bytes < 32) return fail("fann_probe_gather: 32-byte loads need rows >= 32 bytes");
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaStream_t stream = (cudaStream_t)stream_;
    const int grid = sms * (ctas_per_sm ? (int)ctas_per_sm : 1);
    const size_t ring_smem = (size_t)kWarps * kRingDepth * kStageBytes + kWarps * kRingDepth * 8;
#define LAUNCH_RING(K)                                                                                     \
    do {                                                                                                   \
        cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ring_smem);              \
        K<<<grid, kThreads, ring_smem, stream>>>(codes, ids, n, N, sink);                                  \
    } while (0)
    switch (flavor) {
    case FANN_PROBE_LDG16:
        if (row_bytes == 16) probe_ldg16_kernel<1, 8, false><<<grid, kThreads, 0, stream>>>(codes, ids, n, N, sink);
        else if (row_bytes == 32) probe_ldg16_kernel<2, 4, false><<<grid, kThreads, 0, stream>>>(codes, ids, n, N, sink);
        else probe_ldg16_kernel<4, 2, false><<<grid, kThreads, 0, stream>>>(codes, ids, n, N, sink);
        break;
    case FANN_PROBE_LDG16_L2_64:
        if (row_bytes == 16) probe_ldg16_kernel<1, 8, true><<<grid, kThreads, 0, stream>>>(codes, ids, n, N, sink);
        else if (row_bytes == 32) probe_ldg16_kernel<2, 4, true><<<grid, kThreads, 0, stream>>>(codes, ids, n, N, sink);
        else probe_ldg16_kernel<4, 2, true><<<grid, kThreads, 0, stream>>>(codes, ids, n, N, sink);
        break;
    case FANN_PROBE_LDG32:
        if (row_bytes == 32) probe_ldg32_kernel<1, 4><<<grid, kThreads, 0, stream>>>(codes, ids, n, N, sink);
        else probe_ldg32_kernel<2, 2><<<grid, kThreads, 0, stream>>>(codes, ids, n, N, sink);
        break;
    case FANN_PROBE_CPASYNC_RING:
        if (row_bytes == 16) LAUNCH_RING(probe_cpasync_kernel<1>);
        else if (row_bytes == 32) LAUNCH_RING(probe_cpasync_kernel<2>);
        else LAUNCH_RING(probe_cpasync_kernel<4>);
        break;
    default: {
        if (((uintptr_t)codes & 127) != 0) return fail("fann_probe_gather: TMA needs a 128-byte aligned code array");
        CUtensorMap map;
        if (make_row_map(&map, codes, row_bytes, N) != 0) return -1;
#define LAUNCH_TMA(K)                                                                                      \
    do {                                                                                                   \
        cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ring_smem);              \
        K<<<grid, kThreads, ring_smem, stream>>>(map, ids, n, N, sink);                                    \
    } while (0)
        if (row_bytes == 16) LAUNCH_TMA(probe_tma_gather4_kernel<16>);
        else if (row_bytes == 32) LAUNCH_TMA(probe_tma_gather4_kernel<32>);
        else LAUNCH_TMA(probe_tma_gather4_kernel<64>);
        break;
    }
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail("fann_probe_gather: launch failed: %s", cudaGetErrorString(e));
    return 0;
}
