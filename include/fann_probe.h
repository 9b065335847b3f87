/*
 * fann_probe.h -- MEASUREMENT ONLY.  Not part of the product library: built by bench.py into its own
 * shared object (paper_2409_16576_b200/libfann_probe.so) from csrc/fann_probe.cu; libfann.so and fann.h
 * carry none of it.
 *
 * The row-gather ceiling of step (6) ("reads the PQ codes from HBM"): read the stored code
 * rows of ids[0 .. n) and do nothing else.  Timed by the caller, it gives the rate at which this GPU can
 * gather those rows at all, whatever kernel does the arithmetic.
 */
#ifndef FANN_PROBE_H
#define FANN_PROBE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    FANN_PROBE_LDG16      = 0,   /* row_bytes/16 lanes per row, 16-byte ld.global.nc, 8 loads in flight per lane    */
    FANN_PROBE_LDG16_L2_64 = 1,  /* the same with a 64-byte L2 fetch (default fetches 128 bytes per miss)            */
    FANN_PROBE_LDG32      = 2,   /* row_bytes/32 lanes per row, 32-byte ld.global.nc.v8 (row_bytes >= 32)            */
    FANN_PROBE_CPASYNC_RING = 3, /* the scan kernel's fill path: per-warp ring of 3 stages (2 KB each), 16-byte      */
                                 /* cp.async (LDGSTS) with a 64-byte L2 fetch, two stages ahead                     */
    FANN_PROBE_TMA_GATHER4 = 4   /* sm_100 cp.async.bulk.tensor.2d tile::gather4: one lane per warp issues one       */
                                 /* instruction per 4 rows into the same per-warp ring, mbarrier completion         */
};

/*
 * codes      device, [N][row_bytes] uint8 (row_bytes = 16, 32 or 64; 16-byte aligned; for TMA 128-byte aligned base)
 * ids        device, [n] uint32; IDs >= N read row 0
 * sink       device, 4 bytes (keeps the loads alive; never written in practice)
 * ctas_per_sm  512-thread CTAs per SM (0 = 1, the scan kernel's launch shape)
 * Enqueues one kernel on `stream` (a cudaStream_t as void*), returns 0, or a negative value with a message
 * from fann_probe_last_error().
 */
int fann_probe_gather(const uint8_t *codes, uint32_t row_bytes, uint64_t N, const uint32_t *ids, uint64_t n,
                      uint32_t *sink, uint32_t flavor, uint32_t ctas_per_sm, void *stream);
const char *fann_probe_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* FANN_PROBE_H */
