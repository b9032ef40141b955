/*
 * ebic_debug.h -- NOT the boundary.  Knobs, introspection, read-backs of loader products and measurement
 * probes exported by the same libebic.so for the parity tests (tests/) and the benchmark (bench.py).  A user of
 * the library needs include/ebic.h only; nothing here changes a result -- every fitness kernel gives
 * bit-identical counts (tolerance 0), the knobs only select which one runs and how it is tuned.
 * The library reads no environment variable: what the defaults are is stated here and in DESIGN.md 6.4.
 */
#ifndef EBIC_DEBUG_H_
#define EBIC_DEBUG_H_

#include "ebic.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Fitness kernels (all compute include/ebic.h's count[k] exactly). */
enum {
    EBIC_KERNEL_AUTO = 0,      /* PAIRTILE if the tile-major pair table exists and the evaluation is large enough
                                  for staged tiles to pay (>= 4e6 (tile, pair-use) units, more when the
                                  population uses each bit column fewer than 16 times), else PAIRBITS if the pair
                                  table exists, else RANK8 (cols <= 127), else TILED_F32 / UNION_F32 (whichever
                                  applies), else DIRECT                                                        */
    EBIC_KERNEL_DIRECT = 1,    /* one thread per row, column-major global loads (any shape)                    */
    EBIC_KERNEL_TILED_F32 = 2, /* float32 row tiles of ALL columns staged in shared memory by TMA bulk copies  */
    EBIC_KERNEL_RANK8 = 3,     /* per-row order-preserving 8-bit rank tiles (cols <= 127)                      */
    EBIC_KERNEL_PAIRBITS = 4,  /* AND of pair-relation bit columns gathered through L2 (pair table built)      */
    EBIC_KERNEL_UNION_F32 = 5, /* float32 tiles of the COLUMN UNION of a batch of individuals (any cols)       */
    EBIC_KERNEL_PREFIX = 6,    /* PAIRBITS with shared-prefix groups: individuals that start with the same
                                  columns share the AND of those bit columns (population <= 8,192; larger
                                  populations run plain PAIRBITS)                                              */
    EBIC_KERNEL_PAIRTILE = 7   /* 1,024-row tiles of ALL cols^2 bit columns staged in shared memory by TMA and reused
                                  by the whole population, lane = individual (cols <= 42; needs the tile-major copy
                                  of the pair table, which ebic_create builds next to the pair-major one when a
                                  tile fits shared memory)                                                     */
};

/* Selects the fitness kernel.  EBIC_ERR_ARG if it cannot run this shape (RANK8 builds its rank tiles on demand,
 * synchronously; PAIRBITS needs the table: ebic_set_pairbits). */
int ebic_set_kernel(ebic_ctx *ctx, int32_t kernel);

/*
 * Pair-relation table: bit r of pair (a,b) = ( M[r][b] >= M[r][a] ), cols^2 * ceil(rows/1024) * 128 bytes of
 * device memory, one contiguous bit column per ordered pair.  on != 0 builds it if absent (EBIC_ERR_OOM if it
 * does not fit; EBIC_ERR_ARG if cols > 46340 or the table would exceed 64 GiB), on == 0 frees it (and builds
 * the rank tiles if cols <= 127, as ebic_create does when it builds no table).  Where a 1,024-row tile of all
 * cols^2 bit columns fits shared memory (cols <= 42) and memory allows, the build also writes the tile-major copy
 * of the same bits that PAIRTILE stages (as many bytes again; ebic_set_tuning knob 6).  Synchronises the device.
 */
int ebic_set_pairbits(ebic_ctx *ctx, int32_t on);

/* Extraction source: 1 (default) = the pair table when it exists, 0 = always the float32 columns. */
int ebic_set_extract_source(ebic_ctx *ctx, int32_t use_pairbits);

/*
 * Early exit (default on): a warp stops walking a chromosome once none of the rows it holds can still match.
 * Results are identical; only the number of executed visits changes.  Off = every column of every chromosome is
 * visited for every row ("plain work": executed visits == padded rows * sum(L), or * sum(L-1) pair fetches).
 */
int ebic_set_early_exit(ebic_ctx *ctx, int32_t on);

/*
 * Tuning knobs of the launch configuration (DESIGN.md 6.4 says how the defaults were chosen).  `knob`:
 *   0  PAIRBITS warp tasks per resident warp slot (default 12; 1..64): sets the rows per task
 *   1  PAIRBITS L2 prefetch distance in row chunks (default 1; 0 = off, <= 8)
 *   2  PAIRBITS shared-memory landing ring for chromosomes of >= 9 columns (default 1)
 *   3  ingest sorts every block of 64 individuals by length, so the two warps of a PAIRBITS CTA finish together
 *      (default 1)
 *   4  programmatic dependent launch between the ingest, fitness and extraction kernels (default 1)
 *   5  UNION_F32: individuals per batch (default 0 = chosen from the shape; 1..256)
 *   6  the next pair-table build also writes the tile-major copy PAIRTILE needs, when a tile fits (default 1)
 *   7  AUTO picks PAIRTILE from this many (1,024-row tile, consecutive-pair use) units on (default 0 = the rule
 *      stated at EBIC_KERNEL_AUTO)
 *   8  PAIRBITS row chunks requested into L2 by the kernel's prologue (default 1; 1..16, at least the distance)
 *   9  replay a repeated all-device call from a captured CUDA graph (default 1; include/ebic.h, ebic_eval_extract)
 *  10  PAIRBITS on a sparse population (fewer pair uses than 2 * cols^2): bytes of every bit column a record names
 *      that the ingest kernel requests into L2 ahead of the fitness kernel (multiple of 16, <= 1 MiB, capped at one
 *      column; 0 = off; DESIGN.md 6.4 gives the measurement behind the default)
 * EBIC_ERR_ARG for an unknown knob or a value outside its range.
 */
int ebic_set_tuning(ebic_ctx *ctx, int32_t knob, int32_t value);

/*
 * Instrumentation for roofline accounting.  `on` is a bit set:
 *   bit 0  the fitness kernels add the number of (row, column-visit) operand fetches they actually executed --
 *          the PAIRBITS kernel the number of (row, pair) bit fetches -- to a device counter (one extra global
 *          atomic per warp); ebic_get_info(ctx, 10) synchronises the device, returns the counter and resets it.
 *          Never on inside a timed region.
 *   bit 1  every ebic_eval_fitness brackets its fitness kernel launch(es) -- not the ingest kernel -- with a
 *          pair of CUDA events on the call's stream (ring of 256 pairs); the event between the ingest and the
 *          fitness kernel keeps the two from overlapping, so the figure includes the kernel's whole prologue.
 *          ebic_get_info(ctx, 11) synchronises the device and returns the mean duration in ns,
 *          ebic_get_info(ctx, 12) the number of evals timed.  Setting the mode restarts the ring.
 * Off (0) by default.
 */
int ebic_set_instrumentation(ebic_ctx *ctx, int32_t on);

/*
 * Introspection.  `what`:
 *   0 rows, 1 cols, 2 padded leading dimension ld, 3 missing_mode, 4 kernel ebic_eval_fitness will use for a
 *   population shaped like the last one evaluated (before any: 1,600 individuals of 11 columns),
 *   5 rows per tile / per warp task of the last fitness launch, 6 CTAs of that launch, 7 SM count, 8 kernels
 *   launched by this context so far, 9 bytes of device memory the context owns, 10 executed visits since the
 *   last read, 11 mean fitness-kernel time in ns, 12 evals timed (see ebic_set_instrumentation), 13 early exit
 *   on/off, 14 bytes of the pair table (0 = absent), 15 kernel of the last fitness launch (0 = none yet),
 *   16 bytes of the rank tiles (0 = absent), 17 bytes of the tile-major copy of the pair table (0 = absent),
 *   18 kernels in the captured CUDA graph the next identical call would replay (0 = no graph held),
 *   20..24 ebic_create's time in ns, CUDA events on the legacy stream: 20 host-to-device copy + transpose +
 *   padding, 21 NaN bitmask, 22 pair-table kernel, 23 rank-tile kernel (22 / 23 also when built later on demand;
 *   allocations excluded), 24 all of ebic_create including the allocations.
 * Returns -1 for NULL / unknown `what`.
 */
int64_t ebic_get_info(ebic_ctx *ctx, int32_t what);

/*
 * Read-back of loader products for parity tests (synchronous D2H copies on the legacy stream).
 *   what = 0 column-major matrix float32 [cols][ld]; 1 NaN bitmask uint32 [cols][ld/32]; 2 per-column
 *   non-missing counts uint64 [cols]; 3 rank tiles uint8 [cols][ld] (EBIC_ERR_ARG if not built);
 *   4 pair table uint32 [cols*cols][ld/32], pair (a,b) = a*cols + b (EBIC_ERR_ARG if not built);
 *   5 its tile-major copy uint32 [ld/1024][cols*cols][32] (EBIC_ERR_ARG if not built).
 *   dst_bytes must equal the product's size.
 */
int ebic_debug_read(const ebic_ctx *ctx, int32_t what, void *dst, int64_t dst_bytes);

/*
 * Measurement probes (not steps of the path; DESIGN.md 6.1 uses them as roofline denominators next to the
 * figures ncu states).  Each allocates and frees its own memory, runs on the legacy stream, is synchronous,
 * times with CUDA events and returns the best of several passes.  Errors: EBIC_ERR_ARG / _OOM / _CUDA (result 0).
 *
 * ebic_probe_read_bandwidth: GB/s all SMs together read from a device buffer of `buffer_bytes` (>= 1 MiB)
 *   streamed `reps` times with coalesced 128-bit loads that bypass L1, 8 to 16 loads in flight per thread.
 *   A buffer that fits the L2 gives the L2 -> SM bandwidth, one far larger than the L2 gives HBM read bandwidth.
 * ebic_probe_smem_bandwidth: GB/s of conflict-free LDS.128 from shared memory, all SMs (the 128 B/clk/SM data
 *   pipe the tiled kernels are bound by).
 * ebic_probe_smem_gather: GB/s of the PAIRTILE access pattern on its own -- every lane its own pseudo-random
 *   128-byte slot of a 128 KB shared-memory tile, read as eight LDS.128 with the 16-byte unit rotated per lane
 *   (rotate != 0) or not (rotate == 0: the 8-way bank conflicts the rotation removes), AND + popcount as in the
 *   kernel, 16 warps per SM, no staging.
 * ebic_probe_fsetp_rate: ordered float32 compares (FSETP.GE) per second, all SMs, in units of 1e9 lane-compares/s.
 */
int ebic_probe_read_bandwidth(int64_t buffer_bytes, int32_t reps, double *gb_per_s);
int ebic_probe_smem_bandwidth(double *gb_per_s);
int ebic_probe_smem_gather(int32_t rotate, double *gb_per_s);
int ebic_probe_fsetp_rate(double *gcompares_per_s);

#ifdef __cplusplus
}
#endif
#endif /* EBIC_DEBUG_H_ */
