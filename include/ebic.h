/*
 * ebic.h -- C ABI of libebic.so: EBIC population fitness evaluation and matched-row extraction
 * on one NVIDIA B200 (sm_100a).
 *
 * The operation (PAPER.md = arXiv 1807.09932 text; line numbers refer to /root/reference/PAPER.md):
 *   "EBIC search is driven by counting of rows, a greater or equal relation between the values in
 *   columns" and missing values are "no longer counted towards the score of the bicluster"
 *   (section 2 Methods, "Handling missing values"); up to 2^31-1 rows per GPU
 *   and a population of up to 65,535 individuals, 1,600 typical ("Support for
 *   Big Data").  The paper writes no formula; the exact definition used here is the one in
 *   DESIGN.md section 3 (readings R1-R16), identical to the CPU oracle's header:
 *
 *     individual k = ordered column list c_0..c_{L-1} = col_ids[offsets[k] .. offsets[k+1])
 *     ok(k,r)  = AND_{i<L-1} ( M[r][c_{i+1}] >= M[r][c_i] )        IEEE-754 ordered >= on float32
 *                AND ( missing_mode == ON  =>  no M[r][c_i] is NaN )
 *     count[k] = #{ r : ok(k,r) }             mask[k] bit r = ok(k,r)
 *
 * Conventions
 *   - Every function returns a status code (EBIC_OK == 0).  Nothing throws, aborts or prints.
 *   - "device" pointers are CUDA device (or managed) memory of the CURRENT device; "host or device"
 *     pointers are classified with cudaPointerGetAttributes.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - The caller owns every buffer it passes.  The context owns its transposed copy of the matrix,
 *     the NaN bitmask, the rank tiles and its scratch; the input matrix is not retained.
 *   - One call in flight per context at a time (shared scratch).  Different contexts are independent.
 *   - Bit layout of a mask: row r <-> 64-bit word r/64, bit r%64 (LSB first, little endian; the same
 *     bytes viewed as uint8 have row r at byte r/8, bit r%8).  Bits >= rows are zero.
 */
#ifndef EBIC_H_
#define EBIC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ebic_ctx ebic_ctx; /* opaque; owns device memory */

enum {
    EBIC_OK = 0,
    EBIC_ERR_ARG = 1,         /* NULL / non-positive size / unknown mode / bad chosen index       */
    EBIC_ERR_OOM = 2,         /* cudaMalloc failed                                                */
    EBIC_ERR_CUDA = 3,        /* any other CUDA runtime error (no device, launch failure, ...)    */
    EBIC_ERR_BAD_COLUMN = 4,  /* a column id outside [0, cols) was found on the device            */
    EBIC_ERR_BAD_OFFSETS = 5, /* offsets[k] < 0, offsets[k+1] < offsets[k] or offsets[k+1] > n_ids */
    EBIC_ERR_IO = 6           /* ebic_read_delimited: cannot open / not a delimited matrix / ragged line */
};
enum { EBIC_MISSING_OFF = 0, EBIC_MISSING_ON = 1 };

/* Kernel selection for ebic_eval_fitness (all give bit-identical counts). */
enum {
    EBIC_KERNEL_AUTO = 0,    /* fastest applicable: PAIRBITS, RANK8, TILED_F32, DIRECT              */
    EBIC_KERNEL_DIRECT = 1,  /* one thread per row, column-major global loads (any shape)          */
    EBIC_KERNEL_TILED_F32 = 2, /* float32 row tiles staged in shared memory by TMA bulk copies    */
    EBIC_KERNEL_RANK8 = 3,   /* per-row order-preserving 8-bit rank tiles (cols <= 127)           */
    EBIC_KERNEL_PAIRBITS = 4 /* AND of pair-relation bit columns streamed through L2 (pair table built)    */
};

/*
 * Loader (a genes x samples matrix with optional missing values).
 *   matrix        dense ROW-MAJOR float32 [rows][cols]; host or device pointer; any NaN = missing.
 *   rows          1 .. 2^31-1.        cols  1 .. 2^31-1 (memory permitting).
 *   missing_mode  EBIC_MISSING_OFF / EBIC_MISSING_ON.
 *   out           receives the context.
 * Transposes to column-major, builds the packed NaN bitmask and per-column non-missing counts,
 * when cols <= 127 the 8-bit rank tiles and, when it takes at most 8 GiB and half of the free device
 * memory, the pair-relation table (cols^2 bits per padded row; see ebic_set_pairbits).
 * Synchronous: `matrix` may be freed on return.
 * Errors: EBIC_ERR_ARG, EBIC_ERR_OOM, EBIC_ERR_CUDA (then *out == NULL).
 */
int ebic_create(const float *matrix, int64_t rows, int32_t cols, int32_t missing_mode,
                ebic_ctx **out);

/*
 * The same loader for matrices that mark missing cells with a numeric value instead of NaN (PAPER.md
 * line 60: "a predefined numeric value, e.g. 0 or 999"): every element that compares equal to `sentinel`
 * (float ==, so a sentinel of 0 also matches -0) becomes NaN while the matrix is transposed; elements
 * that already are NaN stay missing.  `sentinel` must not be NaN (EBIC_ERR_ARG).  Everything else as
 * ebic_create; with missing_mode OFF the mapped cells still fail every L >= 2 comparison (R4).
 */
int ebic_create_sentinel(const float *matrix, int64_t rows, int32_t cols, int32_t missing_mode,
                         float sentinel, ebic_ctx **out);

/* Frees everything the context owns.  NULL is allowed. */
int ebic_destroy(ebic_ctx *ctx);

/*
 * count[k] for the whole population (population CSR as in BASELINE.json north_star).
 *   offsets  int32 [n_ind+1], col_ids int32 [n_ids]: host or device (both the same kind).
 *   n_ind    0 .. 2^31-2 (0 is a no-op).   n_ids  number of entries of col_ids (>= offsets[n_ind]).
 *   counts   uint64 [n_ind], host or device, overwritten.
 * Asynchronous and stream-ordered when every pointer is a device pointer.  With host pointers the
 * population is copied in and the counts copied out on `cuda_stream`, and the call returns after the
 * stream has been synchronised.
 * Population contents are validated on the device: an individual with a column id outside
 * [0, cols) or with bad offsets gets count 0, the others are unaffected, and a sticky error
 * (EBIC_ERR_BAD_COLUMN / EBIC_ERR_BAD_OFFSETS, the larger code wins) is kept for ebic_status().
 * Returns host-detectable errors only (EBIC_ERR_ARG / _OOM / _CUDA).
 */
int ebic_eval_fitness(ebic_ctx *ctx, const int32_t *offsets, const int32_t *col_ids, int32_t n_ind,
                      int64_t n_ids, uint64_t *counts, void *cuda_stream);

/*
 * Matched-row bitmasks (and optionally counts) of chosen individuals -- the rows of a bicluster
 * (results are biclusters = rows + columns).
 *   chosen   int32 [n_chosen] indices into the CSR population, host or device (same kind as offsets);
 *            an index outside [0, n_ind) yields an all-zero mask and the sticky EBIC_ERR_BAD_OFFSETS.
 *   masks    uint64 [n_chosen][ebic_mask_words(ctx)], host or device, overwritten.
 *   counts   uint64 [n_chosen] or NULL.
 * Same asynchrony, validation and error rules as ebic_eval_fitness.
 */
int ebic_extract_rows(ebic_ctx *ctx, const int32_t *offsets, const int32_t *col_ids, int32_t n_ind,
                      int64_t n_ids, const int32_t *chosen, int32_t n_chosen, uint64_t *masks,
                      uint64_t *counts, void *cuda_stream);

/* ceil(rows / 64): uint64 words per mask.  -1 if ctx is NULL. */
int64_t ebic_mask_words(const ebic_ctx *ctx);

/*
 * Synchronises `cuda_stream`, returns the sticky device error raised since the last ebic_status()
 * (EBIC_OK if none) and clears it.  EBIC_ERR_CUDA if the stream itself reports an error.
 */
int ebic_status(ebic_ctx *ctx, void *cuda_stream);

/* Selects the fitness kernel (EBIC_KERNEL_*).  EBIC_ERR_ARG if it cannot run this shape. */
int ebic_set_kernel(ebic_ctx *ctx, int32_t kernel);

/*
 * Pair-relation table: bit r of pair (a,b) = ( M[r][b] >= M[r][a] ), cols^2 * ceil(rows/1024) * 128
 * bytes of device memory, one contiguous bit column per ordered pair.  With it an L >= 2 chromosome is
 * the AND of its L-1 bit columns (the PAIRBITS kernel; extraction reads it too).  on != 0 builds it if absent (EBIC_ERR_OOM if it does
 * not fit; EBIC_ERR_ARG if cols > 46340 or the table would exceed 64 GiB), on == 0 frees it.  Synchronises the device.
 */
int ebic_set_pairbits(ebic_ctx *ctx, int32_t on);

/* Extraction source: 1 (default) = the pair table when it exists, 0 = always the float32 columns. */
int ebic_set_extract_source(ebic_ctx *ctx, int32_t use_pairbits);

/*
 * Early exit (default on): a warp stops walking a chromosome once none of the rows it holds can still
 * match.  Results are identical; only the number of executed column visits changes (on random
 * populations most rows fail within the first few columns).  Off = every column of every chromosome
 * is visited for every row ("plain work": executed visits == rows * sum(L)).
 */
int ebic_set_early_exit(ebic_ctx *ctx, int32_t on);

/*
 * Instrumentation for roofline accounting.  `on` is a bit set:
 *   bit 0  the tiled fitness kernels add the number of (row, column-visit) operand fetches they
 *          actually executed -- the PAIRBITS kernel the number of (row, pair) bit fetches -- to a
 *          device counter (one extra global atomic per warp);
 *          ebic_get_info(ctx, 10) synchronises the device, returns the counter and resets it.
 *          Never on inside a timed region.
 *   bit 1  every ebic_eval_fitness brackets its fitness kernel launch(es) -- not the ingest kernel --
 *          with a pair of CUDA events on the call's stream (ring of 256 pairs);
 *          ebic_get_info(ctx, 11) synchronises the device and returns their mean duration in ns,
 *          ebic_get_info(ctx, 12) the number of evals timed.  Setting the mode restarts the ring.
 * Off (0) by default.
 */
int ebic_set_instrumentation(ebic_ctx *ctx, int32_t on);

/*
 * Introspection for tests and the benchmark.  `what`:
 *   0 rows, 1 cols, 2 padded leading dimension ld, 3 missing_mode, 4 kernel ebic_eval_fitness will
 *   use, 5 rows per shared-memory tile of that kernel, 6 CTAs of its last launch, 7 SM count,
 *   8 kernels launched by this context so far, 9 bytes of device memory the context owns,
 *   10 executed column visits since the last read, 11 mean fitness-kernel time in ns, 12 evals
 *   timed (see ebic_set_instrumentation), 13 early exit on/off, 14 bytes of the pair table (0 = absent), 15 kernel (EBIC_KERNEL_*)
 *   of the last fitness launch (0 = none yet).
 * Returns -1 for NULL / unknown `what`.
 */
int64_t ebic_get_info(ebic_ctx *ctx, int32_t what);

/*
 * Read-back of loader products for parity tests (synchronous D2H copies on the legacy stream).
 *   ebic_debug_read(ctx, what, dst, dst_bytes): what = 0 column-major matrix float32 [cols][ld];
 *   1 NaN bitmask uint32 [cols][ld/32]; 2 per-column non-missing counts uint64 [cols];
 *   3 rank tiles uint8 [cols][ld] (EBIC_ERR_ARG if not built);
 *   4 pair table uint32 [cols*cols][ld/32], pair (a,b) = a*cols + b (EBIC_ERR_ARG if not built).
 *   dst_bytes must equal the product's size.
 */
int ebic_debug_read(const ebic_ctx *ctx, int32_t what, void *dst, int64_t dst_bytes);

/*
 * Input files ("The data values might be separated by either comma, tabulator or
 * semicolon. An upper left header is not required, which simplifies porting files between EBIC and R").
 * Reads a text matrix on the HOST: line 1 = column names, every later line = a row name followed by the
 * row's values.  `delimiter` is ',', '\t', ';' or 0 = detect from line 1 (a tab wins over a semicolon
 * over a comma).  The upper-left corner label may be present (header has as many fields as a data line)
 * or absent (one fewer, as R's write.table writes it).  Names are skipped and must not contain the
 * delimiter; values are parsed with strtof (correctly rounded to float32; inf, exponents accepted), may
 * be double-quoted, and an empty field, NA, N/A, NaN, nan or null is a missing cell = NaN (a numeric
 * marker such as 999 is handled by ebic_create_sentinel).  "\n" and "\r\n" line ends; blank lines skipped.
 *   *matrix  receives a malloc'ed ROW-MAJOR float32 [*rows][*cols] ready for ebic_create; the caller
 *            releases it with ebic_free_host.
 * Errors: EBIC_ERR_ARG (NULL, unknown delimiter), EBIC_ERR_IO (cannot open, fewer than two lines, no
 * delimiter found, header/data field counts disagree, ragged line, a field that is not a number),
 * EBIC_ERR_OOM.  On error *matrix == NULL.  No CUDA call is made.
 */
int ebic_read_delimited(const char *path, char delimiter, float **matrix, int64_t *rows, int32_t *cols);

/* Releases a buffer returned by ebic_read_delimited.  NULL is allowed. */
void ebic_free_host(void *p);

/*
 * Measurement utility (not a step of the path): read bandwidth, in GB/s, that all SMs together get
 * from a freshly allocated device buffer of `buffer_bytes` (>= 1 MiB) streamed `reps` times with
 * coalesced 128-bit loads that bypass L1 (best of 3 passes after a warm-up pass, CUDA events on the
 * legacy stream).  A buffer that fits the L2 (e.g. 64 MiB) gives the L2 -> SM bandwidth -- the
 * roofline bench.py uses for the PAIRBITS kernel on matrices too wide for L1 residency --, one far
 * larger than the L2 gives HBM read bandwidth.  Synchronous; allocates and frees its own memory.
 * Errors: EBIC_ERR_ARG, EBIC_ERR_OOM, EBIC_ERR_CUDA (*gb_per_s = 0).
 */
int ebic_probe_read_bandwidth(int64_t buffer_bytes, int32_t reps, double *gb_per_s);

/* Static string for a status code. */
const char *ebic_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* EBIC_H_ */
