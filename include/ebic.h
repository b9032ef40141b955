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
 *   DESIGN.md section 3 (readings R1-R17), identical to the CPU oracle's header:
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
 *     bytes viewed as uint8 have row r at byte r/8, bit r%8).  Bits >= rows are zero (R16).
 *   - The library reads no environment variable.  Knobs, read-backs of loader products and measurement probes
 *     used by the tests and by bench.py live in include/ebic_debug.h, not here.
 *
 * Which passage defines which call: ebic_create / ebic_create_sentinel / ebic_read_delimited -- PAPER.md lines
 * 59-61 (the input matrix, its limits, its missing-value marker, its file format); ebic_eval_fitness -- PAPER.md
 * line 60 (row counting under >=) with the population limits of line 59; ebic_extract_rows -- PAPER.md line 62
 * (a bicluster is returned as rows + columns); ebic_eval_extract -- both, one GA generation; ebic_eval_fitness_noalloc -- line 60 again; ebic_mask_words /
 * ebic_status / ebic_strerror / ebic_destroy / ebic_free_host -- bookkeeping the paper does not describe
 * (BASELINE.json north_star (1)).
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
    EBIC_ERR_IO = 6,          /* ebic_read_delimited: cannot open / not a delimited matrix / ragged line */
    EBIC_ERR_LIMIT = 7        /* ebic_eval_fitness_noalloc: population larger than the fixed scratch holds */
};
enum { EBIC_MISSING_OFF = 0, EBIC_MISSING_ON = 1 };

/*
 * Loader (a genes x samples matrix with optional missing values).
 *   matrix        dense ROW-MAJOR float32 [rows][cols]; host or device pointer; any NaN = missing.
 *   rows          1 .. 2^31-1.        cols  1 .. 2^31-1 (memory permitting).
 *   missing_mode  EBIC_MISSING_OFF / EBIC_MISSING_ON.
 *   out           receives the context.
 * Transposes to column-major, builds the packed NaN bitmask and per-column non-missing counts and, when it
 * takes at most 32 GiB and half of the free device memory, the pair-relation table (cols^2 bits per padded row:
 * bit r of pair (a,b) = M[r][b] >= M[r][a]); without the table and with cols <= 127, the
 * 8-bit rank tiles instead.
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
 *   n_ind    0 .. 2^31-2 (0 is a no-op).
 *   n_ids    number of entries of col_ids.  Not in north_star's signature: it is the bound that lets the
 *            device validate offsets without trusting them (R8: offsets[k+1] > n_ids is an error,
 *            not an out-of-bounds read), and the size of the host-to-device copy when col_ids is a host pointer.
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
 *   n_ind, n_ids  as in ebic_eval_fitness: `chosen` indexes the same CSR, and the kernel validates the chosen
 *            individuals itself (it does not depend on an earlier ebic_eval_fitness call).
 *   chosen   int32 [n_chosen] indices into the CSR population, host or device (same kind as offsets);
 *            an index outside [0, n_ind) yields an all-zero mask and the sticky EBIC_ERR_BAD_OFFSETS.
 *   masks    uint64 [n_chosen][ebic_mask_words(ctx)], host or device, overwritten.
 *   counts   uint64 [n_chosen] or NULL.
 * Same asynchrony, validation and error rules as ebic_eval_fitness.
 */
int ebic_extract_rows(ebic_ctx *ctx, const int32_t *offsets, const int32_t *col_ids, int32_t n_ind,
                      int64_t n_ids, const int32_t *chosen, int32_t n_chosen, uint64_t *masks,
                      uint64_t *counts, void *cuda_stream);

/*
 * One GA generation in one call: ebic_eval_fitness followed by ebic_extract_rows on the same population, with
 * the population uploaded once (host pointers) and one stream synchronisation; with device outputs the extraction
 * kernel is chained behind the fitness kernel with programmatic dependent launch and runs alongside its last
 * wave; with host outputs the masks -- which do not depend on the counts -- are extracted first and copied back on
 * a stream the context owns while the fitness kernel runs (everything has completed when the call returns, also when
 * it returns an error: no copy into `masks` is left in flight).  That overlap needs PINNED host outputs
 * (cudaHostAlloc / cudaHostRegister): into pageable memory the runtime copies through its own staging buffer and keeps
 * the calling thread until the copy is done, so the fitness kernel is launched after it -- same results, no overlap.
 * Repetition: a GA loop passes the same device buffers every generation.  When a call with device pointers on a
 * non-default stream repeats the previous call's arguments exactly (pointers, sizes, stream), the library captures
 * its launch sequence into a CUDA graph and replays that graph from then on -- the results are those of the plain
 * launches; only the launch overhead changes (ebic_eval_fitness and ebic_extract_rows do the same).  Buffers passed
 * to such a call must therefore stay valid until the work has run, as with any stream-ordered call.  Arguments as in the two calls (`mask_counts` may be NULL).  n_ind == 0 or n_chosen == 0 skips that
 * half.  `counts`, `masks` and `mask_counts` must not overlap each other (the two kernels may run concurrently).
 */
int ebic_eval_extract(ebic_ctx *ctx, const int32_t *offsets, const int32_t *col_ids, int32_t n_ind,
                      int64_t n_ids, uint64_t *counts, const int32_t *chosen, int32_t n_chosen,
                      uint64_t *masks, uint64_t *mask_counts, void *cuda_stream);

/*
 * ebic_eval_fitness for callers that must not allocate device memory once their set-up is over.
 *
 * Who that is.  ebic_eval_fitness keeps per-call scratch (one validated record per individual) in buffers it
 * grows with cudaFree + cudaMalloc whenever a population is larger than any it has seen.  Some hosts cannot live
 * with that in their generation loop: a service whose own pool has taken the rest of the HBM after start-up (the
 * cudaMalloc then fails in the middle of a run, hours in), a loop that shares the GPU with latency-bound streams
 * (cudaFree waits for the whole device, cudaMalloc may too), and embedders whose rules simply forbid driver
 * allocations after initialisation.  For them this call computes the same count[k] (same
 * definition, same validation, same sticky errors as ebic_eval_fitness) and makes no cudaMalloc, cudaFree or
 * other allocating call: its scratch is a fixed array compiled into libebic.so.
 *
 * The price of that array.
 *   - It is EBIC_NOALLOC_MAX_IND * 136 bytes = 2,176 KiB, and every GPU on which the process loads the library
 *     holds it until the process exits, used or not.
 *   - n_ind > EBIC_NOALLOC_MAX_IND is refused with EBIC_ERR_LIMIT before anything is launched (`counts`
 *     untouched); use ebic_eval_fitness for such populations.
 *   - There is ONE array per GPU, shared by every context and every call on that GPU.  It still holds the
 *     previous call's records on entry; the call needs none of them zeroed, because its first kernel rewrites
 *     every record of 0 .. n_ind-1 before its second kernel reads exactly those.  Two calls that may run at the
 *     same time on one GPU (different streams, different contexts, different host threads) race on it and return
 *     garbage: issue them on one stream, or order the streams yourself.  Calls on one stream are safe back to
 *     back.  ebic_eval_fitness and the other calls do not touch the array.
 *   - The first call on each GPU looks up the array's device address (cudaGetSymbolAddress, once, under a lock)
 *     before it launches.  Make that first call during set-up, outside any stream capture.
 *
 * Arguments as in ebic_eval_fitness, except that offsets, col_ids and counts must ALL be device pointers (a host
 * buffer would need a staging allocation: EBIC_ERR_ARG).  Always asynchronous and stream-ordered on `cuda_stream`.
 * The context is the one ebic_create made during set-up (ebic_create does allocate); it runs PAIRBITS when the
 * context holds the pair table and DIRECT otherwise, whatever ebic_set_kernel says, with the context's early-exit
 * setting; the context's own scratch and its captured launch graph are neither used nor disturbed.
 */
#define EBIC_NOALLOC_MAX_IND 16384
int ebic_eval_fitness_noalloc(ebic_ctx *ctx, const int32_t *offsets, const int32_t *col_ids, int32_t n_ind,
                              int64_t n_ids, uint64_t *counts, void *cuda_stream);

/* ceil(rows / 64): uint64 words per mask.  -1 if ctx is NULL. */
int64_t ebic_mask_words(const ebic_ctx *ctx);

/*
 * Synchronises `cuda_stream`, returns the sticky device error raised since the last ebic_status()
 * (EBIC_OK if none) and clears it.  EBIC_ERR_CUDA if the stream itself reports an error.
 */
int ebic_status(ebic_ctx *ctx, void *cuda_stream);

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

/* Static string for a status code. */
const char *ebic_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* EBIC_H_ */
