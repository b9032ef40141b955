/*
 * oracle/ebic_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, link, import or call this file.  It shares no code, header, table or helper with the
 * CUDA path under paper_1807_09932_b200/csrc/ and neither includes the other.
 *
 * What it computes (plain definition; tolerance 0 -- exactly one result is correct):
 *
 *   Matrix M, float32, rows x cols, ROW-MAJOR exactly as the user supplied it (never the GPU
 *   loader's transposed copy).  Individual k is the ordered list
 *       c_0 .. c_{L-1} = col_ids[offsets[k] .. offsets[k+1])                (BASELINE.json north_star)
 *   and for row r
 *
 *       ok(k,r) =  AND_{i=0..L-2} ( M[r][c_{i+1}] >= M[r][c_i] )            IEEE-754 ordered >=, float32
 *                  AND ( missing_mode == ON  =>  no M[r][c_i] is NaN, i = 0..L-1 )
 *       count[k] = #{ r : ok(k,r) }          mask[k] bit r = ok(k,r)
 *
 *   Passages followed: PAPER.md line 60 (section 2 Methods, bullet "Handling missing values"):
 *   "EBIC search is driven by counting of rows, a greater or equal relation between the values in
 *   columns", and missing values are "no longer counted towards the score of the bicluster".
 *   PAPER.md line 59 (bullet "Support for Big Data"): up to 2^31-1 rows (the minus sign is lost in
 *   the extracted text), population up to 65,535.  Everything else below is a READING, because the
 *   paper writes down no formula; the readings are SURVEY.md section 8(c) and DESIGN.md section 3:
 *
 *   R1  trend direction: non-decreasing in chromosome order, ties match.
 *   R2  missing-value rule ("Rule A"): in mode ON a row counts for an individual iff every one of
 *       the individual's columns is non-missing in that row and every consecutive pair holds.
 *   R3  missing marker at this interface = any float32 NaN (any sign, payload, quiet/signalling).
 *   R4  mode OFF with NaN present: plain IEEE, a pair touching NaN is false; so ON and OFF differ
 *       only for L = 1 (OFF counts every row).
 *   R5  L = 1: ON -> rows whose value in that column is not NaN; OFF -> all rows.
 *   R6  L = 0: vacuous truth, count = rows, mask all ones (tail bits zero), both modes.
 *   R7  duplicate columns are legal and get no special case.
 *   R8  column id outside [0, cols) -> that individual is invalid: count 0 / mask all zero, and the
 *       call returns ORACLE_ERR_BAD_COLUMN.  offsets[k] < 0, offsets[k+1] < offsets[k] or
 *       offsets[k+1] > n_ids (the length of col_ids) -> that individual is invalid the same way
 *       and the call returns ORACLE_ERR_BAD_OFFSETS.  If both kinds occur the larger code
 *       (BAD_OFFSETS) is returned.  Valid individuals are unaffected.
 *   R9  -0.0 >= +0.0 and +0.0 >= -0.0 are true; infinities are ordinary values; denormals compare
 *       by value (no flush-to-zero: compile WITHOUT -ffast-math / -Ofast).
 *   R10 counts are uint64; all row arithmetic is int64.
 *   R16 bitmask: row r <-> word r/64, bit r%64 of a little-endian uint64 (LSB first), ceil(rows/64)
 *       words per individual, bits >= rows are zero.
 *
 * Loop nest exactly as north_star words it: individuals (outer) x rows x consecutive column pairs.
 * No early exit, no blocking, no vectorisation tricks.  NaN is tested on the bit pattern so no
 * compiler flag can delete the test.  The only concession to run time is an OpenMP "parallel for"
 * over the OUTER (individual) loop, which does not change the nest or any arithmetic.
 *
 * Pins (tests/test_oracle_*.py, all run with -m "not gpu"): hand-enumerated fixtures under
 * tests/golden/, exact planted recovery, invariants, ON/OFF identity, reversal identity,
 * permutation partition, Binomial closed form, special matrices, an independent numpy restatement
 * and a pure-Python brute force.  No function here is "parity unpinned".
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum {
    ORACLE_OK = 0,
    ORACLE_ERR_ARG = 1,
    ORACLE_ERR_BAD_COLUMN = 4,
    ORACLE_ERR_BAD_OFFSETS = 5
};
enum { ORACLE_MISSING_OFF = 0, ORACLE_MISSING_ON = 1 };

/* R3: NaN on the bit pattern: exponent all ones and a non-zero mantissa. */
static int oracle_is_missing(float v)
{
    uint32_t bits;
    memcpy(&bits, &v, sizeof bits);
    return (bits & 0x7fffffffu) > 0x7f800000u;
}

/* ok(k,r) of the header, written out term by term.  `row` points at M[r][0]. */
static int oracle_row_ok(const float *row, const int32_t *ids, int32_t L, int32_t missing_mode)
{
    int ok = 1;
    int32_t i;
    for (i = 0; i + 1 < L; ++i) {
        float lo = row[ids[i]];
        float hi = row[ids[i + 1]];
        if (!(hi >= lo)) /* ordered >=: false when either side is NaN (R4) */
            ok = 0;
    }
    if (missing_mode == ORACLE_MISSING_ON) {
        for (i = 0; i < L; ++i)
            if (oracle_is_missing(row[ids[i]])) /* R2 */
                ok = 0;
    }
    return ok;
}

/* R8.  Returns 0 if individual k is well formed, else the error code it raises. */
static int oracle_check_individual(const int32_t *offsets, const int32_t *col_ids, int64_t n_ids,
                                   int32_t cols, int32_t k)
{
    int32_t b = offsets[k], e = offsets[k + 1], i;
    if (b < 0 || e < b || (int64_t)e > n_ids)
        return ORACLE_ERR_BAD_OFFSETS;
    for (i = b; i < e; ++i)
        if (col_ids[i] < 0 || col_ids[i] >= cols)
            return ORACLE_ERR_BAD_COLUMN;
    return ORACLE_OK;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * count[k] for every individual of the population.
 * M: host, row-major [rows][cols].  offsets: [n_ind+1].  col_ids: [n_ids].
 * counts: [n_ind], overwritten.  n_threads <= 0 -> all cores OpenMP reports.
 */
int oracle_eval_fitness(const float *M, int64_t rows, int32_t cols, int32_t missing_mode,
                        const int32_t *offsets, const int32_t *col_ids, int32_t n_ind,
                        int64_t n_ids, uint64_t *counts, int32_t n_threads)
{
    int status = ORACLE_OK;
    int32_t k;
    if (!M || rows <= 0 || cols <= 0 || n_ind < 0 || n_ids < 0 ||
        (missing_mode != ORACLE_MISSING_OFF && missing_mode != ORACLE_MISSING_ON))
        return ORACLE_ERR_ARG;
    if (n_ind == 0)
        return ORACLE_OK;
    if (!offsets || !counts)
        return ORACLE_ERR_ARG;
#ifdef _OPENMP
    if (n_threads <= 0)
        n_threads = omp_get_max_threads();
#else
    (void)n_threads;
#endif

#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
    for (k = 0; k < n_ind; ++k) {                         /* individuals (outer) */
        int err = oracle_check_individual(offsets, col_ids, n_ids, cols, k);
        uint64_t c = 0;
        if (err == ORACLE_OK) {
            const int32_t *ids = col_ids + offsets[k];
            int32_t L = offsets[k + 1] - offsets[k];
            int64_t r;
            for (r = 0; r < rows; ++r)                    /* rows */
                c += (uint64_t)oracle_row_ok(M + r * (int64_t)cols, ids, L, missing_mode);
        } else {
#pragma omp critical
            if (err > status)
                status = err;
        }
        counts[k] = c;
    }
    return status;
}

/*
 * mask[j] (and optionally count[j]) for the chosen individuals chosen[0..n_chosen).
 * masks: [n_chosen][ceil(rows/64)] uint64, overwritten (R16).  counts may be NULL.
 * A chosen index outside [0, n_ind) names no individual: its mask is all zero, its count 0 and the
 * call returns ORACLE_ERR_BAD_OFFSETS (same treatment as an individual with bad offsets, R8).
 */
int oracle_extract_rows(const float *M, int64_t rows, int32_t cols, int32_t missing_mode,
                        const int32_t *offsets, const int32_t *col_ids, int32_t n_ind,
                        int64_t n_ids, const int32_t *chosen, int32_t n_chosen, uint64_t *masks,
                        uint64_t *counts)
{
    int status = ORACLE_OK;
    int64_t words;
    int32_t j;
    if (!M || rows <= 0 || cols <= 0 || n_ind < 0 || n_ids < 0 || n_chosen < 0 ||
        (missing_mode != ORACLE_MISSING_OFF && missing_mode != ORACLE_MISSING_ON))
        return ORACLE_ERR_ARG;
    if (n_chosen == 0)
        return ORACLE_OK;
    if (!offsets || !chosen || !masks)
        return ORACLE_ERR_ARG;
    words = (rows + 63) / 64;

    for (j = 0; j < n_chosen; ++j) {
        int32_t k = chosen[j];
        uint64_t *mask = masks + (int64_t)j * words;
        uint64_t c = 0;
        int err = (k < 0 || k >= n_ind) ? ORACLE_ERR_BAD_OFFSETS
                                        : oracle_check_individual(offsets, col_ids, n_ids, cols, k);
        int64_t w, r;
        for (w = 0; w < words; ++w)
            mask[w] = 0;
        if (err == ORACLE_OK) {
            const int32_t *ids = col_ids + offsets[k];
            int32_t L = offsets[k + 1] - offsets[k];
            for (r = 0; r < rows; ++r) {
                if (oracle_row_ok(M + r * (int64_t)cols, ids, L, missing_mode)) {
                    mask[r / 64] |= (uint64_t)1 << (r % 64);
                    ++c;
                }
            }
        } else if (err > status) {
            status = err;
        }
        if (counts)
            counts[j] = c;
    }
    return status;
}
