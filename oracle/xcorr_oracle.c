/*
 * oracle/xcorr_oracle.c -- CPU oracle for the X-engine (CMAC) of an FX correlator.
 *
 * TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  The
 * product (paper_0906_1887_b200/) never does, and this file shares no code,
 * header, table or helper with the CUDA path.
 *
 * What it computes is the definition itself, written out:
 *
 *   "an FX correlator ... does a channel-by-channel multiplication ('X') of the
 *    first spectrum with the complex conjugate of the second to form the
 *    correlation product ... The results of the cross-multiplications are
 *    accumulated for each baseline."                       (sec. 2)
 *   "The correlation products for a given frequency channel can be represented
 *    in a matrix of size N_I x N_I formed by the outer product of a vector with
 *    its complex conjugate"                          (Fig. 2 :115)
 *   N_I(N_I+1)/2 products including auto-correlations      (sec. 2)
 *   accumulators are summed over the integration and read out (Fig. 1)
 *
 *   V[c][b(i,j)] = sum_{t=0}^{T-1} x[t][c][i] * conj(x[t][c][j]),   i >= j
 *
 * with x = a + ib:   Re V = sum_t (a_i a_j + b_i b_j)
 *                    Im V = sum_t (b_i a_j - a_i b_j)
 *
 * Readings where the paper is silent:
 *   R1  the LOWER-index input j is the conjugated one (north_star).
 *   R2  packed order is the row-major lower triangle: (0,0),(1,0),(1,1),(2,0)...
 *       -- here simply the order in which the i, j<=i loops visit the pairs.
 *   R3  raw sums; no division by the update count (PAPER.md:84 divides at read-out).
 *   R6  int8 path: exact integers; accumulate in int64 and REFUSE (return -2)
 *       if any sum does not fit int32.
 *   R7  float path: inputs are float32, every product and sum is float64.
 *
 * Input  x   : [T][C][N] interleaved (re, im), input index fastest.
 * Output vis : [c_end - c_begin][N(N+1)/2] interleaved (re, im).
 *
 * Loops are the plain five (c, t, i, j<=i) in that order, no blocking, no SIMD
 * intrinsics.  `threads` > 1 only spreads whole channels over OpenMP threads
 * (channels are independent); the per-channel arithmetic and its
 * order are identical to threads == 1.
 *
 * Compile: gcc -O2 -std=c99 -ffp-contract=off -fopenmp (see oracle/__init__.py).
 * Pins: tests/test_oracle_pins.py (P1..P9 + tests/golden/).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_EALLOC (-1)
#define ORACLE_EOVERFLOW (-2)

/* Packed lower triangle, complex int8 -> complex int32 (int64-checked). */
int oracle_xengine_ci8(const int8_t *x, long n_time, long n_chan, long n_inputs,
                       long c_begin, long c_end, int32_t *vis, int threads)
{
    const long nb = n_inputs * (n_inputs + 1) / 2;
    int status = ORACLE_OK;
    (void)threads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 1 ? threads : 1)
    for (long c = c_begin; c < c_end; ++c) {
        int64_t *acc = (int64_t *)calloc((size_t)(2 * nb), sizeof(int64_t));
        if (!acc) {
#pragma omp critical
            status = ORACLE_EALLOC;
            continue;
        }
        for (long t = 0; t < n_time; ++t) {
            const int8_t *xt = x + 2 * ((t * n_chan + c) * n_inputs);
            long b = 0;
            for (long i = 0; i < n_inputs; ++i) {
                const int64_t a_i = xt[2 * i], b_i = xt[2 * i + 1];
                for (long j = 0; j <= i; ++j, ++b) {
                    const int64_t a_j = xt[2 * j], b_j = xt[2 * j + 1];
                    acc[2 * b] += a_i * a_j + b_i * b_j;     /* Re x_i conj(x_j) */
                    acc[2 * b + 1] += b_i * a_j - a_i * b_j; /* Im x_i conj(x_j) */
                }
            }
        }
        int32_t *out = vis + 2 * nb * (c - c_begin);
        for (long k = 0; k < 2 * nb; ++k) {
            if (acc[k] > INT32_MAX || acc[k] < INT32_MIN) {
#pragma omp critical
                status = ORACLE_EOVERFLOW;
            }
            out[k] = (int32_t)acc[k];
        }
        free(acc);
    }
    return status;
}

/* Packed lower triangle, complex float32 -> complex float64. */
int oracle_xengine_cf32(const float *x, long n_time, long n_chan, long n_inputs,
                        long c_begin, long c_end, double *vis, int threads)
{
    const long nb = n_inputs * (n_inputs + 1) / 2;
    (void)threads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 1 ? threads : 1)
    for (long c = c_begin; c < c_end; ++c) {
        double *acc = vis + 2 * nb * (c - c_begin);
        memset(acc, 0, (size_t)(2 * nb) * sizeof(double));
        for (long t = 0; t < n_time; ++t) {
            const float *xt = x + 2 * ((t * n_chan + c) * n_inputs);
            long b = 0;
            for (long i = 0; i < n_inputs; ++i) {
                const double a_i = xt[2 * i], b_i = xt[2 * i + 1];
                for (long j = 0; j <= i; ++j, ++b) {
                    const double a_j = xt[2 * j], b_j = xt[2 * j + 1];
                    acc[2 * b] += a_i * a_j + b_i * b_j;
                    acc[2 * b + 1] += b_i * a_j - a_i * b_j;
                }
            }
        }
    }
    return ORACLE_OK;
}

/*
 * The "even dumber" routine: the FULL N x N matrix of one channel, every (i, j),
 * straight from Fig. 2: M[i][j] = sum_t x_i conj(x_j).  Used only
 * to pin the packed routine (Hermitian symmetry, real non-negative diagonal,
 * N(N+1)/2 distinct products).  Written with explicit complex multiplication
 * (re, im of the product spelled out per term) rather than the expanded sums
 * above, so that a sign slip in one routine does not repeat in the other.
 */
int oracle_full_matrix_ci8(const int8_t *x, long n_time, long n_chan, long n_inputs,
                           long c, int64_t *full /* [N][N][2] */)
{
    memset(full, 0, (size_t)(2 * n_inputs * n_inputs) * sizeof(int64_t));
    for (long t = 0; t < n_time; ++t) {
        const int8_t *xt = x + 2 * ((t * n_chan + c) * n_inputs);
        for (long i = 0; i < n_inputs; ++i) {
            for (long j = 0; j < n_inputs; ++j) {
                /* (p + iq) * (r + is) with (r + is) = conj(x_j) = a_j - i b_j */
                const int64_t p = xt[2 * i], q = xt[2 * i + 1];
                const int64_t r = xt[2 * j], s = -(int64_t)xt[2 * j + 1];
                full[2 * (i * n_inputs + j)] += p * r - q * s;
                full[2 * (i * n_inputs + j) + 1] += p * s + q * r;
            }
        }
    }
    return ORACLE_OK;
}

int oracle_full_matrix_cf32(const float *x, long n_time, long n_chan, long n_inputs,
                            long c, double *full /* [N][N][2] */)
{
    memset(full, 0, (size_t)(2 * n_inputs * n_inputs) * sizeof(double));
    for (long t = 0; t < n_time; ++t) {
        const float *xt = x + 2 * ((t * n_chan + c) * n_inputs);
        for (long i = 0; i < n_inputs; ++i) {
            for (long j = 0; j < n_inputs; ++j) {
                const double p = xt[2 * i], q = xt[2 * i + 1];
                const double r = xt[2 * j], s = -(double)xt[2 * j + 1];
                full[2 * (i * n_inputs + j)] += p * r - q * s;
                full[2 * (i * n_inputs + j) + 1] += p * s + q * r;
            }
        }
    }
    return ORACLE_OK;
}

/*
 * One visibility on its own: V[c][(i, j)] for a single pair -- what the
 * full-size parity tests sample when the whole cube is too slow to recompute.
 * Same two lines of arithmetic as the packed routine.
 */
int oracle_one_visibility_ci8(const int8_t *x, long n_time, long n_chan, long n_inputs,
                              long c, long i, long j, int64_t *re_im /* [2] */)
{
    int64_t re = 0, im = 0;
    for (long t = 0; t < n_time; ++t) {
        const int8_t *xt = x + 2 * ((t * n_chan + c) * n_inputs);
        const int64_t a_i = xt[2 * i], b_i = xt[2 * i + 1];
        const int64_t a_j = xt[2 * j], b_j = xt[2 * j + 1];
        re += a_i * a_j + b_i * b_j;
        im += b_i * a_j - a_i * b_j;
    }
    re_im[0] = re;
    re_im[1] = im;
    return ORACLE_OK;
}

int oracle_one_visibility_cf32(const float *x, long n_time, long n_chan, long n_inputs,
                               long c, long i, long j, double *re_im /* [2] */)
{
    double re = 0.0, im = 0.0;
    for (long t = 0; t < n_time; ++t) {
        const float *xt = x + 2 * ((t * n_chan + c) * n_inputs);
        const double a_i = xt[2 * i], b_i = xt[2 * i + 1];
        const double a_j = xt[2 * j], b_j = xt[2 * j + 1];
        re += a_i * a_j + b_i * b_j;
        im += b_i * a_j - a_i * b_j;
    }
    re_im[0] = re;
    re_im[1] = im;
    return ORACLE_OK;
}

/*
 * 4-bit packed input: the paper's "1-byte mode" ("4+4 bits ... halves the volume";
 * samples are two's complement).  Reading R18: one byte per complex sample,
 * LOW nibble = Re, HIGH nibble = Im, each a two's-complement 4-bit integer in [-8, 7].
 * The visibilities are the same definition as above applied to the unpacked values.
 */
static int nibble_to_int(unsigned v /* 0..15 */) { return v >= 8 ? (int)v - 16 : (int)v; }

void oracle_unpack_ci4(uint8_t byte, int *re, int *im)
{
    *re = nibble_to_int(byte & 15u);
    *im = nibble_to_int((unsigned)byte >> 4);
}

int oracle_xengine_ci4(const uint8_t *x, long n_time, long n_chan, long n_inputs,
                       long c_begin, long c_end, int32_t *vis, int threads)
{
    const long nb = n_inputs * (n_inputs + 1) / 2;
    int status = ORACLE_OK;
    (void)threads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 1 ? threads : 1)
    for (long c = c_begin; c < c_end; ++c) {
        int64_t *acc = (int64_t *)calloc((size_t)(2 * nb), sizeof(int64_t));
        if (!acc) {
#pragma omp critical
            status = ORACLE_EALLOC;
            continue;
        }
        for (long t = 0; t < n_time; ++t) {
            const uint8_t *xt = x + (t * n_chan + c) * n_inputs;
            long b = 0;
            for (long i = 0; i < n_inputs; ++i) {
                int ai, bi;
                oracle_unpack_ci4(xt[i], &ai, &bi);
                for (long j = 0; j <= i; ++j, ++b) {
                    int aj, bj;
                    oracle_unpack_ci4(xt[j], &aj, &bj);
                    acc[2 * b] += (int64_t)ai * aj + (int64_t)bi * bj;     /* Re x_i conj(x_j) */
                    acc[2 * b + 1] += (int64_t)bi * aj - (int64_t)ai * bj; /* Im x_i conj(x_j) */
                }
            }
        }
        int32_t *out = vis + 2 * nb * (c - c_begin);
        for (long k = 0; k < 2 * nb; ++k) out[k] = (int32_t)acc[k]; /* |V| <= T*2*64 always fits */
        free(acc);
    }
    return status;
}

/*
 * Read-out (Fig. 1 caption): "the accumulators are ... divided by the number of times they
 * were updated" -> the time-averaged visibility.  Plain division in float64.
 */
void oracle_readout_i32(const int32_t *vis, long n_scalars, double count, double *out)
{
    for (long k = 0; k < n_scalars; ++k) out[k] = (double)vis[k] / count;
}
void oracle_readout_f64(const double *vis, long n_scalars, double count, double *out)
{
    for (long k = 0; k < n_scalars; ++k) out[k] = vis[k] / count;
}

/*
 * Long accumulations (the accumulators are read "after a specified time, usually a few
 * seconds"; every batch of spectra is ADDED to the persistent accumulators).  The
 * definition is the same sum over ALL samples of all batches; only the output word is wider: int64, so
 * that no int8 input can overflow for any realistic T (|V| <= T * 2 * 128^2 < 2^63 for T < 2.8e14).
 * Same five loops as oracle_xengine_ci8, without the int32 check.
 */
int oracle_xengine_ci8_wide(const int8_t *x, long n_time, long n_chan, long n_inputs,
                            long c_begin, long c_end, int64_t *vis, int threads)
{
    const long nb = n_inputs * (n_inputs + 1) / 2;
    (void)threads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads > 1 ? threads : 1)
    for (long c = c_begin; c < c_end; ++c) {
        int64_t *acc = vis + 2 * nb * (c - c_begin);
        memset(acc, 0, (size_t)(2 * nb) * sizeof(int64_t));
        for (long t = 0; t < n_time; ++t) {
            const int8_t *xt = x + 2 * ((t * n_chan + c) * n_inputs);
            long b = 0;
            for (long i = 0; i < n_inputs; ++i) {
                const int64_t a_i = xt[2 * i], b_i = xt[2 * i + 1];
                for (long j = 0; j <= i; ++j, ++b) {
                    const int64_t a_j = xt[2 * j], b_j = xt[2 * j + 1];
                    acc[2 * b] += a_i * a_j + b_i * b_j;     /* Re x_i conj(x_j) */
                    acc[2 * b + 1] += b_i * a_j - a_i * b_j; /* Im x_i conj(x_j) */
                }
            }
        }
    }
    return ORACLE_OK;
}

void oracle_readout_i64(const int64_t *vis, long n_scalars, double count, double *out)
{
    for (long k = 0; k < n_scalars; ++k) out[k] = (double)vis[k] / count;
}
