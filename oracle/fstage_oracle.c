/*
 * oracle/fstage_oracle.c -- CPU oracle for the F-stage (unpack + Fourier transform) of the FX correlator.
 *
 * TEST INFRASTRUCTURE (same rules as xcorr_oracle.c): only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file; it shares nothing with the CUDA path.
 *
 * What it computes ("1- unpacking a block of data, which involves reordering samples ...
 * 2- Fourier transforming into frequency space"; "taking a block of N_I x N_C complex samples
 * which are ordered with input varying most quickly, converting to floating-point format and putting the
 * samples into N_I arrays of length N_C"; "the FFT is N_C channels in input and output"):
 *
 *   X[b][k][i] = sum_{n=0}^{N_C-1} x[b][n][i] * exp(-2 pi i k n / N_C),     k = 0 .. N_C-1
 *
 * for every block b of N_C consecutive samples and every input i: the plain discrete Fourier transform,
 * written out as the O(N_C^2) double sum in float64 -- no FFT factorisation, so that it can be checked
 * against the definition by eye.  The output is laid out [b][k][i], which IS the X-engine's
 * [time][chan][input] (one spectrum per time step, "the samples (in frequency space) for all
 * inputs in a channel for a single time instant").
 *
 * Readings where the paper is silent (R19-R21):
 *   R19 sign and scale: forward transform with exp(-2 pi i k n / N), unnormalised -- the convention of the
 *       FFT library the paper calls ("the built-in FFT library in CUDA", forward direction).
 *   R20 channel order: natural DFT order, k = 0 (DC) first; no fftshift.
 *   R21 raw samples: complex int8 pairs (re, im), two's complement (PAPER.md:69 stores the 5+5-bit samples
 *       in 16-bit words without giving the bit positions; any 5-bit value is an int8 value), converted
 *       exactly to floating point.
 * The twiddle argument is reduced exactly in integers, (k n) mod N, before the cosine / sine are taken, so
 * that the only rounding is that of cos, sin, the products and the running sum (all float64).
 *
 * Input  x : [B][N][I] interleaved int8 (re, im), input index fastest.
 * Output X : [B][N][I] interleaved float64 (re, im).
 * Pins: tests/test_oracle_fstage_pins.py (F1..F7, tests/golden/f6_dft_worked_example.txt).
 */
#include <math.h>
#include <stdint.h>

int oracle_fstage_ci8(const int8_t *x, long n_batch, long n_fft, long n_inputs, double *out, int threads)
{
    const double two_pi = 6.283185307179586476925286766559;
    (void)threads;
#pragma omp parallel for num_threads(threads) schedule(static) if (threads > 1)
    for (long b = 0; b < n_batch; ++b) {
        const int8_t *xb = x + 2 * b * n_fft * n_inputs;
        double *ob = out + 2 * b * n_fft * n_inputs;
        for (long i = 0; i < n_inputs; ++i) {
            for (long k = 0; k < n_fft; ++k) {
                double re = 0.0, im = 0.0;
                for (long n = 0; n < n_fft; ++n) {
                    const double a = (double)xb[2 * (n * n_inputs + i)];     /* Re x[n] */
                    const double c = (double)xb[2 * (n * n_inputs + i) + 1]; /* Im x[n] */
                    const double phi = two_pi * (double)((k * n) % n_fft) / (double)n_fft;
                    const double wr = cos(phi), wi = -sin(phi);              /* exp(-i phi) */
                    re += a * wr - c * wi;
                    im += a * wi + c * wr;
                }
                ob[2 * (k * n_inputs + i)] = re;
                ob[2 * (k * n_inputs + i) + 1] = im;
            }
        }
    }
    return 0;
}

/*
 * The same transform for the paper's "1-byte mode" ("the data samples were reduced from 2-byte words
 * to a single byte, at the cost of 1 bit of precision in the real and imaginary parts ... reduces the total amount of
 * global memory reads in the unpack phase"): x is [B][N][I] BYTES, low nibble = Re, high nibble = Im, 4-bit two's
 * complement (DESIGN reading R18, the same byte as the X-engine's CORR_CI4 input).  The nibble decode is written out
 * here again (v >= 8 ? v - 16 : v) so that this file stands alone; pin F8 checks it against the int8 routine above on
 * data unpacked by numpy, and P11's hand-written byte table pins the byte layout.
 */
int oracle_fstage_ci4(const uint8_t *x, long n_batch, long n_fft, long n_inputs, double *out, int threads)
{
    const double two_pi = 6.283185307179586476925286766559;
    (void)threads;
#pragma omp parallel for num_threads(threads) schedule(static) if (threads > 1)
    for (long b = 0; b < n_batch; ++b) {
        const uint8_t *xb = x + b * n_fft * n_inputs;
        double *ob = out + 2 * b * n_fft * n_inputs;
        for (long i = 0; i < n_inputs; ++i) {
            for (long k = 0; k < n_fft; ++k) {
                double re = 0.0, im = 0.0;
                for (long n = 0; n < n_fft; ++n) {
                    const unsigned byte = xb[n * n_inputs + i];
                    const unsigned lo = byte & 15u, hi = byte >> 4;
                    const double a = (double)(lo >= 8 ? (int)lo - 16 : (int)lo); /* Re x[n] */
                    const double c = (double)(hi >= 8 ? (int)hi - 16 : (int)hi); /* Im x[n] */
                    const double phi = two_pi * (double)((k * n) % n_fft) / (double)n_fft;
                    const double wr = cos(phi), wi = -sin(phi);                  /* exp(-i phi) */
                    re += a * wr - c * wi;
                    im += a * wi + c * wr;
                }
                ob[2 * (k * n_inputs + i)] = re;
                ob[2 * (k * n_inputs + i) + 1] = im;
            }
        }
    }
    return 0;
}

/*
 * The X-engine definition on float64 spectra (same formula and loop order as oracle_xengine_cf32 in
 * xcorr_oracle.c), so that the F -> X chain can be followed in float64 end to end.
 * x : [T][C][N] float64 pairs; vis : [C][N(N+1)/2] float64 pairs.
 */
int oracle_xengine_cf64(const double *x, long n_time, long n_chan, long n_inputs, double *vis, int threads)
{
    const long nb = n_inputs * (n_inputs + 1) / 2;
    (void)threads;
#pragma omp parallel for num_threads(threads) schedule(static) if (threads > 1)
    for (long c = 0; c < n_chan; ++c) {
        double *out = vis + 2 * nb * c;
        for (long k = 0; k < 2 * nb; ++k) out[k] = 0.0;
        for (long t = 0; t < n_time; ++t) {
            const double *xt = x + 2 * (t * n_chan + c) * n_inputs;
            long b = 0;
            for (long i = 0; i < n_inputs; ++i) {
                const double ai = xt[2 * i], bi = xt[2 * i + 1];
                for (long j = 0; j <= i; ++j, ++b) {
                    const double aj = xt[2 * j], bj = xt[2 * j + 1];
                    out[2 * b] += ai * aj + bi * bj;     /* Re x_i conj(x_j) */
                    out[2 * b + 1] += bi * aj - ai * bj; /* Im x_i conj(x_j) */
                }
            }
        }
    }
    return 0;
}
