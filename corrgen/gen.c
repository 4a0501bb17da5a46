/*
 * corrgen/gen.c -- seeded, counter-based synthetic voltage generators.
 *
 * This module only makes INPUTS.  It holds none of the correlator's arithmetic
 * (no products, no accumulation, no triangle indexing) and is the one piece of
 * code that both the CPU oracle's tests and the CUDA path's tests/bench share.
 *
 * The samples stand in for the MWA-32T voltage streams the paper measured on
 * (PAPER.md:65-71 section 3, :164-166 section 5): noise-like, few-bit,
 * complex, ordered [time][chan][input] with the input index fastest -- the
 * order the paper's aggregator emits.
 *
 * Every sample is a pure function of (seed, sample index), so any element can
 * be regenerated on its own and the fill is trivially parallel:
 *
 *   e        = (t*C + c)*N + i                      complex sample index
 *   h1, h2   = mix64(key(seed) ^ 2e), mix64(key(seed) ^ (2e+1))
 *   u1, u2   = ((h >> 11) + 0.5) * 2^-53            uniforms in (0,1)
 *   g_re/im  = sqrt(-2 ln u1) * cos/sin(2 pi u2)    Box-Muller, float64
 *
 * kinds:
 *   GAUSS_I8   re,im = clip(rint(sigma*g + tone), -clip, clip)        int8
 *   UNIFORM_I8 re,im = (h1>>32) % (2*clip+1) - clip , (h2>>32) % ...  int8
 *   GAUSS_F32  re,im = (float)(sigma*g + tone)                        float32
 * tone (common per-channel source, PAPER.md:176, :202 for the analogue):
 *   amp * cos/sin(w_c*t + phi_{c,i}),  w_c = 2 pi ((c mod 16)+1)/64,
 *   phi_{c,i} = 2 pi * uniform(mix64(key(seed ^ TONE_SALT) ^ (c*N+i)))
 *
 * rint() is round-half-to-even (the default FP environment).
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define TWO_PI 6.283185307179586476925286766559
#define TONE_SALT 0x746f6e655f706869ULL /* "tone_phi" */

static inline uint64_t mix64(uint64_t x)
{
    x += 0x9E3779B97F4A7C15ULL;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
    return x ^ (x >> 31);
}

static inline double unit_open(uint64_t h)
{
    return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

static inline void gauss_pair(uint64_t key, uint64_t e, double *g_re, double *g_im)
{
    const uint64_t h1 = mix64(key ^ (2 * e));
    const uint64_t h2 = mix64(key ^ (2 * e + 1));
    const double r = sqrt(-2.0 * log(unit_open(h1)));
    const double a = TWO_PI * unit_open(h2);
    *g_re = r * cos(a);
    *g_im = r * sin(a);
}

static inline double tone_phase(uint64_t seed, long c, long n_inputs, long i)
{
    const uint64_t key = mix64(seed ^ TONE_SALT);
    return TWO_PI * unit_open(mix64(key ^ (uint64_t)(c * n_inputs + i)));
}

static inline double clipd(double v, double lim)
{
    return v > lim ? lim : (v < -lim ? -lim : v);
}

/* Gaussian (+ optional tone) complex int8, time rows [t_begin, t_end) of a
 * [T][C][N] cube; out points at row t_begin. */
void corrgen_gauss_i8(int8_t *out, long t_begin, long t_end, long n_chan, long n_inputs,
                      uint64_t seed, double sigma, double clip, double tone_amp, int threads)
{
    const uint64_t key = mix64(seed);
    (void)threads;
#pragma omp parallel for schedule(static) num_threads(threads > 0 ? threads : 1)
    for (long t = t_begin; t < t_end; ++t) {
        for (long c = 0; c < n_chan; ++c) {
            const double w = TWO_PI * (double)((c % 16) + 1) / 64.0;
            for (long i = 0; i < n_inputs; ++i) {
                const uint64_t e = (uint64_t)((t * n_chan + c) * n_inputs + i);
                double g_re, g_im;
                gauss_pair(key, e, &g_re, &g_im);
                double re = sigma * g_re, im = sigma * g_im;
                if (tone_amp != 0.0) {
                    const double ph = w * (double)t + tone_phase(seed, c, n_inputs, i);
                    re += tone_amp * cos(ph);
                    im += tone_amp * sin(ph);
                }
                int8_t *o = out + 2 * (((t - t_begin) * n_chan + c) * n_inputs + i);
                o[0] = (int8_t)clipd(rint(re), clip);
                o[1] = (int8_t)clipd(rint(im), clip);
            }
        }
    }
}

/* Uniform integers in [-clip, clip] for re and im. */
void corrgen_uniform_i8(int8_t *out, long t_begin, long t_end, long n_chan, long n_inputs,
                        uint64_t seed, int clip, int threads)
{
    const uint64_t key = mix64(seed);
    const uint64_t span = (uint64_t)(2 * clip + 1);
    (void)threads;
#pragma omp parallel for schedule(static) num_threads(threads > 0 ? threads : 1)
    for (long t = t_begin; t < t_end; ++t) {
        for (long c = 0; c < n_chan; ++c) {
            for (long i = 0; i < n_inputs; ++i) {
                const uint64_t e = (uint64_t)((t * n_chan + c) * n_inputs + i);
                const uint64_t h1 = mix64(key ^ (2 * e));
                const uint64_t h2 = mix64(key ^ (2 * e + 1));
                int8_t *o = out + 2 * (((t - t_begin) * n_chan + c) * n_inputs + i);
                o[0] = (int8_t)((long)((h1 >> 32) % span) - clip);
                o[1] = (int8_t)((long)((h2 >> 32) % span) - clip);
            }
        }
    }
}

/* Gaussian (+ optional tone) complex float32. */
void corrgen_gauss_f32(float *out, long t_begin, long t_end, long n_chan, long n_inputs,
                       uint64_t seed, double sigma, double tone_amp, int threads)
{
    const uint64_t key = mix64(seed);
    (void)threads;
#pragma omp parallel for schedule(static) num_threads(threads > 0 ? threads : 1)
    for (long t = t_begin; t < t_end; ++t) {
        for (long c = 0; c < n_chan; ++c) {
            const double w = TWO_PI * (double)((c % 16) + 1) / 64.0;
            for (long i = 0; i < n_inputs; ++i) {
                const uint64_t e = (uint64_t)((t * n_chan + c) * n_inputs + i);
                double g_re, g_im;
                gauss_pair(key, e, &g_re, &g_im);
                double re = sigma * g_re, im = sigma * g_im;
                if (tone_amp != 0.0) {
                    const double ph = w * (double)t + tone_phase(seed, c, n_inputs, i);
                    re += tone_amp * cos(ph);
                    im += tone_amp * sin(ph);
                }
                float *o = out + 2 * (((t - t_begin) * n_chan + c) * n_inputs + i);
                o[0] = (float)re;
                o[1] = (float)im;
            }
        }
    }
}
