/*
 * corr_diag.h -- DIAGNOSTICS of the B200 X-engine library.  Not part of the product ABI (include/corr.h):
 * these entry points exist only in libcorr_diag.so, the same sources compiled with -DCORR_DIAG, which also
 * carries a second, probe-instrumented instantiation of the int8 kernels.  The product library libcorr.so
 * has one instantiation of each hot kernel and none of this.
 *
 * Used by bench.py for the roofline denominators MEASURED_PEAKS.json does not hold (int8 tensor rate, FP32
 * FMA rate) and by the where-the-time-goes study of DESIGN.md section 7.  Results computed while a probe
 * mode is on are garbage by design; no test of results uses them.
 */
#ifndef CORR_DIAG_H_
#define CORR_DIAG_H_

#include "corr.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Experiment keys of corr_set_option (corr.h): A/B switches of the where-the-time-goes study, kept out of the product
 * header because no user of the library needs them.  Both builds accept them -- the parity tests force these paths in
 * the product kernels (tests/test_parity_gpu.py, tests/test_fuzz_gpu.py) -- but they may change or go without notice.
 */
enum { CORR_OPT_UNITS = 4,      /* > 0: at most that many CTAs walk the schedule (single-CTA plans); 0 = all SMs */
       CORR_OPT_PDL = 6,        /* programmatic dependent launch of the single-CTA int8 kernel: 0 never; 1 (default) inside a
                                   stream capture and for inputs above 64 MB; 2 always                           */
       CORR_OPT_COLLECT = 7     /* 0: 512-wide pair tiles read A twice per k-step; 1 (default): collector reuse */ };
/* CORR_OPT_PAIRS = 2: CTA pairs from N_I = 128 up (the supported values 0 | 1 are in corr.h) */

/*
 * corr_set_probe -- switches engines of the CI8 kernel off so that the others can be timed alone.  Bit
 * mask: 1 = skip the MMAs, 2 = skip the TMA loads (producer only hand-shakes), 4 = no epilogue, 8 = no
 * producer and no stage hand-shake at all, 16 = epilogue without its global stores, 128 = results stay correct, the
 * MMA issuer and the first TMA producer of every CTA (pair) count the SM cycles they spend waiting; 0 = normal.
 * corr_probe_stats (after a launch with bit 128, synchronised by the caller): out[0..3] = mean over the CTAs (pairs)
 * of the kernel's cycles, the MMA issuer's cycles waiting for a loaded stage, its cycles waiting for a free
 * TMEM accumulator, and the producer's cycles waiting for a free stage.
 */
int corr_set_probe(corr_handle *h, int mode);
int corr_probe_stats(corr_handle *h, double *out);

/*
 * corr_probe_mma -- tcgen05.mma.kind::i8 issue rate on the current device (the int8 tensor peak of the
 * roofline).  M in {64,128}, N multiple of 16 <= 256, K = 32; mn_major = 1 for the operand layout the
 * fused corner turn produces, 0 for K-major (add 2 for pseudo-random instead of zero operand bytes).
 * out[0] = kernel ms, out[1] = SM cycles per MMA, out[2] = dense TOP/s over all SMs, out[3] = effective
 * SM MHz during the loop.  No global-memory traffic.
 */
int corr_probe_mma(int m, int n, int mn_major, int iters, double *out);

/*
 * corr_probe_ffma -- FP32 FMA issue rate on the current device (the "alu" roofline denominator of the
 * float X-engine): one CTA of 1024 threads per SM, 16 independent register-resident FMA chains per thread,
 * `iters` rounds; packed = 0: scalar fma.rn.f32, 1: fma.rn.f32x2 (what xengine_f32_n64_kernel issues).
 * out[0] = kernel ms, out[1] = TFLOP/s over all SMs (2 flops per FMA, over the slowest SM's loop),
 * out[2] = effective SM MHz during the loop.
 */
int corr_probe_ffma(int packed, int iters, double *out);

#ifdef __cplusplus
}
#endif
#endif /* CORR_DIAG_H_ */
