/*
 * corr.h -- C ABI of the B200 X-engine (cross-multiply-accumulate, CMAC) library.
 *
 * What the library computes (the operation, from the paper):
 *   "an FX correlator ... does a channel-by-channel multiplication ('X') of the first
 *    spectrum with the complex conjugate of the second ... accumulated for each
 *    baseline"                                                   (sec. 2)
 *   "The correlation products for a given frequency channel can be represented in a
 *    matrix of size N_I x N_I formed by the outer product of a vector with its complex
 *    conjugate"; auto-correlations on the diagonal, the two halves redundant
 *                                                      (Fig. 2 at :115)
 *   N_I(N_I+1)/2 products per channel, autos included
 *   accumulators summed over the integration, then read out       (Fig. 1)
 *
 *   V[c][b(i,j)] = sum_{t=0}^{T-1} x[t][c][i] * conj(x[t][c][j]),  i >= j,
 *   b(i,j) = i(i+1)/2 + j   (row-major lower triangle; readings R1, R2)
 *
 * Raw sums are emitted; the division by the update count the paper does at read-out
 * is left to the caller (reading R3).
 *
 * Every pointer named d_* is DEVICE memory; h_* is HOST memory.  No torch types, no
 * exceptions cross this boundary.  There is no CPU fallback: every entry point that
 * computes needs an sm_100 device and fails with an error code otherwise.
 */
#ifndef CORR_H_
#define CORR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct corr_handle corr_handle; /* opaque */

/* dtype of the voltage samples */
enum { CORR_CI8 = 0,   /* (int8 re, int8 im) -> (int32 re, int32 im), exact            */
       CORR_CF32 = 1,  /* (float re, float im) -> (float re, float im), FP32 FMA sums  */
       CORR_CI4 = 2    /* one byte per sample: low nibble Re, high nibble Im, 4-bit two's
                          complement (the paper's "1-byte mode"; DESIGN R18)
                          -> (int32 re, int32 im), exact; d_in is [n_time][n_chan][n_inputs] bytes */ };

/* status codes */
enum { CORR_OK = 0, CORR_EINVAL = 1, CORR_EUNSUPPORTED = 2, CORR_EALLOC = 3,
       CORR_ECUDA = 4, CORR_EARCH = 5 };

/* how the corner turn (the "unpack" transpose) is realised, CI8 only */
enum { CORR_TURN_FUSED = 0,     /* the TMA box load of the CMAC kernel is the corner turn   */
       CORR_TURN_STANDALONE = 1 /* corr_corner_turn into handle scratch, then the CMAC kernel */ };

/*
 * corr_create -- plan one X-engine shape on the current CUDA device.
 *   n_inputs N_I : multiple of 32, 32..4096   (the paper needs G | N_I)
 *   n_chan   C   : >= 1
 *   n_time   T   : >= 1; for CORR_CI8 also T <= 65535 so that no int8 input can
 *                  overflow int32 (|V| <= T*2*128^2; reading R6)
 *   dtype        : CORR_CI8, CORR_CF32 or CORR_CI4 (T <= 65535 for CORR_CI4 as well)
 * Returns NULL on failure; corr_last_error()/corr_last_status() say why
 * (CORR_EINVAL, CORR_EUNSUPPORTED shape, CORR_EARCH not sm_100, CORR_EALLOC, CORR_ECUDA).
 * The handle owns its device workspaces (tile schedule, corner-turn scratch) until
 * corr_destroy.  One handle is used from one host thread at a time.
 */
corr_handle *corr_create(int n_inputs, int n_chan, int n_time, int dtype);

/*
 * corr_xengine -- one whole integration.  Asynchronous on `stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream); no host sync.
 *   d_in  : device, [n_time][n_chan][n_inputs] interleaved complex (input index fastest:
 *           the order the paper's aggregator emits).
 *           CI8: int8 re, int8 im (2 B/sample).  CF32: float re, float im (8 B/sample).
 *           16-byte aligned; read only.
 *   d_vis : device, [n_chan][N_I(N_I+1)/2] interleaved complex (int32 or float pairs),
 *           OVERWRITTEN with the raw sums of this call (reading R4); 16-byte aligned;
 *           must not alias d_in.  Im of every autocorrelation is exactly 0.
 * An integration that does not fill the chip (config 1: 8 MB) is LATENCY-bound through this call -- a launch, a
 * pipeline fill and one exposed DRAM round trip per call, 0.2 of the HBM roofline however it is enqueued; the
 * throughput path for such inputs is corr_xengine_batch below (0.8 of the roofline at 32 integrations per launch).
 * Returns CORR_OK, CORR_EINVAL (NULL / misaligned pointers, NULL handle) or CORR_ECUDA.
 */
int corr_xengine(corr_handle *h, const void *d_in, void *d_vis, void *stream);

/* corr_destroy -- frees the handle's workspaces.  NULL is a no-op.  Returns CORR_OK. */
int corr_destroy(corr_handle *h);

/* Thread-local text / code of the last failure on this thread; never NULL. */
const char *corr_last_error(void);
int corr_last_status(void);

/* Sizes in bytes of one integration's input and output for this handle. */
size_t corr_in_bytes(const corr_handle *h);  /* T*C*N*2 (CI8), T*C*N (CI4) or T*C*N*8 (CF32) */
size_t corr_vis_bytes(const corr_handle *h); /* C*N(N+1)/2*8                    */

/* Number of kernel launches one corr_xengine call enqueues (for bench accounting). */
int corr_launches_per_call(const corr_handle *h);

/*
 * corr_set_turn -- CI8 only: choose the corner-turn realisation (default CORR_TURN_FUSED).
 * CORR_TURN_STANDALONE allocates an in_bytes-sized scratch on first use.
 */
int corr_set_turn(corr_handle *h, int mode);

/*
 * corr_set_accumulate -- accumulate mode (each batch's products are ADDED to the
 * accumulators).  on != 0: corr_xengine adds the sums of its integration to d_vis instead of overwriting
 * it; the caller zeroes d_vis and calls corr_set_accumulate(h, 1) at the START of every accumulation --
 * the call resets the handle's update counter.  int32 accumulators cannot hold an arbitrary number of
 * batches: corr_xengine returns CORR_EUNSUPPORTED (and adds nothing) once another batch could overflow
 * them for SOME input, i.e. when (count + 1) * T * 2 * 128^2 >= 2^31 (CORR_CI8) or
 * (count + 1) * T * 2 * 8^2 >= 2^31 (CORR_CI4); CORR_CF32 has no such bound.  For longer accumulations
 * use corr_accumulate_wide.  corr_accumulate_count returns the number of batches added so far.
 */
int corr_set_accumulate(corr_handle *h, int on);
long long corr_accumulate_count(const corr_handle *h);

/*
 * corr_accumulate_wide -- one batch added into accumulators twice as wide (read out "after a
 * specified time, usually a few seconds"): the integration of d_in is computed into a
 * handle-owned buffer (corr_vis_bytes) and then folded, acc[k] += vis[k], into
 *   d_acc : device, [n_chan][N_I(N_I+1)/2] (int64 re, int64 im) for CORR_CI8 / CORR_CI4 -- exact for any
 *           number of batches -- or (double re, double im) for CORR_CF32; corr_acc_bytes(h) bytes,
 *           16-byte aligned, zeroed by the caller before the first batch.
 * Independent of corr_set_accumulate.  Asynchronous on `stream`.  Every call on one handle stages its batch in the
 * same handle-owned buffer: calls on ONE handle must be stream-ordered (one stream, or events between streams) --
 * two accumulations double-buffered over two streams need two handles.  Returns CORR_OK, CORR_EINVAL, CORR_EALLOC
 * or CORR_ECUDA.  corr_normalize_wide is the read-out of d_acc (count = samples accumulated) into
 * (float re, float im), d_out of corr_vis_bytes(h) bytes.
 */
int corr_accumulate_wide(corr_handle *h, const void *d_in, void *d_acc, void *stream);
int corr_normalize_wide(corr_handle *h, const void *d_acc, double count, void *d_out, void *stream);
size_t corr_acc_bytes(const corr_handle *h); /* 2 * corr_vis_bytes */

/*
 * corr_accumulate_wide_static -- corr_accumulate_wide for callers that must not allocate device memory.
 *
 * Who needs it: a correlator's real-time loop, or a plug-in living inside a host application that has already
 * handed all of the GPU's memory to its own pool.  cudaMalloc / cudaFree synchronise the whole device (every
 * stream stalls while they run, which a loop with a sample-rate deadline cannot afford), they can fail once another
 * owner holds the memory, and some hosts simply forbid them after start-up.  corr_accumulate_wide allocates its
 * batch buffer (corr_vis_bytes) on the handle's first call; this entry point never does.  The batch of
 * PAPER.md:125 / :166 is computed into a buffer that is part of the library image itself: a fixed device array
 * of CORR_STATIC_BATCH_BYTES, which every GPU that loads the library carries from load to process exit, used or
 * not.  The batch is then folded, acc[k] += vis[k], into the caller's d_acc exactly as corr_accumulate_wide does
 * (same arguments, same results bit for bit).  With a CORR_CI8 / CORR_CI4 handle the whole sequence corr_create ->
 * corr_accumulate_wide_static -> corr_normalize_wide -> corr_destroy makes no device allocation at all (a
 * CORR_CF32 handle allocates its work-item table in corr_create, none afterwards).
 *
 * Limits and rules:
 *   - corr_vis_bytes(h) <= CORR_STATIC_BATCH_BYTES, else CORR_EUNSUPPORTED and nothing is enqueued (of the paper-
 *     shaped configurations c1, c2 and c5-sized cubes up to 16 MiB fit; N_I = 256 x 512 channels does not);
 *   - no cudaMalloc, cudaFree or allocating library routine is called, on any call;
 *   - the FIRST call on each device looks up the array's device address (one query, with that device current,
 *     which may make the CUDA runtime finish loading the library's module): make that call during set-up,
 *     before any stream capture and before the deadline-bound loop starts; later calls on that device only launch;
 *   - the array is shared by every handle, stream and thread of the process on that GPU and keeps whatever the
 *     last call left in it.  Nothing in it has to start at zero -- each call overwrites (or, for time-sliced plans,
 *     clears on `stream` and then fills) the corr_vis_bytes(h) it uses before folding them -- but two calls whose
 *     GPU work can overlap (different streams without an event between them, or two host threads) RACE on it and
 *     corrupt both accumulations.  Keep all calls on one device stream-ordered.
 * Asynchronous on `stream`.  Returns CORR_OK, CORR_EINVAL, CORR_EUNSUPPORTED or CORR_ECUDA (never CORR_EALLOC).
 */
#define CORR_STATIC_BATCH_BYTES (16u << 20)
int corr_accumulate_wide_static(corr_handle *h, const void *d_in, void *d_acc, void *stream);

/*
 * corr_normalize -- read-out (the accumulators are "divided by the number of times they were
 * updated"): d_out[c][b] = d_vis[c][b] / count as (float re, float im); d_vis holds int32 pairs (CI8, CI4)
 * or float pairs (CF32).  d_out has corr_vis_bytes(h) bytes, 16-byte aligned, may not alias d_vis unless the
 * dtype is CF32.  Asynchronous on `stream`.
 */
int corr_normalize(corr_handle *h, const void *d_vis, double count, void *d_out, void *stream);

/*
 * corr_xengine_batch -- n whole integrations in ONE launch ("it is most efficient to transfer
 * and process large batches of data per call"; 32 blocks of spectra per GPU call).  An
 * integration too small to fill the chip (config 1: 8 MB) costs a launch, a pipeline fill and one exposed
 * DRAM round trip per call; here the tile schedule spans all n inputs, so every SM streams for the whole call.
 *   d_in  : HOST array of n device pointers, each as corr_xengine's d_in
 *   d_vis : HOST array of n device pointers, each as corr_xengine's d_vis.  No d_vis[k] may overlap another entry's
 *           d_vis or ANY entry's d_in (CORR_EINVAL, nothing enqueued): in the single launch all integrations run
 *           at once.  Only in accumulate mode (call by call on `stream`) may several entries name one d_vis.
 *   n     : >= 1; more than 64 integrations are issued as several launches of <= 64
 * Same result as n corr_xengine calls (bit-exact for CI8).  The single-launch path covers CORR_CI8 shapes
 * that run on single CTAs (corr_plan_info: CORR_KERNEL_I8 -- N_I <= 192, and N_I < 512 with 1024 < T < 2048); every other
 * case (CTA-pair plans, CORR_CI4, CORR_CF32, the standalone corner turn, accumulate mode) falls back to n
 * ordinary calls on `stream`.  Returns as corr_xengine.
 */
int corr_xengine_batch(corr_handle *h, const void *const *d_in, void *const *d_vis, int n, void *stream);

/*
 * corr_set_chan_window -- channel-sharded use ("The products are formed
 * independently for each frequency channel"): the handle (created with n_chan = the window's
 * width) reads channels chan0 .. chan0 + n_chan - 1 of a buffer d_in[n_time][n_chan_total][n_inputs] IN
 * PLACE -- no copy, the TMA tensor map / the float kernels take the full row as their time stride -- and
 * writes its own [n_chan][N_I(N_I+1)/2] block to d_vis.  After the call corr_in_bytes(h) is the size of
 * the FULL buffer.  n_chan_total >= chan0 + n_chan, chan0 >= 0; (n_chan_total, 0) with n_chan_total ==
 * n_chan restores the default.  CORR_EINVAL otherwise.  All dtypes, both corner-turn realisations.
 */
int corr_set_chan_window(corr_handle *h, int n_chan_total, int chan0);

/*
 * corr_set_option -- forces a plan family, for the tests that must reach every schedule and for measurements
 * (DESIGN.md section 7).  Each call re-plans the handle; the defaults are what corr_create chose.  CORR_EINVAL for an
 * unknown key or a value out of range.  The keys below are the supported ones; the experiment switches of the
 * where-the-time-goes study (CTA count, dependent launches, collector reuse, CTA pairs below N_I = 256) are declared in
 * corr_diag.h and are no part of this ABI.
 */
enum { CORR_OPT_DIAG_PLAN = 1,  /* N_I <= 64: value = 256 * gsize + slices forces `gsize` (1, 2, 4) adjacent
                                   panels per work item and `slices` (1..64) time slices (slices = 0: only the
                                   group width is forced, whatever the input size, corr_xengine_batch
                                   included); 0 = automatic                                                 */
       CORR_OPT_PAIRS = 2,      /* 0: single-CTA slab items only; 1 (default): CTA pairs (cta_group::2) where planned */
       CORR_OPT_WIDE = 3,       /* 0: no 512-wide pair tiles; 1 (default): for T >= 2048; 2: for every T       */
       CORR_OPT_F32_GENERIC = 5,/* 1: N_I = 64 float input runs the generic kernel instead of the N_I = 64 one */
       CORR_OPT_RESIDENT = 8,   /* 0: no resident-A plan (N_I >= 256, T <= 1024, or <= 1152 up to N_I = 512: a CTA pair keeps
                                   its A panel of the whole integration in shared memory); 1 (default): where it
                                   was measured to pay; 2: wherever it fits (T <= 1152)                        */
       CORR_OPT_MIX = 9         /* 0: N_I <= 64 with more work groups than SMs: every group in the same number of time
                                   slices; 1 (default): whole groups plus sliced left-over groups                */ };
int corr_set_option(corr_handle *h, int key, int value);

/*
 * corr_plan_info -- what the handle's current plan (corr_create, then every corr_set_option / corr_set_turn) will launch
 * for corr_xengine; read-only, for benchmarks, profiles and tests that have to name the kernel and schedule they measured
 * instead of re-deriving the planner's thresholds.  info: HOST array of CORR_PLAN_INFO_LEN ints indexed by CORR_PLAN_*;
 * kernel: optional HOST buffer that receives the kernel's function name (NULL or kernel_len = 0 to skip).
 */
enum { CORR_PLAN_KERNEL = 0,  /* CORR_KERNEL_* below                                                          */
       CORR_PLAN_GSIZE = 1,   /* N_I <= 64: adjacent panels (CI8 / CI4) or channels (CF32, N_I = 64) per work item; else 0 / 1 */
       CORR_PLAN_SLICES = 2,  /* time slices per group (the sliced groups' count when CORR_PLAN_MIXED)        */
       CORR_PLAN_GRID = 3,    /* CTAs per launch                                                             */
       CORR_PLAN_MIXED = 4,   /* 1: whole groups plus sliced left-over groups                                */
       CORR_PLAN_STAGES = 5,  /* depth of the TMA stage ring (int8 / 4-bit kernels)                          */
       CORR_PLAN_WIDE = 6,    /* 1: the pair plan contains 512-wide tiles                                    */
       CORR_PLAN_SMEM = 7,    /* dynamic shared memory per CTA, bytes (int8 / 4-bit kernels)                 */
       CORR_PLAN_INFO_LEN = 8 };
enum { CORR_KERNEL_I8 = 0, CORR_KERNEL_I8_PAIR = 1, CORR_KERNEL_I8_PAIR_RESIDENT = 2, CORR_KERNEL_I4 = 3,
       CORR_KERNEL_F32 = 4, CORR_KERNEL_F32_N64 = 5 };
int corr_plan_info(const corr_handle *h, int *info, char *kernel, size_t kernel_len);

/*
 * corr_corner_turn -- the standalone corner-turn kernel, CI8 or CF32:
 *   d_in  [T][C][N] samples  ->  d_out [C][T][N] samples (per-channel, time-major tiles),
 * 16-byte vectorised coalesced loads and stores through a shared-memory tile.  Pure byte
 * permutation.  d_out has corr_in_bytes(h) bytes, 16-byte aligned, must not alias d_in.
 */
int corr_corner_turn(corr_handle *h, const void *d_in, void *d_out, void *stream);

/*
 * Streaming driver (staging + H2D of the next batch
 * overlapped with the CMAC of the previous one).
 *   h_in  : n_integrations pointers to PINNED host buffers, corr_in_bytes(h) each
 *   d_vis : device, n_integrations * corr_vis_bytes(h) bytes (integration k at offset k*vis_bytes)
 * Copies integration k+1 on a side stream while the X-engine runs integration k on the
 * compute stream (two device input buffers owned by the handle).  Blocks until done.
 * On success writes to stats (if not NULL): [0] wall seconds (host clock around the whole run),
 * [1] device seconds (CUDA events, first copy start -> last kernel end),
 * [2] sum of kernel seconds, [3] sum of H2D copy seconds.
 */
int corr_stream_run(corr_handle *h, const void *const *h_in, int n_integrations,
                    void *d_vis, double *stats);

/* ------------------------------------------------------------------------------------------------
 * F-stage: the two steps in front of the CMAC in the paper's correlator,
 *   "1- unpacking a block of data, which involves reordering samples ... 2- Fourier transforming into
 *    frequency space"
 *   "taking a block of N_I x N_C complex samples which are ordered with input varying most quickly,
 *    converting to floating-point format and putting the samples into N_I arrays of length N_C"
 *
 *   "the FFT is N_C channels in input and output"
 *
 *   X[b][k][i] = sum_{n=0}^{N_C-1} x[b][n][i] * exp(-2 pi i k n / N_C)
 *
 * forward sign, unnormalised, natural channel order k = 0 (DC) first (readings R19, R20).
 *   d_raw  : device, [n_batch][n_fft][n_inputs] complex int8 (int8 re, int8 im; any 5+5-bit sample of
 *            PAPER.md:69 is one; reading R21), input index fastest; 16-byte aligned; read only.
 *   d_spec : device, [n_batch][n_fft][n_inputs] (float re, float im), overwritten; 16-byte aligned; must
 *            not alias d_raw.  With n_batch = n_time * n_bands this IS corr_xengine's CF32 input
 *            [n_time][n_chan = n_bands * n_fft][n_inputs].
 * corr_fstage_create: n_fft must be 128 (the paper's N_C), n_inputs a multiple of 32 and
 * <= 4096, n_batch >= 1; NULL + corr_last_error() otherwise (CORR_EINVAL / CORR_EUNSUPPORTED / CORR_EARCH /
 * CORR_ECUDA / CORR_EALLOC).  corr_fstage_run is asynchronous on `stream`; returns CORR_OK, CORR_EINVAL or
 * CORR_ECUDA.  FP32 arithmetic: |dX| <= 1e-5 * ||x[b][:][i]||_2 per channel against the float64 definition
 * (DESIGN.md section 6).  The handle owns device memory only once corr_stream_run_fx has been used; corr_fstage_destroy(NULL) is a no-op.
 */
typedef struct corr_fstage corr_fstage; /* opaque */
corr_fstage *corr_fstage_create(int n_inputs, int n_fft, int n_batch);
int corr_fstage_run(corr_fstage *f, const void *d_raw, void *d_spec, void *stream);
int corr_fstage_destroy(corr_fstage *f);
/*
 * corr_fstage_set_input -- raw sample format: CORR_CI8 (default, above) or CORR_CI4, the paper's "1-byte mode"
 * ("reduced from 2-byte words to a single byte, at the cost of 1 bit of precision ... reduces the
 * total amount of global memory reads in the unpack phase"): d_raw is [n_batch][n_fft][n_inputs] BYTES, low nibble
 * Re, high nibble Im, 4-bit two's complement (DESIGN reading R18).  corr_fstage_in_bytes follows.  CORR_EINVAL otherwise.
 */
int corr_fstage_set_input(corr_fstage *f, int dtype);
size_t corr_fstage_in_bytes(const corr_fstage *f);  /* n_batch * n_fft * n_inputs * 2 (CI8) or * 1 (CI4) */
size_t corr_fstage_out_bytes(const corr_fstage *f); /* n_batch * n_fft * n_inputs * 8 */

/*
 * corr_stream_run_fx -- the streaming driver fed with RAW VOLTAGES: per integration the
 * host->device copy moves corr_fstage_in_bytes(f) bytes of complex int8 (a quarter of the float spectra),
 * then F-stage and X-engine run back to back on the compute stream while the next copy is in flight --
 * the paper's whole chain unpack -> FFT -> CMAC on the device.
 *   h     : CORR_CF32 handle with n_time * n_chan * n_inputs == n_batch * n_fft * n_inputs of f
 *   h_raw : n_integrations pointers to PINNED host buffers of corr_fstage_in_bytes(f) bytes
 *   d_vis, stats : as corr_stream_run ([2] = sum of F + X kernel seconds).
 * The F-stage handle owns two raw buffers and one spectra buffer on the device from the first call on.
 * Tolerance of the chain against float64 arithmetic on the same raw voltages: |dV| <= 2e-5 sqrt(|V_ii V_jj|) --
 * two FP32 stages in a row, each good to 1e-5 of its own scale.
 */
int corr_stream_run_fx(corr_handle *h, corr_fstage *f, const void *const *h_raw, int n_integrations,
                       void *d_vis, double *stats);

#ifdef __cplusplus
}
#endif
#endif /* CORR_H_ */
