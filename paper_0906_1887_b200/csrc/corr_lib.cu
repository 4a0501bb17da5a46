// corr_lib.cu -- host side of the C ABI declared in include/corr.h.
// Plans the tile schedule (descendant of the paper's constant-memory pair lookup table,
// PAPER.md:117), encodes TMA tensor maps, launches the sm_100a kernels.  No CPU compute path.
#include "../../include/corr.h"
#include "../../include/corr_diag.h"  // the experiment keys of corr_set_option; its entry points are compiled under CORR_DIAG only

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <mutex>
#include <queue>
#include <vector>

#include "corner_turn.cuh"
#include "fengine.cuh"
#include "readout.cuh"
#ifdef CORR_DIAG
#include "probe_mma.cuh"
#endif
#include "xengine_f32.cuh"
#include "xengine_f32_n64.cuh"
#include "xengine_i8.cuh"

// Batch buffer of corr_accumulate_wide_static (include/corr.h): device memory that belongs to the library image, so
// that the entry point has nothing to allocate.  Host code may NOT use this name as a pointer -- on the host it is only
// a stand-in for the symbol; static_batch_ptr() below asks the runtime for the array's address on the current device.
static __device__ __align__(256) unsigned char g_static_batch[CORR_STATIC_BATCH_BYTES];

// corr::fold_wide_kernel (readout.cuh) with the batch read from g_static_batch: device code names the array directly.
// acc[k] += batch[k], int32 -> int64 or float -> double, n scalars (a multiple of 4), 16-byte vectors, grid-stride.
__global__ void __launch_bounds__(256) fold_wide_static_kernel(void *acc, long long n, int is_int) {
  const long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
  for (long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; k < n / 4; k += stride) {
    if (is_int) {
      const int4 v = reinterpret_cast<const int4 *>(g_static_batch)[k];
      longlong2 *a = reinterpret_cast<longlong2 *>(acc) + 2 * k;
      longlong2 a0 = a[0], a1 = a[1];
      a0.x += v.x; a0.y += v.y; a1.x += v.z; a1.y += v.w;
      a[0] = a0; a[1] = a1;
    } else {
      const float4 v = reinterpret_cast<const float4 *>(g_static_batch)[k];
      double2 *a = reinterpret_cast<double2 *>(acc) + 2 * k;
      double2 a0 = a[0], a1 = a[1];
      a0.x += v.x; a0.y += v.y; a1.x += v.z; a1.y += v.w;
      a[0] = a0; a[1] = a1;
    }
  }
}

namespace {

thread_local char g_err[512] = "";
thread_local int g_status = CORR_OK;

int fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  g_status = code;
  return code;
}
#define CUDA_TRY(call)                                                                        \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) return fail(CORR_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

struct MapCacheEntry {
  const void *ptr;
  corr::I8Maps maps;  // box heights 256, 128, 64 time rows
};

constexpr int kMaxSmemI8 = 232448;  // sm_100 opt-in maximum of dynamic shared memory per CTA (227 KB)

}  // namespace

// One planned launch of the int8 kernels: schedule + problem (passed by value into the constant bank), grid, shared memory.
struct I8Plan {
  corr::I8Params ip;
  int grid;
  size_t smem;
  int zero_vis;  // d_vis is zeroed before the launch (items reduce-add: time slices or a mixed plan)
  int zero_from_chan;  // ... from this channel on (mixed plans: the whole groups in front store plainly)
  int n_batch;  // 0: not planned yet
};

struct corr_handle {
  int n_inputs, n_chan, n_time, dtype;
  int n_chan_total, chan0;  // channel window (corr_set_chan_window): d_in is [T][n_chan_total][N], this handle owns chan0 .. chan0 + n_chan - 1
  long long n_baselines;
  size_t in_bytes, vis_bytes;  // buffer sizes (in_bytes: of the FULL cube when the handle owns a channel window)
  size_t work_bytes;           // input bytes this handle actually reads per call: what the planner and the launch mode go by
  int n_sms;
  int turn_mode;
  int probe;
  int accumulate;
  long long acc_count;      // batches added since corr_set_accumulate(h, 1)
  // plan options (corr_set_option)
  int opt_diag_plan, opt_pairs, opt_wide, opt_units, opt_f32_generic, opt_pdl, opt_collect, opt_resident, opt_mix;
  // CI8 / CI4 plans
  int pair_mode;
  I8Plan plan;        // corr_xengine
  I8Plan plan_batch;  // corr_xengine_batch, planned for the batch size last seen
  void *d_scratch;    // corner-turn output (standalone mode)
  void *d_wide_vis;   // one batch's sums on their way into the wide accumulators (corr_accumulate_wide)
  unsigned long long *d_diag_stats;  // diagnostics build only (corr_probe_stats)
  std::vector<MapCacheEntry> maps;
  // CF32 plan
  int2 *d_items_f32;
  int n_items_f32;
  int f32_threads;
  int n64_groups, n64_slices, n64_slice_len, n64_full;  // CF32 with N_I = 64: xengine_f32_n64_kernel
  // streaming driver
  void *d_stream_in[2];
  cudaStream_t s_copy, s_compute;
};

struct corr_fstage {
  int n_inputs, n_fft, n_batch, in_dtype;
  int device;  // the twiddle table lives in this device's constant memory
  size_t in_bytes, out_bytes;
  void *d_raw[2];  // streaming driver: double-buffered raw voltages
  void *d_spec;    // streaming driver: spectra of the integration in flight
};

namespace {

// Schedule planning (host side of the uniform decode in xengine_i8.cuh) for a launch over n_batch integrations.
void plan_i8(const corr_handle *h, int n_batch, I8Plan *out) {
  corr::I8Params &ip = out->ip;
  memset(&ip, 0, sizeof ip);
  out->n_batch = n_batch;
  out->zero_vis = 0;
  out->zero_from_chan = 0;
  const int N = h->n_inputs, C = h->n_chan, T = h->n_time;
  const int panels_per_chan = h->pair_mode ? 1 : (2 * N + 127) / 128;
  ip.n_time = T; ip.n_inputs = N; ip.n_chan = C; ip.pair_mode = h->pair_mode;
  ip.n_baselines = h->n_baselines;
  ip.n_batch = n_batch;
  ip.diag = panels_per_chan == 1;
  const bool use_pairs = h->dtype == CORR_CI8 && h->opt_pairs && n_batch == 1;  // the 4-bit path and batched launches are single-CTA only
  int max_load = 1;
  if (ip.diag) {
    ip.n_panels = h->pair_mode ? (C + 1) / 2 : C;
    // Items are the diagonal blocks of `gsize` ADJACENT panels over one time slice.  Large inputs: gsize = 4
    // (512-byte HBM runs) and as many time slices as fill the grid evenly (slices accumulate with reduce-add
    // into a zeroed d_vis).  Small inputs (<= 64 MB) are latency-bound: the zeroing node, the reduce-adds and
    // their completion waits cost more than the load itself, so the plan with the least modelled time is
    // taken, which usually is whole integrations (no slices) of 1 or 2 panels spread over more SMs.
    const int G = h->n_sms;
    int best_g = 4, best_s = 1;
    double best_t = 1e30;
    const bool small = h->work_bytes <= (64u << 20);
    const int forced_g = h->opt_diag_plan >> 8;  // CORR_OPT_DIAG_PLAN: the group width is forced in every branch below
    if (n_batch > 1) {
      // batched launch: whole integrations (no zeroing nodes), the panel-group width that keeps the SMs evenly
      // loaded.  When one time row has no more panels than there are SMs, the CTAs working side by side consume
      // whole rows between them and even single 128-byte runs fetch at the full rate (c1 in batches of 32: 1.47 us
      // per integration with 1 panel per item, 1.51 with 2, 1.59 with 4); otherwise narrower HBM runs fetch slower
      // (128-byte runs at a 96 KB stride: 3.7 TB/s, 512-byte runs: 5.4 TB/s).
      const bool rows_shared = ip.n_panels <= G;
      const double rate[5] = {0.0, rows_shared ? 1.0 : 0.70, rows_shared ? 1.0 : 0.92, 0.0, 1.0};
      for (int g = 1; g <= 4; g <<= 1) {
        if (forced_g && g != forced_g) continue;
        const long long n = 1LL * ((ip.n_panels + g - 1) / g) * n_batch;
        const long long rounds = (n + G - 1) / G;
        const double t = rounds * g / rate[g];
        if (t < best_t * 0.999) { best_t = t; best_g = g; }
      }
    } else if (small) {
      for (int g = 4; g >= 1; g >>= 1) {
        if (forced_g && g != forced_g) continue;
        const int base = (ip.n_panels + g - 1) / g;
        for (int s = 1; s <= 64; ++s) {
          int len = ((T + s - 1) / s + 63) / 64 * 64;
          if (len < 128 && s > 1) break;
          const int s_eff = (T + len - 1) / len;
          if (s_eff != s) continue;
          const long long n = 1LL * base * s;
          const long long rounds = (n + G - 1) / G;
          // modelled time: rounds x (item bytes at ~80 GB/s per SM) + the fixed cost of a sliced launch
          const double t = 1e-9 * rounds * (1.0 * g * 128 * std::min(len, T)) / 80.0 + (s > 1 ? 4e-6 : 0.0);
          if (t < best_t - 1e-7) { best_t = t; best_g = g; best_s = s; }
        }
      }
    }
    int mix_sl = 0, mix_len = 0;  // > 0: mixed plan (whole groups + the left-over groups in mix_sl slices of mix_len)
    if (n_batch == 1 && !small) {
      // Large inputs stream from HBM: model the busiest CTA's time for every (group width g, plan) and take the least.
      //   per sample a CTA streams g x 128 B at its share of the HBM rate (narrower runs fetch a little slower);
      //   per item it pays the part of the epilogue the next item's loads cannot hide: all of it with g = 4 (the four
      //   accumulators fill TMEM), little with g = 2 (double-buffered), more when the item reduce-adds;
      //   uniform plan: every group in s slices; mixed plan: a x G whole groups (plain stores, no zeroing) + the b
      //   left-over groups in s slices (c2: 148 whole + 44 groups in thirds).
      const double bw = 6.5e12 / G;
      const int g_lo = forced_g ? forced_g : 2, g_hi = forced_g ? forced_g : 4;
      for (int g = g_hi; g >= g_lo; g >>= 1) {
        const double ts = g * 128.0 / (bw * (g == 4 ? 1.0 : g == 2 ? 0.92 : 0.70));
        const double epi = g == 4 ? 4.0e-6 : 0.5e-6, epi_add = g == 4 ? 5.0e-6 : 1.0e-6;
        const int groups = (ip.n_panels + g - 1) / g;
        for (int sl = 1; sl <= 64; ++sl) {
          const int len = sl == 1 ? T : ((T + sl - 1) / sl + 63) / 64 * 64;
          if (sl > 1 && (len < 128 || (T + len - 1) / len != sl)) { if (len < 128) break; continue; }
          const long long rounds = (1LL * groups * sl + G - 1) / G;
          const double t = rounds * (std::min(len, T) * ts + (sl > 1 ? epi_add : epi)) + (sl > 1 ? 3e-6 : 0.0);
          if (t < best_t * 0.98) { best_t = t; best_g = g; best_s = sl; mix_sl = 0; }
          const int a = groups / G, b = groups % G;
          if (sl > 1 && a >= 1 && b > 0 && h->opt_mix && !(h->opt_diag_plan & 255)) {
            const long long r2 = (1LL * b * sl + G - 1) / G;
            const double tm = a * (T * ts + epi) + r2 * (len * ts + epi_add) + 2e-6;
            if (tm < best_t * 0.98) { best_t = tm; best_g = g; best_s = 1; mix_sl = sl; mix_len = len; }
          }
        }
      }
    }
    if (h->opt_diag_plan & 255) {  // corr_set_option(CORR_OPT_DIAG_PLAN): 256 * gsize + slices forces a uniform plan
      const int g = h->opt_diag_plan >> 8, sl = h->opt_diag_plan & 255;
      const int len = ((T + sl - 1) / sl + 63) / 64 * 64;
      if (sl == 1 || (len >= 128 && (T + len - 1) / len == sl)) { best_g = g; best_s = sl; mix_sl = 0; }
    }
    ip.gsize = best_g;
    ip.n_groups = (ip.n_panels + best_g - 1) / best_g;
    ip.n_kinds = 1;
    max_load = best_g;
    ip.n_slices = best_s;
    ip.slice_len = best_s == 1 ? T : ((T + best_s - 1) / best_s + 63) / 64 * 64;
    if (mix_sl > 1) {
      ip.mix_full = (ip.n_groups / G) * G; ip.mix_cut = ip.n_groups % G; ip.mix_len = mix_len;
      ip.n_groups = ip.mix_full + ip.mix_cut * mix_sl;   // group SLOTS of the walk
      // only the sliced groups' channels are zeroed: whole groups store (CI8); the 4-bit kernel reduce-adds everywhere
      out->zero_vis = 1;
      out->zero_from_chan = h->dtype == CORR_CI8 ? ip.mix_full * ip.gsize * (h->pair_mode ? 2 : 1) : 0;
    }
  } else {
    ip.n_panels = panels_per_chan;
    ip.n_groups = C;
    int k = 0;
    // CTA pairs (cta_group::2) from N_I = 512 up; already from N_I = 256 when the integration is long
    // enough (T >= 2048) for 512-wide tiles, whose epilogue cannot overlap the next tile's MMAs
    // ... and only up to N_I = 448: from 8 panels per channel on, 256-wide tiles find their panels in L2 and hide every
    // epilogue, which beats the 512-wide tiles' leaner operand traffic (N_I = 512 / 1024 / 2048 at T = 4000: 287 -> 238,
    // 480 -> 406, 819 -> 726 us)
    const bool long_ok = ((T >= 2048 && panels_per_chan < 8) || h->opt_wide == 2) && panels_per_chan >= 4;
    const bool wide_ok = long_ok && h->opt_wide;
    const int min_pair_panels = h->opt_pairs == 2 ? 2 : 8;  // CORR_OPT_PAIRS = 2 (experiments): CTA pairs from N_I = 128 up
    // the resident-A plan already from N_I = 256 (N_I = 256 / 384 at T = 1000: 185 -> 175, 252 -> 217 us against single-CTA slabs)
    const int min_res_panels = h->opt_pairs == 2 ? 2 : 4;
    // ... by measurement (round 3, 0.5 GB inputs, resident / best other plan): with 5 or 7 panels per channel (N_I = 288, 320,
    // 416, 448) the unit of two row pairs wastes a third / a quarter of its MMAs and single-CTA slabs win (1.03-1.16 at T = 500 ..
    // 1100); up to 1024 samples (4-stage B ring) the plan wins everywhere else (0.73-0.99); with 9 sub-stages (T <= 1152, 3-stage
    // ring) it still wins with 4, 6 and 8 panels (N_I = 256 / 384 / 512 at T = 1100: 0.96 / 0.90 / 0.92) and ties or loses above
    // (1.0-1.09 from N_I = 576 up); a 2-stage ring (T <= 1280) loses everywhere (1.05-1.3).  CORR_OPT_RESIDENT = 2 forces the
    // plan wherever it fits.
    const bool res_fits = T <= 128 * corr::kResMaxSub;
    const bool res_pays = T <= (panels_per_chan <= 8 ? 128 * corr::kResMaxSub : 1024) && panels_per_chan != 5 && panels_per_chan != 7;
    if (use_pairs && panels_per_chan >= min_res_panels && !long_ok && res_fits && (res_pays || h->opt_resident == 2) && h->opt_resident && h->turn_mode == CORR_TURN_FUSED) {
      // resident-A plan (xengine_i8_resident.cuh): the A panel of the whole integration stays in shared memory; an item
      // is a unit of two row pairs (pp - 1 - u and u: pp + 1 tiles in every unit)
      ip.pair2 = 1;
      ip.resident = 1;
      ip.a_sub = (T + 127) / 128;
      const int pp = (panels_per_chan + 1) / 2;
      for (int u = 0; u < (pp + 1) / 2; ++u) ip.kinds[k++] = static_cast<unsigned short>(u);
      max_load = 1;
    } else if (use_pairs && (panels_per_chan >= min_pair_panels || long_ok)) {
      ip.pair2 = 1;
      const int pp = (panels_per_chan + 1) / 2;
      max_load = 2;
      for (int Ip = pp - 1; Ip >= 0; --Ip) {
        const int ncols = 2 * Ip + 2;  // column panels 0 .. 2*Ip+1 are needed by row pair Ip
        for (int J0 = 0; J0 < ncols;) {
          const int wide = (wide_ok && ncols - J0 >= 4) ? 1 : 0;
          ip.kinds[k++] = static_cast<unsigned short>(Ip | ((J0 >> 1) << 6) | (wide << 11));
          if (wide) max_load = 3;
          J0 += wide ? 4 : 2;
        }
      }
    } else {
      for (int I = panels_per_chan - 1; I >= 0; --I)
        for (int J0 = 0; J0 <= I; J0 += 2) {
          const int nblk = std::min(2, I - J0 + 1);
          max_load = std::max(max_load, (I < J0 + nblk) ? nblk : nblk + 1);
          ip.kinds[k++] = static_cast<unsigned short>(I | ((J0 >> 1) << 6) | ((nblk - 1) << 11));
        }
    }
    ip.n_kinds = k;
    ip.n_slices = 1;
    ip.slice_len = T;
  }
  if (ip.n_slices > 1) out->zero_vis = 1;
  ip.n_items = ip.n_groups * ip.n_kinds * ip.n_slices * n_batch;
  ip.rot = ip.n_kinds > 1 ? 1 : 0;
  // 32 KB stages: 1 x 256, 2 x 128 or 4 x 64 time rows of 128 B; 48 KB when items fetch 3 panels (3 x 128).  The 4-bit
  // mode also keeps the packed bytes of every stage (half as many again): 24 KB stages (3 x 64 rows) there, so that the
  // ring stays 5 deep instead of 2
  ip.stage_bytes = (!ip.diag && max_load == 3) ? (h->dtype == CORR_CI4 ? 3 * 64 * 128 : 3 * 128 * 128) : 4 * 64 * 128;
  const int epi_bytes = corr::kEpiWarps * corr::kEpiWarpBytes;  // epilogue staging behind the stage ring
  const int bar_bytes = 512;  // 4 * kMaxStages + 4 mbarriers and the TMEM base address
  if (ip.resident) ip.stage_bytes = corr::kResSubBytes;
  const int a_bytes = ip.resident ? ip.a_sub * corr::kResSubBytes : 0;
  const int ring_bytes = h->dtype == CORR_CI4 ? ip.stage_bytes * 3 / 2 : ip.stage_bytes;  // + packed (raw) ring
  ip.stages = std::min<int>(corr::kMaxStages, (kMaxSmemI8 - bar_bytes - epi_bytes - a_bytes) / ring_bytes);
  out->smem = static_cast<size_t>(ring_bytes) * ip.stages + a_bytes + epi_bytes + bar_bytes;
  ip.units = std::min(ip.n_items, ip.pair2 ? h->n_sms / 2 : h->n_sms);
  if (h->opt_units > 0 && !ip.pair2) ip.units = std::min(ip.units, h->opt_units);  // experiments: fewer, fatter CTAs
  out->grid = ip.pair2 ? 2 * ip.units : ip.units;
  const int deltas[2] = {ip.units + ip.rot, ip.rot};
  for (int w = 0; w < 2; ++w) { ip.dq[w] = deltas[w] / ip.n_kinds; ip.dr[w] = deltas[w] % ip.n_kinds; }
}

void plan_f32(corr_handle *h, std::vector<int2> &items) {
  items.clear();
  const int blocks = (h->n_inputs + corr::kF32Block - 1) / corr::kF32Block;
  for (int c = 0; c < h->n_chan; ++c)
    for (int I = 0; I < blocks; ++I)
      for (int J = 0; J <= I; ++J) items.push_back(make_int2(c, I | (J << 16)));
  h->n_items_f32 = static_cast<int>(items.size());
  // N_I = 64: (kN64Chan-channel group, time slice) units; as many slices as fill the SMs evenly (cost = rounds x rows per
  // slice, plus 32 rows for the zeroing node and the reduce-adds of a sliced plan)
  h->n64_groups = h->n64_slices = h->n64_slice_len = h->n64_full = 0;
  if (h->n_inputs == 64 && !h->opt_f32_generic) {
    const int T = h->n_time, G = h->n_sms;
    h->n64_groups = (h->n_chan + corr::kN64Chan - 1) / corr::kN64Chan;
    // (A) every group cut into the same number of slices: cost = rounds x rows per slice (+ 32 rows for the zeroing
    // node and the reduce-adds of a sliced plan)
    long long best = -1;
    for (int sl = 1; sl <= 32; ++sl) {
      const int len = ((T + sl - 1) / sl + corr::kN64TB - 1) / corr::kN64TB * corr::kN64TB;
      if ((T + len - 1) / len != sl) continue;
      const long long rounds = (1LL * h->n64_groups * sl + G - 1) / G;
      const long long cost = rounds * len + (sl > 1 ? 32 : 0);
      if (best < 0 || cost < best) { best = cost; h->n64_slices = sl; h->n64_slice_len = len; h->n64_full = 0; }
    }
    // (B) a x G whole groups (a per SM, plain stores, no zeroing) and only the b left-over groups cut into G / b
    // slices: fewer CTAs, and the zeroing node covers the sliced groups' channels only (c5: 148 whole groups + 72
    // groups in halves instead of 220 groups in halves)
    const int a = h->n64_groups / G, b = h->n64_groups % G;
    if (a >= 1 && b > 0) {
      int sl = std::min(32, G / b);
      int len = ((T + sl - 1) / sl + corr::kN64TB - 1) / corr::kN64TB * corr::kN64TB;
      sl = (T + len - 1) / len;
      const long long cost = 1LL * a * T + len + (sl > 1 ? 8 : 0) - 16;  // one CTA start-up per SM less than (A)
      if (sl > 1 && cost < best) { best = cost; h->n64_slices = sl; h->n64_slice_len = len; h->n64_full = a * G; }
    }
  }
  h->f32_threads = blocks == 1 ? 160 : corr::kF32Threads;  // 136 active tiles on a diagonal block
}

int encode_map(corr_handle *h, const void *base, bool turned, int box_rows, CUtensorMap *out) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return fail(CORR_ECUDA, "cuTensorMapEncodeTiled entry point not available");
  const bool packed = h->dtype == CORR_CI4;  // one byte per sample, 64-byte boxes, no swizzle (expanded in smem)
  const cuuint64_t row = static_cast<cuuint64_t>(packed ? 1 : 2) * h->n_inputs;  // bytes per (t, c)
  CUresult r;
  if (!turned) {
    // the handle's channel window of d_in[T][n_chan_total][N]: x runs over the window only (anything past it is
    // out of bounds = zero fill), the time stride is the FULL row, the base is moved to the window's first channel
    const void *win = static_cast<const char *>(base) + static_cast<size_t>(h->chan0) * row;
    cuuint64_t dims[2] = {row * h->n_chan, static_cast<cuuint64_t>(h->n_time)};
    cuuint64_t strides[1] = {row * h->n_chan_total};
    cuuint32_t box[2] = {packed ? 64u : 128u, static_cast<cuuint32_t>(box_rows)};
    cuuint32_t es[2] = {1, 1};
    r = enc(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void *>(win), dims, strides, box, es,
            CU_TENSOR_MAP_INTERLEAVE_NONE, packed ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  } else {
    const cuuint64_t grow = h->pair_mode ? 2 * row : row;
    const cuuint64_t groups = h->pair_mode ? h->n_chan / 2 : h->n_chan;
    cuuint64_t dims[3] = {grow, static_cast<cuuint64_t>(h->n_time), groups};
    cuuint64_t strides[2] = {grow, grow * h->n_time};
    cuuint32_t box[3] = {128, static_cast<cuuint32_t>(box_rows), 1};
    cuuint32_t es[3] = {1, 1, 1};
    r = enc(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void *>(base), dims, strides, box, es,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  if (r != CUDA_SUCCESS) return fail(CORR_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  return CORR_OK;
}

int get_map(corr_handle *h, const void *base, bool turned, const corr::I8Maps **out) {
  for (const MapCacheEntry &e : h->maps)
    if (e.ptr == base) { *out = &e.maps; return CORR_OK; }
  if (h->maps.size() >= 2 * corr::kMaxBatch) h->maps.erase(h->maps.begin());
  MapCacheEntry e;
  e.ptr = base;
  const int rows[3] = {256, 128, 64};
  for (int m = 0; m < 3; ++m) {
    int rc = encode_map(h, base, turned, rows[m], &e.maps.m[m]);
    if (rc != CORR_OK) return rc;
  }
  h->maps.push_back(e);
  *out = &h->maps.back().maps;
  return CORR_OK;
}

// (Re)plans the handle from its shape, window and options; frees / rebuilds the float work-item table.
int replan(corr_handle *h) {
  h->maps.clear();
  h->plan_batch.n_batch = 0;
  if (h->dtype != CORR_CF32) {
    h->pair_mode = (h->n_inputs == 32) ? 1 : 0;
    plan_i8(h, 1, &h->plan);
    return CORR_OK;
  }
  std::vector<int2> items;
  plan_f32(h, items);
  cudaFree(h->d_items_f32);
  h->d_items_f32 = nullptr;
  cudaError_t e = cudaMalloc(&h->d_items_f32, items.size() * sizeof(int2));
  if (e == cudaSuccess) e = cudaMemcpy(h->d_items_f32, items.data(), items.size() * sizeof(int2), cudaMemcpyHostToDevice);
  if (e != cudaSuccess)
    return fail(e == cudaErrorMemoryAllocation ? CORR_EALLOC : CORR_ECUDA, "corr: work-item table: %s", cudaGetErrorString(e));
  return CORR_OK;
}

size_t sample_bytes(int dtype) { return dtype == CORR_CI8 ? 2 : dtype == CORR_CI4 ? 1 : 8; }

}  // namespace

// ============================================================================ C ABI
extern "C" {

const char *corr_last_error(void) { return g_err; }
int corr_last_status(void) { return g_status; }

corr_handle *corr_create(int n_inputs, int n_chan, int n_time, int dtype) {
  g_status = CORR_OK;
  g_err[0] = 0;
  if (n_inputs <= 0 || n_chan <= 0 || n_time <= 0) {
    fail(CORR_EINVAL, "corr_create: n_inputs, n_chan, n_time must be positive (got %d, %d, %d)", n_inputs, n_chan, n_time);
    return nullptr;
  }
  if (dtype != CORR_CI8 && dtype != CORR_CF32 && dtype != CORR_CI4) {
    fail(CORR_EINVAL, "corr_create: unknown dtype %d", dtype);
    return nullptr;
  }
  if (n_inputs % 32 != 0 || n_inputs > 4096) {
    fail(CORR_EUNSUPPORTED, "corr_create: n_inputs must be a multiple of 32 and <= 4096 (got %d)", n_inputs);
    return nullptr;
  }
  if (dtype != CORR_CF32 && n_time > 65535) {
    fail(CORR_EUNSUPPORTED, "corr_create: %s needs n_time <= 65535 so that int32 cannot overflow (got %d)",
         dtype == CORR_CI4 ? "CORR_CI4" : "CORR_CI8", n_time);
    return nullptr;
  }
  if (static_cast<unsigned long long>(n_chan) * n_inputs * 2ull >= (1ull << 31)) {
    fail(CORR_EUNSUPPORTED, "corr_create: n_chan * n_inputs too large");
    return nullptr;
  }
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    fail(CORR_ECUDA, "corr_create: no usable CUDA device (%s)", cudaGetErrorString(cudaGetLastError()));
    return nullptr;
  }
  if (prop.major != 10) {
    fail(CORR_EARCH, "corr_create: device is sm_%d%d; this library is sm_100a only", prop.major, prop.minor);
    return nullptr;
  }
  corr_handle *h = new (std::nothrow) corr_handle();
  if (!h) {
    fail(CORR_EALLOC, "corr_create: host allocation failed");
    return nullptr;
  }
  h->n_inputs = n_inputs;
  h->n_chan = n_chan;
  h->n_time = n_time;
  h->dtype = dtype;
  h->n_chan_total = n_chan;
  h->chan0 = 0;
  h->n_baselines = static_cast<long long>(n_inputs) * (n_inputs + 1) / 2;
  h->in_bytes = static_cast<size_t>(n_time) * n_chan * n_inputs * sample_bytes(dtype);
  h->work_bytes = h->in_bytes;
  h->vis_bytes = static_cast<size_t>(n_chan) * h->n_baselines * 8;
  h->n_sms = prop.multiProcessorCount;
  h->turn_mode = CORR_TURN_FUSED;
  h->probe = 0;
  h->accumulate = 0;
  h->acc_count = 0;
  h->opt_diag_plan = 0; h->opt_pairs = 1; h->opt_wide = 1; h->opt_units = 0; h->opt_f32_generic = 0; h->opt_pdl = 1; h->opt_collect = 1; h->opt_resident = 1; h->opt_mix = 1;
  h->d_items_f32 = nullptr;
  h->d_scratch = nullptr;
  h->d_wide_vis = nullptr;
  h->d_diag_stats = nullptr;
  h->d_stream_in[0] = h->d_stream_in[1] = nullptr;
  h->s_copy = h->s_compute = nullptr;

  // The dynamic shared-memory cap is an attribute of the FUNCTION, not of a handle: it is raised once to the
  // device maximum so that handles with different footprints can be alive (and launched) side by side.
  cudaError_t e = cudaSuccess;
  if (dtype != CORR_CF32) {
    e = cudaFuncSetAttribute(corr::xengine_i8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemI8);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(corr::xengine_i8_batch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemI8);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(corr::xengine_i4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemI8);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(corr::xengine_i8_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmemI8);
  } else {
    e = cudaFuncSetAttribute(corr::xengine_f32_n64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::kN64Smem);
  }
  if (e != cudaSuccess) {
    fail(CORR_ECUDA, "corr_create: %s", cudaGetErrorString(e));
    corr_destroy(h);
    return nullptr;
  }
  if (replan(h) != CORR_OK) {
    corr_destroy(h);
    return nullptr;
  }
  return h;
}

int corr_destroy(corr_handle *h) {
  if (!h) return CORR_OK;
  cudaFree(h->d_items_f32);
  cudaFree(h->d_scratch);
  cudaFree(h->d_wide_vis);
  cudaFree(h->d_diag_stats);
  cudaFree(h->d_stream_in[0]);
  cudaFree(h->d_stream_in[1]);
  if (h->s_copy) cudaStreamDestroy(h->s_copy);
  if (h->s_compute) cudaStreamDestroy(h->s_compute);
  delete h;
  return CORR_OK;
}

size_t corr_in_bytes(const corr_handle *h) { return h ? h->in_bytes : 0; }
size_t corr_vis_bytes(const corr_handle *h) { return h ? h->vis_bytes : 0; }
size_t corr_acc_bytes(const corr_handle *h) { return h ? 2 * h->vis_bytes : 0; }
int corr_launches_per_call(const corr_handle *h) {
  if (!h) return 0;
  return (h->dtype == CORR_CI8 && h->turn_mode == CORR_TURN_STANDALONE) ? 2 : 1;  // kernels; a memset node precedes them when the integration is time-sliced
}

int corr_plan_info(const corr_handle *h, int *info, char *kernel, size_t kernel_len) {
  if (!h || !info) return fail(CORR_EINVAL, "corr_plan_info: NULL argument");
  for (int k = 0; k < CORR_PLAN_INFO_LEN; ++k) info[k] = 0;
  const char *name;
  if (h->dtype == CORR_CF32) {
    const bool n64 = h->n64_groups > 0;
    name = n64 ? "xengine_f32_n64_kernel" : "xengine_f32_kernel";
    info[CORR_PLAN_KERNEL] = n64 ? CORR_KERNEL_F32_N64 : CORR_KERNEL_F32;
    info[CORR_PLAN_GSIZE] = n64 ? corr::kN64Chan : 1;
    info[CORR_PLAN_SLICES] = n64 ? h->n64_slices : 1;
    info[CORR_PLAN_GRID] = n64 ? h->n64_full + (h->n64_groups - h->n64_full) * h->n64_slices : h->n_items_f32;
    info[CORR_PLAN_MIXED] = n64 && h->n64_full > 0 && h->n64_full < h->n64_groups;
  } else {
    const corr::I8Params &ip = h->plan.ip;
    const bool i4 = h->dtype == CORR_CI4;
    name = i4 ? "xengine_i4_kernel" : ip.pair2 ? "xengine_i8_pair_kernel" : "xengine_i8_kernel";
    info[CORR_PLAN_KERNEL] = i4 ? CORR_KERNEL_I4 : ip.pair2 ? (ip.resident ? CORR_KERNEL_I8_PAIR_RESIDENT : CORR_KERNEL_I8_PAIR) : CORR_KERNEL_I8;
    info[CORR_PLAN_GSIZE] = ip.diag ? ip.gsize : 0;
    info[CORR_PLAN_SLICES] = ip.mix_cut > 0 ? ip.mix_len ? (h->n_time + ip.mix_len - 1) / ip.mix_len : 1 : ip.n_slices;
    info[CORR_PLAN_GRID] = h->plan.grid;
    info[CORR_PLAN_MIXED] = ip.mix_cut > 0;
    info[CORR_PLAN_STAGES] = ip.stages;
    bool wide = false;
    if (ip.pair2 && !ip.resident)
      for (int k = 0; k < ip.n_kinds; ++k) wide = wide || ((ip.kinds[k] >> 11) & 1);
    info[CORR_PLAN_WIDE] = wide;
    info[CORR_PLAN_SMEM] = static_cast<int>(h->plan.smem);
  }
  if (kernel && kernel_len) snprintf(kernel, kernel_len, "%s", name);
  return CORR_OK;
}

int corr_set_option(corr_handle *h, int key, int value) {
  if (!h) return fail(CORR_EINVAL, "corr_set_option: NULL handle");
  switch (key) {
    case CORR_OPT_DIAG_PLAN: {
      const int g = value >> 8, sl = value & 255;
      if (value != 0 && !((g == 1 || g == 2 || g == 4) && sl >= 0 && sl <= 64))
        return fail(CORR_EINVAL, "corr_set_option: CORR_OPT_DIAG_PLAN wants 256 * gsize (1, 2, 4) + slices (1..64), got %d", value);
      h->opt_diag_plan = value;
      break;
    }
    case CORR_OPT_PAIRS: h->opt_pairs = value < 0 ? 0 : (value > 2 ? 2 : value); break;
    case CORR_OPT_WIDE: h->opt_wide = value < 0 ? 0 : (value > 2 ? 2 : value); break;
    case CORR_OPT_COLLECT: h->opt_collect = value ? 1 : 0; break;
    case CORR_OPT_RESIDENT: h->opt_resident = value < 0 ? 0 : (value > 2 ? 2 : value); break;
    case CORR_OPT_MIX: h->opt_mix = value ? 1 : 0; break;
    case CORR_OPT_UNITS:
      if (value < 0) return fail(CORR_EINVAL, "corr_set_option: CORR_OPT_UNITS must be >= 0");
      h->opt_units = value;
      break;
    case CORR_OPT_F32_GENERIC: h->opt_f32_generic = value ? 1 : 0; break;
    case CORR_OPT_PDL: h->opt_pdl = value < 0 ? 0 : (value > 2 ? 2 : value); break;
    default: return fail(CORR_EINVAL, "corr_set_option: unknown key %d", key);
  }
  return replan(h);
}

int corr_set_chan_window(corr_handle *h, int n_chan_total, int chan0) {
  if (!h) return fail(CORR_EINVAL, "corr_set_chan_window: NULL handle");
  if (chan0 < 0 || n_chan_total < 1 || static_cast<long long>(chan0) + h->n_chan > n_chan_total)
    return fail(CORR_EINVAL, "corr_set_chan_window: window %d..%d does not fit %d channels", chan0, chan0 + h->n_chan - 1, n_chan_total);
  if (static_cast<unsigned long long>(n_chan_total) * h->n_inputs * 2ull >= (1ull << 31))
    return fail(CORR_EUNSUPPORTED, "corr_set_chan_window: n_chan_total * n_inputs too large");
  h->n_chan_total = n_chan_total;
  h->chan0 = chan0;
  h->in_bytes = static_cast<size_t>(h->n_time) * n_chan_total * h->n_inputs * sample_bytes(h->dtype);
  h->maps.clear();  // the tensor maps carry the window
  for (int b = 0; b < 2; ++b) {  // streaming buffers are sized for the full buffer
    cudaFree(h->d_stream_in[b]);
    h->d_stream_in[b] = nullptr;
  }
  return CORR_OK;
}

#ifdef CORR_DIAG
int corr_probe_mma(int m, int n, int mn_major, int iters, double *out) {
  const int fill = mn_major >> 1;  // bit 1 of mn_major: pseudo-random operand bytes; bits 2,3: A == B, wide smem walk
  mn_major &= 1;
  if ((m != 64 && m != 128) || n < 16 || n > 256 || (n % 16) || iters < 16 || !out)
    return fail(CORR_EINVAL, "corr_probe_mma: bad argument");
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  unsigned long long *d_cyc = nullptr;
  CUDA_TRY(cudaMalloc(&d_cyc, 2 * sms * sizeof(unsigned long long)));
  corr::ProbeParams pp{iters, m, n, fill, mn_major, d_cyc};
  const int smem = 225 * 1024;
  CUDA_TRY(cudaFuncSetAttribute(corr::probe_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  corr::probe_mma_kernel<<<sms, 128, smem>>>(pp);  // warm-up
  cudaEventRecord(e0);
  corr::probe_mma_kernel<<<sms, 128, smem>>>(pp);
  cudaEventRecord(e1);
  cudaError_t e = cudaDeviceSynchronize();
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  std::vector<unsigned long long> cyc(2 * sms);
  cudaMemcpy(cyc.data(), d_cyc, 2 * sms * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
  cudaFree(d_cyc);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess) return fail(CORR_ECUDA, "corr_probe_mma: %s", cudaGetErrorString(e));
  double mean = 0, ns = 0;
  for (int b = 0; b < sms; ++b) { mean += static_cast<double>(cyc[2 * b]); ns += static_cast<double>(cyc[2 * b + 1]); }
  mean /= sms;
  ns /= sms;
  out[0] = ms;
  out[1] = mean / iters;
  out[2] = 2.0 * m * n * 32.0 * iters * sms / (ns * 1e-9) / 1e12;  // over the issue loop itself
  out[3] = mean / ns * 1e3;                                        // effective SM MHz during the loop
  return CORR_OK;
}

int corr_probe_ffma(int packed, int iters, double *out) {
  if (iters < 16 || !out) return fail(CORR_EINVAL, "corr_probe_ffma: bad argument");
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms, threads = 1024, smem = 200 * 1024;  // one CTA per SM, all resident at once
  CUDA_TRY(cudaFuncSetAttribute(corr::probe_ffma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  unsigned long long *d_cyc = nullptr;
  float *d_sink = nullptr;
  CUDA_TRY(cudaMalloc(&d_cyc, 2 * blocks * sizeof(unsigned long long)));
  if (cudaMalloc(&d_sink, static_cast<size_t>(blocks) * threads * sizeof(float)) != cudaSuccess) {
    cudaFree(d_cyc);
    return fail(CORR_EALLOC, "corr_probe_ffma: %s", cudaGetErrorString(cudaGetLastError()));
  }
  corr::ProbeFfmaParams pp{iters, packed ? 1 : 0, 0.999999f, 1e-7f, d_sink, d_cyc};
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  corr::probe_ffma_kernel<<<blocks, threads, smem>>>(pp);  // warm-up
  cudaEventRecord(e0);
  corr::probe_ffma_kernel<<<blocks, threads, smem>>>(pp);
  cudaEventRecord(e1);
  cudaError_t e = cudaDeviceSynchronize();
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  std::vector<unsigned long long> cyc(2 * blocks);
  cudaMemcpy(cyc.data(), d_cyc, 2 * blocks * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
  cudaFree(d_cyc);
  cudaFree(d_sink);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess) return fail(CORR_ECUDA, "corr_probe_ffma: %s", cudaGetErrorString(e));
  double mean = 0, ns = 0, ns_max = 0;
  for (int b = 0; b < blocks; ++b) {
    mean += static_cast<double>(cyc[2 * b]);
    ns += static_cast<double>(cyc[2 * b + 1]);
    ns_max = std::max(ns_max, static_cast<double>(cyc[2 * b + 1]));
  }
  mean /= blocks;
  ns /= blocks;
  out[0] = ms;
  out[1] = 2.0 * 16.0 * iters * static_cast<double>(blocks) * threads / (ns_max * 1e-9) / 1e12;  // the slowest SM's loop
  out[2] = mean / ns * 1e3;
  return CORR_OK;
}

int corr_set_probe(corr_handle *h, int mode) {
  if (!h) return fail(CORR_EINVAL, "corr_set_probe: NULL handle");
  h->probe = mode;
  if ((mode & ~128) && h->dtype != CORR_CF32 && h->plan.ip.resident) {
    // the engine switches live in the streaming producers / issuer only: fall back to the streaming pair plan
    h->opt_resident = 0;
    if (int rc = replan(h)) return rc;
  }
  if ((mode & 128) && !h->d_diag_stats) {
    CUDA_TRY(cudaMalloc(&h->d_diag_stats, 4 * 256 * sizeof(unsigned long long)));
    CUDA_TRY(cudaMemset(h->d_diag_stats, 0, 4 * 256 * sizeof(unsigned long long)));
  }
  return CORR_OK;
}

int corr_probe_stats(corr_handle *h, double *out) {
  if (!h || !out || !h->d_diag_stats) return fail(CORR_EINVAL, "corr_probe_stats: no statistics (corr_set_probe(h, 128) first)");
  const int units = h->plan.ip.units;
  std::vector<unsigned long long> st(4 * 256);
  CUDA_TRY(cudaMemcpy(st.data(), h->d_diag_stats, st.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
  for (int k = 0; k < 4; ++k) out[k] = 0.0;
  for (int u = 0; u < units; ++u)
    for (int k = 0; k < 4; ++k) out[k] += static_cast<double>(st[4 * u + k]) / units;
  return CORR_OK;
}
#endif  // CORR_DIAG

int corr_set_accumulate(corr_handle *h, int on) {
  if (!h) return fail(CORR_EINVAL, "corr_set_accumulate: NULL handle");
  h->accumulate = on ? 1 : 0;
  h->acc_count = 0;
  return CORR_OK;
}
long long corr_accumulate_count(const corr_handle *h) { return h ? h->acc_count : 0; }

static int launch_normalize(corr_handle *h, const void *d_sums, double count, void *d_out, void *stream, int kind, const char *who) {
  if (!h || !d_sums || !d_out) return fail(CORR_EINVAL, "%s: NULL argument", who);
  if (!(count > 0)) return fail(CORR_EINVAL, "%s: count must be positive", who);
  if ((reinterpret_cast<uintptr_t>(d_sums) | reinterpret_cast<uintptr_t>(d_out)) & 15)
    return fail(CORR_EINVAL, "%s: pointers must be 16-byte aligned", who);
  corr::NormParams np;
  np.vis = d_sums;
  np.out = static_cast<float *>(d_out);
  np.n = static_cast<long long>(h->vis_bytes / 4);
  np.inv_count = static_cast<float>(1.0 / count);
  np.inv_count_d = 1.0 / count;
  np.kind = kind;
  if (np.n % 4) return fail(CORR_EUNSUPPORTED, "%s: odd number of visibilities", who);
  const int blocks = static_cast<int>(std::min<long long>((np.n / 4 + 255) / 256, static_cast<long long>(h->n_sms) * 8));
  corr::normalize_kernel<<<blocks, 256, 0, static_cast<cudaStream_t>(stream)>>>(np);
  CUDA_TRY(cudaGetLastError());
  return CORR_OK;
}

int corr_normalize(corr_handle *h, const void *d_vis, double count, void *d_out, void *stream) {
  return launch_normalize(h, d_vis, count, d_out, stream, (h && h->dtype == CORR_CF32) ? corr::kSumF32 : corr::kSumI32, "corr_normalize");
}

int corr_normalize_wide(corr_handle *h, const void *d_acc, double count, void *d_out, void *stream) {
  if (d_acc && d_acc == d_out) return fail(CORR_EINVAL, "corr_normalize_wide: d_acc and d_out alias");
  return launch_normalize(h, d_acc, count, d_out, stream, (h && h->dtype == CORR_CF32) ? corr::kSumF64 : corr::kSumI64, "corr_normalize_wide");
}

static int xengine_impl(corr_handle *h, const void *d_in, void *d_vis, void *stream, const int accumulate);

int corr_accumulate_wide(corr_handle *h, const void *d_in, void *d_acc, void *stream) {
  if (!h || !d_in || !d_acc) return fail(CORR_EINVAL, "corr_accumulate_wide: NULL argument");
  if (reinterpret_cast<uintptr_t>(d_acc) & 15) return fail(CORR_EINVAL, "corr_accumulate_wide: d_acc must be 16-byte aligned");
  if (!h->d_wide_vis) {
    cudaError_t e = cudaMalloc(&h->d_wide_vis, h->vis_bytes);
    if (e != cudaSuccess) return fail(CORR_EALLOC, "corr_accumulate_wide: batch buffer of %zu bytes: %s", h->vis_bytes, cudaGetErrorString(e));
  }
  // the batch itself is an ordinary overwriting integration (int32 / float sums of T samples cannot overflow)
  const int rc = xengine_impl(h, d_in, h->d_wide_vis, stream, 0);
  if (rc != CORR_OK) return rc;
  corr::FoldParams fp;
  fp.vis = h->d_wide_vis;
  fp.acc = d_acc;
  fp.n = static_cast<long long>(h->vis_bytes / 4);
  fp.is_int = h->dtype != CORR_CF32;
  if (fp.n % 4) return fail(CORR_EUNSUPPORTED, "corr_accumulate_wide: odd number of visibilities");
  const int blocks = static_cast<int>(std::min<long long>((fp.n / 4 + 255) / 256, static_cast<long long>(h->n_sms) * 8));
  corr::fold_wide_kernel<<<blocks, 256, 0, static_cast<cudaStream_t>(stream)>>>(fp);
  CUDA_TRY(cudaGetLastError());
  return CORR_OK;
}

// Device address of g_static_batch on the CURRENT device, looked up once per device (each device that loads the
// module has its own copy of the array at its own address).  Host-only bookkeeping; no device memory is allocated.
static int static_batch_ptr(void **out) {
  enum { kMaxDevices = 64 };
  static void *ptr[kMaxDevices] = {};
  static std::mutex mu;
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(CORR_EUNSUPPORTED, "corr_accumulate_wide_static: device ordinal %d not supported", dev);
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[dev]) {
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_batch);
    if (e != cudaSuccess || !p)
      return fail(CORR_ECUDA, "corr_accumulate_wide_static: address of the static batch buffer on device %d: %s", dev,
                  cudaGetErrorString(e));
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return CORR_OK;
}

// corr_accumulate_wide with the batch staged in g_static_batch instead of a handle-owned cudaMalloc'ed buffer: for
// callers that cannot allocate (see include/corr.h for who they are, the size limit and the sharing rules).
int corr_accumulate_wide_static(corr_handle *h, const void *d_in, void *d_acc, void *stream) {
  if (!h || !d_in || !d_acc) return fail(CORR_EINVAL, "corr_accumulate_wide_static: NULL argument");
  if (reinterpret_cast<uintptr_t>(d_acc) & 15) return fail(CORR_EINVAL, "corr_accumulate_wide_static: d_acc must be 16-byte aligned");
  if (h->vis_bytes > static_cast<size_t>(CORR_STATIC_BATCH_BYTES))
    return fail(CORR_EUNSUPPORTED,
                "corr_accumulate_wide_static: one batch of visibilities is %zu bytes, the static buffer holds %u "
                "(CORR_STATIC_BATCH_BYTES); use corr_accumulate_wide, which allocates its buffer",
                h->vis_bytes, static_cast<unsigned>(CORR_STATIC_BATCH_BYTES));
  if ((h->vis_bytes / 4) % 4) return fail(CORR_EUNSUPPORTED, "corr_accumulate_wide_static: odd number of visibilities");
  void *d_batch = nullptr;
  if (int rc = static_batch_ptr(&d_batch)) return rc;
  // the batch is an ordinary overwriting integration: every element of the region used is written (sliced plans
  // memset theirs on `stream` first), so the previous call's contents never reach the fold
  const int rc = xengine_impl(h, d_in, d_batch, stream, 0);
  if (rc != CORR_OK) return rc;
  const long long n = static_cast<long long>(h->vis_bytes / 4);
  const int blocks = static_cast<int>(std::min<long long>((n / 4 + 255) / 256, static_cast<long long>(h->n_sms) * 8));
  fold_wide_static_kernel<<<blocks, 256, 0, static_cast<cudaStream_t>(stream)>>>(d_acc, n, h->dtype != CORR_CF32);
  CUDA_TRY(cudaGetLastError());
  return CORR_OK;
}

int corr_set_turn(corr_handle *h, int mode) {
  if (!h) return fail(CORR_EINVAL, "corr_set_turn: NULL handle");
  if (h->dtype != CORR_CI8) return fail(CORR_EUNSUPPORTED, "corr_set_turn: only the CI8 path has two corner-turn realisations");
  if (mode != CORR_TURN_FUSED && mode != CORR_TURN_STANDALONE) return fail(CORR_EINVAL, "corr_set_turn: unknown mode %d", mode);
  if (mode == CORR_TURN_STANDALONE) {
    if (h->pair_mode && (h->n_chan & 1))
      return fail(CORR_EUNSUPPORTED, "corr_set_turn: standalone turn with n_inputs == 32 needs an even n_chan");
    if (!h->d_scratch) {
      const size_t bytes = static_cast<size_t>(h->n_time) * h->n_chan * h->n_inputs * 2;
      cudaError_t e = cudaMalloc(&h->d_scratch, bytes);
      if (e != cudaSuccess) return fail(CORR_EALLOC, "corr_set_turn: scratch of %zu bytes: %s", bytes, cudaGetErrorString(e));
    }
  }
  h->turn_mode = mode;
  return replan(h);  // the resident-A plan reads d_in through 2-D maps only: the standalone turn takes the streaming plan
}

static int launch_turn(corr_handle *h, const void *d_in, void *d_out, cudaStream_t st) {
  corr::TurnParams tp;
  const size_t w = static_cast<size_t>(h->n_inputs) * (h->dtype == CORR_CI8 ? 2 : 8);
  const bool pair = (h->dtype == CORR_CI8) && h->pair_mode;
  const size_t wg = pair ? 2 * w : w;
  tp.in = static_cast<const uint4 *>(d_in);
  tp.out = static_cast<uint4 *>(d_out);
  tp.n_time = h->n_time;
  tp.n_groups = pair ? h->n_chan / 2 : h->n_chan;
  tp.wc = static_cast<int>(wg / 16);
  tp.in_row_chunks = static_cast<long long>(h->n_chan_total) * static_cast<long long>(w / 16);
  tp.in_off_chunks = static_cast<long long>(h->chan0) * static_cast<long long>(w / 16);
  const int max_rows = static_cast<int>(corr::kTurnTileBytes / wg);  // (t, g) rows per tile
  if (max_rows < 1) return fail(CORR_EUNSUPPORTED, "corr_corner_turn: row of %zu bytes exceeds the tile", wg);
  tp.tt = std::min(std::min(32, max_rows), h->n_time);
  tp.gg = std::max(1, std::min(max_rows / tp.tt, tp.n_groups));
  tp.g_tiles = (tp.n_groups + tp.gg - 1) / tp.gg;
  const long long tiles = static_cast<long long>(tp.g_tiles) * ((tp.n_time + tp.tt - 1) / tp.tt);
  if (tiles > 0x7fffffffLL) return fail(CORR_EUNSUPPORTED, "corr_corner_turn: %lld tiles exceed the grid limit", tiles);
  corr::corner_turn_kernel<<<static_cast<unsigned>(tiles), corr::kTurnThreads, 0, st>>>(tp);
  CUDA_TRY(cudaGetLastError());
  return CORR_OK;
}

int corr_corner_turn(corr_handle *h, const void *d_in, void *d_out, void *stream) {
  if (!h || !d_in || !d_out) return fail(CORR_EINVAL, "corr_corner_turn: NULL argument");
  if ((reinterpret_cast<uintptr_t>(d_in) | reinterpret_cast<uintptr_t>(d_out)) & 15)
    return fail(CORR_EINVAL, "corr_corner_turn: pointers must be 16-byte aligned");
  if (d_in == d_out) return fail(CORR_EINVAL, "corr_corner_turn: d_in and d_out alias");
  if (h->dtype == CORR_CI4) return fail(CORR_EUNSUPPORTED, "corr_corner_turn: not provided for the 4-bit packed input");
  if (h->dtype == CORR_CI8 && h->pair_mode && (h->n_chan & 1))
    return fail(CORR_EUNSUPPORTED, "corr_corner_turn: n_inputs == 32 needs an even n_chan");
  return launch_turn(h, d_in, d_out, static_cast<cudaStream_t>(stream));
}

// accumulate mode on int32 accumulators: refuse the batch that could overflow them for some input (reading R6)
static int accumulate_guard(corr_handle *h, long long batches) {
  if (!h->accumulate || h->dtype == CORR_CF32) return CORR_OK;
  const long long per_sample = h->dtype == CORR_CI4 ? 2LL * 8 * 8 : 2LL * 128 * 128;
  if ((h->acc_count + batches) * h->n_time * per_sample >= (1LL << 31))
    return fail(CORR_EUNSUPPORTED,
                "corr_xengine: accumulate mode: batch %lld of T = %d samples could overflow the int32 accumulators "
                "(count * T * %lld >= 2^31); read out and restart, or use corr_accumulate_wide",
                h->acc_count + batches, h->n_time, per_sample);
  return CORR_OK;
}

// One integration; `accumulate` != 0 adds into d_vis (accumulate mode) instead of overwriting.  The flag is an argument so
// that callers which need an overwriting integration (the wide accumulators' batch) do not have to flip the handle's state.
static int xengine_impl(corr_handle *h, const void *d_in, void *d_vis, void *stream, const int accumulate) {
  if (!h) return fail(CORR_EINVAL, "corr_xengine: NULL handle");
  if (!d_in || !d_vis) return fail(CORR_EINVAL, "corr_xengine: NULL device pointer");
  if ((reinterpret_cast<uintptr_t>(d_in) | reinterpret_cast<uintptr_t>(d_vis)) & 15)
    return fail(CORR_EINVAL, "corr_xengine: d_in and d_vis must be 16-byte aligned");
  if (d_in == d_vis) return fail(CORR_EINVAL, "corr_xengine: d_in and d_vis alias");
  if (accumulate)
    if (int rc = accumulate_guard(h, 1)) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (h->dtype == CORR_CF32) {
    if (h->n64_groups > 0) {
      corr::F32N64Params np;
      np.in = static_cast<const float2 *>(d_in);
      np.vis = static_cast<float2 *>(d_vis);
      np.n_time = h->n_time; np.n_chan = h->n_chan;
      np.n_chan_total = h->n_chan_total; np.chan0 = h->chan0;
      np.n_groups = h->n64_groups; np.n_slices = h->n64_slices; np.slice_len = h->n64_slice_len;
      np.n_full = h->n64_full;
      np.add = accumulate ? 1 : 0;
      if (h->n64_slices > 1 && !accumulate) {  // the sliced groups' channels are zeroed: their slices reduce-add
        const size_t chan0 = static_cast<size_t>(h->n64_full) * corr::kN64Chan;
        const size_t off = chan0 * h->n_baselines * 8;
        CUDA_TRY(cudaMemsetAsync(static_cast<char *>(d_vis) + off, 0, h->vis_bytes - off, st));
      }
      const int units = h->n64_full + (h->n64_groups - h->n64_full) * h->n64_slices;
      corr::xengine_f32_n64_kernel<<<units, corr::kN64Threads, corr::kN64Smem, st>>>(np);
      CUDA_TRY(cudaGetLastError());
      if (accumulate) ++h->acc_count;
      return CORR_OK;
    }
    corr::F32Params fp;
    fp.in = static_cast<const float2 *>(d_in);
    fp.vis = static_cast<float2 *>(d_vis);
    fp.items = h->d_items_f32;
    fp.n_items = h->n_items_f32;
    fp.n_time = h->n_time;
    fp.n_chan = h->n_chan;
    fp.n_inputs = h->n_inputs;
    fp.n_chan_total = h->n_chan_total;
    fp.chan0 = h->chan0;
    fp.n_baselines = h->n_baselines;
    fp.accumulate = accumulate;
    corr::xengine_f32_kernel<<<h->n_items_f32, h->f32_threads, 0, st>>>(fp);
    CUDA_TRY(cudaGetLastError());
    if (accumulate) ++h->acc_count;
    return CORR_OK;
  }
  const bool turned = h->turn_mode == CORR_TURN_STANDALONE;
  const void *src = d_in;
  if (turned) {
    int rc = launch_turn(h, d_in, h->d_scratch, st);
    if (rc != CORR_OK) return rc;
    src = h->d_scratch;
  }
  const corr::I8Maps *maps = nullptr;
  int rc = get_map(h, src, turned, &maps);
  if (rc != CORR_OK) return rc;
  corr::I8Params ip = h->plan.ip;
  const int grid = h->plan.grid;
  const size_t smem = h->plan.smem;
  ip.turned = turned ? 1 : 0;
  ip.vis = static_cast<int2 *>(d_vis);
  ip.probe = h->probe;
  ip.diag_stats = h->d_diag_stats;
  ip.out_shift = h->dtype == CORR_CI4 ? 8 : 0;
  ip.accumulate = accumulate;
  ip.collect = h->opt_collect;
  if (h->plan.zero_vis && !accumulate) {  // slices accumulate with red.add
    const size_t off = static_cast<size_t>(std::min(h->plan.zero_from_chan, h->n_chan)) * h->n_baselines * 8;
    CUDA_TRY(cudaMemsetAsync(static_cast<char *>(d_vis) + off, 0, h->vis_bytes - off, st));
  }
  if (h->dtype == CORR_CI4) corr::xengine_i4_kernel<<<grid, corr::kI4Threads, smem, st>>>(*maps, ip);
  else if (ip.pair2) corr::xengine_i8_pair_kernel<<<grid, corr::kI8Threads, smem, st>>>(*maps, ip);
  else {
    // programmatic dependent launch: the kernel may start while the preceding kernel of the stream drains (it waits with
    // griddepcontrol.wait before its first global-memory access); worth ~1 us per call on launch-bound inputs (c1: 7.5 ->
    // 6.2 us in a replayed graph).  For small inputs only while the stream is being captured into a CUDA graph: launched
    // call by call the attribute costs more host time per launch than it saves on the device; inputs above 64 MB run long
    // enough to hide that (c2: 160.7 -> 158.6 us call by call).
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (h->opt_pdl && cudaStreamIsCapturing(st, &cap) != cudaSuccess) { cap = cudaStreamCaptureStatusNone; (void)cudaGetLastError(); }
    if (h->opt_pdl == 2 || (h->opt_pdl && (cap == cudaStreamCaptureStatusActive || h->work_bytes > (64u << 20)))) {
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(grid); cfg.blockDim = dim3(corr::kI8Threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      attr[0].val.programmaticStreamSerializationAllowed = 1;
      cfg.attrs = attr; cfg.numAttrs = 1;
      CUDA_TRY(cudaLaunchKernelEx(&cfg, corr::xengine_i8_kernel, *maps, ip));
    } else {
      corr::xengine_i8_kernel<<<grid, corr::kI8Threads, smem, st>>>(*maps, ip);
    }
  }
  CUDA_TRY(cudaGetLastError());
  if (accumulate) ++h->acc_count;
  return CORR_OK;
}

int corr_xengine(corr_handle *h, const void *d_in, void *d_vis, void *stream) {
  if (!h) return fail(CORR_EINVAL, "corr_xengine: NULL handle");
  return xengine_impl(h, d_in, d_vis, stream, h->accumulate);
}

int corr_xengine_batch(corr_handle *h, const void *const *d_in, void *const *d_vis, int n, void *stream) {
  if (!h) return fail(CORR_EINVAL, "corr_xengine_batch: NULL handle");
  if (!d_in || !d_vis || n < 1) return fail(CORR_EINVAL, "corr_xengine_batch: NULL pointer array or n < 1");
  for (int k = 0; k < n; ++k) {
    if (!d_in[k] || !d_vis[k]) return fail(CORR_EINVAL, "corr_xengine_batch: NULL device pointer at index %d", k);
    if ((reinterpret_cast<uintptr_t>(d_in[k]) | reinterpret_cast<uintptr_t>(d_vis[k])) & 15)
      return fail(CORR_EINVAL, "corr_xengine_batch: d_in[%d] and d_vis[%d] must be 16-byte aligned", k, k);
    if (d_in[k] == d_vis[k]) return fail(CORR_EINVAL, "corr_xengine_batch: d_in[%d] and d_vis[%d] alias", k, k);
  }
  // No output may overlap an input of the batch (any entry's), and outputs may not overlap one another: in the single
  // launch all integrations run concurrently.  Sorted by start address, an interval overlaps an earlier one iff it starts
  // before that one ends.  Accumulate mode runs call by call on `stream`, where several entries adding into one d_vis is
  // well defined, so only there outputs may repeat.  Inputs may repeat freely (they are only read).
  if (n > 1) {
    struct Range { uintptr_t lo, hi; int is_vis, k; };
    std::vector<Range> r;
    r.reserve(2 * static_cast<size_t>(n));
    for (int k = 0; k < n; ++k) {
      const uintptr_t a = reinterpret_cast<uintptr_t>(d_in[k]), v = reinterpret_cast<uintptr_t>(d_vis[k]);
      r.push_back({a, a + h->in_bytes, 0, k});
      r.push_back({v, v + h->vis_bytes, 1, k});
    }
    std::sort(r.begin(), r.end(), [](const Range &x, const Range &y) { return x.lo < y.lo; });
    uintptr_t end_vis = 0, end_in = 0;
    int k_vis = -1, k_in = -1;
    for (const Range &x : r) {
      if (x.lo < end_vis && (!x.is_vis || !h->accumulate))
        return fail(CORR_EINVAL, "corr_xengine_batch: %s[%d] overlaps d_vis[%d]", x.is_vis ? "d_vis" : "d_in", x.k, k_vis);
      if (x.is_vis && x.lo < end_in)
        return fail(CORR_EINVAL, "corr_xengine_batch: d_vis[%d] overlaps d_in[%d]", x.k, k_in);
      if (x.is_vis) { if (x.hi > end_vis) { end_vis = x.hi; k_vis = x.k; } }
      else if (x.hi > end_in) { end_in = x.hi; k_in = x.k; }
    }
  }
  // single-launch path: CI8 on single CTAs, fused corner turn, overwrite semantics; everything else = n ordinary calls
  const bool one_launch = h->dtype == CORR_CI8 && !h->plan.ip.pair2 && h->turn_mode == CORR_TURN_FUSED && !h->accumulate && n > 1;
  if (!one_launch) {
    for (int k = 0; k < n; ++k)
      if (int rc = corr_xengine(h, d_in[k], d_vis[k], stream)) return rc;
    return CORR_OK;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  for (int k0 = 0; k0 < n; k0 += corr::kMaxBatch) {
    const int nb = std::min(corr::kMaxBatch, n - k0);
    if (nb == 1) {
      if (int rc = corr_xengine(h, d_in[k0], d_vis[k0], stream)) return rc;
      continue;
    }
    if (h->plan_batch.n_batch != nb) plan_i8(h, nb, &h->plan_batch);
    corr::I8Params ip = h->plan_batch.ip;
    static thread_local corr::I8Batch bt;  // 25 KB of kernel parameters, copied at launch
    for (int k = 0; k < nb; ++k) {
      const corr::I8Maps *maps = nullptr;
      if (int rc = get_map(h, d_in[k0 + k], false, &maps)) return rc;
      for (int m = 0; m < 3; ++m) bt.m[k][m] = maps->m[m];
      bt.vis[k] = static_cast<int2 *>(d_vis[k0 + k]);
      if (h->plan_batch.zero_vis) CUDA_TRY(cudaMemsetAsync(d_vis[k0 + k], 0, h->vis_bytes, st));
    }
    ip.turned = 0;
    ip.vis = nullptr;
    ip.probe = 0;
    ip.out_shift = 0;
    ip.accumulate = 0;
    corr::xengine_i8_batch_kernel<<<h->plan_batch.grid, corr::kI8Threads, h->plan_batch.smem, st>>>(bt, ip);
    CUDA_TRY(cudaGetLastError());
  }
  return CORR_OK;
}

static int stream_run_impl(corr_handle *h, corr_fstage *f, const void *const *h_in, int n_integrations, void *d_vis,
                           double *stats);

int corr_stream_run(corr_handle *h, const void *const *h_in, int n_integrations, void *d_vis, double *stats) {
  return stream_run_impl(h, nullptr, h_in, n_integrations, d_vis, stats);
}

int corr_stream_run_fx(corr_handle *h, corr_fstage *f, const void *const *h_raw, int n_integrations, void *d_vis,
                       double *stats) {
  if (!f) return fail(CORR_EINVAL, "corr_stream_run_fx: NULL F-stage handle");
  if (!h || h->dtype != CORR_CF32 || h->in_bytes != f->out_bytes || h->n_inputs != f->n_inputs)
    return fail(CORR_EINVAL, "corr_stream_run_fx: the X-engine handle must be CORR_CF32 with n_time * n_chan = n_batch * n_fft");
  return stream_run_impl(h, f, h_raw, n_integrations, d_vis, stats);
}

static int stream_run_impl(corr_handle *h, corr_fstage *f, const void *const *h_in, int n_integrations, void *d_vis,
                           double *stats) {
  if (!h || !h_in || !d_vis || n_integrations <= 0) return fail(CORR_EINVAL, "corr_stream_run: bad argument");
  for (int k = 0; k < n_integrations; ++k)
    if (!h_in[k]) return fail(CORR_EINVAL, "corr_stream_run: h_in[%d] is NULL", k);
  if (!h->s_copy) CUDA_TRY(cudaStreamCreateWithFlags(&h->s_copy, cudaStreamNonBlocking));
  if (!h->s_compute) CUDA_TRY(cudaStreamCreateWithFlags(&h->s_compute, cudaStreamNonBlocking));
  const size_t copy_bytes = f ? f->in_bytes : h->in_bytes;
  void **d_buf = f ? f->d_raw : h->d_stream_in;
  for (int b = 0; b < 2; ++b)
    if (!d_buf[b]) {
      cudaError_t e = cudaMalloc(&d_buf[b], copy_bytes);
      if (e != cudaSuccess) return fail(CORR_EALLOC, "corr_stream_run: input buffer of %zu bytes: %s", copy_bytes, cudaGetErrorString(e));
    }
  if (f && !f->d_spec) {
    cudaError_t e = cudaMalloc(&f->d_spec, f->out_bytes);
    if (e != cudaSuccess) return fail(CORR_EALLOC, "corr_stream_run_fx: spectra buffer of %zu bytes: %s", f->out_bytes, cudaGetErrorString(e));
  }
  const int n = n_integrations;
  std::vector<cudaEvent_t> ev(4 * n, nullptr);  // per integration: copy start, copy end, kernel start, kernel end
  for (cudaEvent_t &e : ev)
    if (cudaEventCreate(&e) != cudaSuccess) {
      for (cudaEvent_t &d : ev)
        if (d) cudaEventDestroy(d);
      return fail(CORR_ECUDA, "corr_stream_run: cudaEventCreate: %s", cudaGetErrorString(cudaGetLastError()));
    }
  int rc = CORR_OK;
  const auto w0 = std::chrono::steady_clock::now();
  for (int k = 0; k < n && rc == CORR_OK; ++k) {
    const int b = k & 1;
    // buffer b is free once the kernel of integration k-2 has finished reading it
    if (k >= 2) cudaStreamWaitEvent(h->s_copy, ev[4 * (k - 2) + 3], 0);
    cudaEventRecord(ev[4 * k + 0], h->s_copy);
    cudaMemcpyAsync(d_buf[b], h_in[k], copy_bytes, cudaMemcpyHostToDevice, h->s_copy);
    cudaEventRecord(ev[4 * k + 1], h->s_copy);
    cudaStreamWaitEvent(h->s_compute, ev[4 * k + 1], 0);
    cudaEventRecord(ev[4 * k + 2], h->s_compute);
    const void *x_in = d_buf[b];
    if (f) {  // raw voltages -> spectra (one buffer: F and X of integration k are ordered on the compute stream)
      rc = corr_fstage_run(f, d_buf[b], f->d_spec, h->s_compute);
      x_in = f->d_spec;
    }
    if (rc == CORR_OK)
      rc = corr_xengine(h, x_in, static_cast<char *>(d_vis) + static_cast<size_t>(k) * h->vis_bytes, h->s_compute);
    cudaEventRecord(ev[4 * k + 3], h->s_compute);
  }
  cudaError_t e1 = cudaStreamSynchronize(h->s_copy);
  cudaError_t e2 = cudaStreamSynchronize(h->s_compute);
  const auto w1 = std::chrono::steady_clock::now();
  if (rc == CORR_OK && (e1 != cudaSuccess || e2 != cudaSuccess))
    rc = fail(CORR_ECUDA, "corr_stream_run: %s", cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
  if (rc == CORR_OK && stats) {
    float ms = 0.f;
    double ksum = 0.0, csum = 0.0;
    cudaEventElapsedTime(&ms, ev[0], ev[4 * (n - 1) + 3]);
    stats[0] = std::chrono::duration<double>(w1 - w0).count();
    stats[1] = ms * 1e-3;
    for (int k = 0; k < n; ++k) {
      cudaEventElapsedTime(&ms, ev[4 * k + 2], ev[4 * k + 3]);
      ksum += ms * 1e-3;
      cudaEventElapsedTime(&ms, ev[4 * k + 0], ev[4 * k + 1]);
      csum += ms * 1e-3;
    }
    stats[2] = ksum;
    stats[3] = csum;
  }
  for (cudaEvent_t &e : ev) cudaEventDestroy(e);
  return rc;
}

// ---------------------------------------------------------------------------- F-stage

corr_fstage *corr_fstage_create(int n_inputs, int n_fft, int n_batch) {
  g_status = CORR_OK;
  g_err[0] = 0;
  if (n_inputs <= 0 || n_fft <= 0 || n_batch <= 0) {
    fail(CORR_EINVAL, "corr_fstage_create: n_inputs, n_fft, n_batch must be positive (got %d, %d, %d)", n_inputs, n_fft, n_batch);
    return nullptr;
  }
  if (n_fft != corr::kFftN) {
    fail(CORR_EUNSUPPORTED, "corr_fstage_create: n_fft must be 128 (the paper's N_C, PAPER.md:164; got %d)", n_fft);
    return nullptr;
  }
  if (n_inputs % corr::kFftTile != 0 || n_inputs > 4096) {
    fail(CORR_EUNSUPPORTED, "corr_fstage_create: n_inputs must be a multiple of 32 and <= 4096 (got %d)", n_inputs);
    return nullptr;
  }
  if (static_cast<long long>(n_batch) * corr::kFftN * n_inputs > 0x7fffffffLL) {  // 32-bit element offsets
    fail(CORR_EUNSUPPORTED, "corr_fstage_create: n_batch * n_inputs too large");
    return nullptr;
  }
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    fail(CORR_ECUDA, "corr_fstage_create: no usable CUDA device (%s)", cudaGetErrorString(cudaGetLastError()));
    return nullptr;
  }
  if (prop.major != 10) {
    fail(CORR_EARCH, "corr_fstage_create: device is sm_%d%d, this library is built for sm_100a only", prop.major, prop.minor);
    return nullptr;
  }
  // twiddles exp(-2 pi i m / 128) in float64, rounded once to float32
  float2 tw[corr::kFftN];
  for (int m = 0; m < corr::kFftN; ++m) {
    const double phi = 2.0 * 3.14159265358979323846 * m / corr::kFftN;
    tw[m] = make_float2(static_cast<float>(cos(phi)), static_cast<float>(-sin(phi)));
  }
  if (cudaMemcpyToSymbol(corr::c_tw128, tw, sizeof tw) != cudaSuccess) {
    fail(CORR_ECUDA, "corr_fstage_create: cudaMemcpyToSymbol: %s", cudaGetErrorString(cudaGetLastError()));
    return nullptr;
  }
  corr_fstage *f = new (std::nothrow) corr_fstage();
  if (!f) { fail(CORR_EALLOC, "corr_fstage_create: out of host memory"); return nullptr; }
  f->n_inputs = n_inputs; f->n_fft = n_fft; f->n_batch = n_batch; f->in_dtype = CORR_CI8;
  f->device = dev;
  f->d_raw[0] = f->d_raw[1] = f->d_spec = nullptr;
  f->in_bytes = static_cast<size_t>(n_batch) * n_fft * n_inputs * 2;
  f->out_bytes = static_cast<size_t>(n_batch) * n_fft * n_inputs * 8;
  return f;
}

int corr_fstage_run(corr_fstage *f, const void *d_raw, void *d_spec, void *stream) {
  if (!f || !d_raw || !d_spec) return fail(CORR_EINVAL, "corr_fstage_run: NULL argument");
  if ((reinterpret_cast<uintptr_t>(d_raw) & 15) || (reinterpret_cast<uintptr_t>(d_spec) & 15))
    return fail(CORR_EINVAL, "corr_fstage_run: pointers must be 16-byte aligned");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != f->device)
    return fail(CORR_EINVAL, "corr_fstage_run: the handle was created on device %d, the current device is %d", f->device, dev);
  corr::FftParams p;
  p.raw = static_cast<const int8_t *>(d_raw);
  p.spec = static_cast<float2 *>(d_spec);
  p.n_batch = f->n_batch; p.n_inputs = f->n_inputs; p.tiles_per_batch = f->n_inputs / corr::kFftTile;
  if (f->in_dtype == CORR_CI4)
    corr::fengine_ci4_kernel<<<f->n_batch * p.tiles_per_batch, corr::kFftThreads, 0, static_cast<cudaStream_t>(stream)>>>(p);
  else
    corr::fengine_kernel<<<f->n_batch * p.tiles_per_batch, corr::kFftThreads, 0, static_cast<cudaStream_t>(stream)>>>(p);
  CUDA_TRY(cudaGetLastError());
  return CORR_OK;
}

int corr_fstage_set_input(corr_fstage *f, int dtype) {
  if (!f) return fail(CORR_EINVAL, "corr_fstage_set_input: NULL handle");
  if (dtype != CORR_CI8 && dtype != CORR_CI4) return fail(CORR_EINVAL, "corr_fstage_set_input: dtype must be CORR_CI8 or CORR_CI4");
  if (dtype != f->in_dtype) {  // the streaming buffers are sized for the input format
    cudaFree(f->d_raw[0]);
    cudaFree(f->d_raw[1]);
    f->d_raw[0] = f->d_raw[1] = nullptr;
  }
  f->in_dtype = dtype;
  f->in_bytes = static_cast<size_t>(f->n_batch) * f->n_fft * f->n_inputs * (dtype == CORR_CI4 ? 1 : 2);
  return CORR_OK;
}

int corr_fstage_destroy(corr_fstage *f) {
  if (f) {
    cudaFree(f->d_raw[0]);
    cudaFree(f->d_raw[1]);
    cudaFree(f->d_spec);
  }
  delete f;
  return CORR_OK;
}

size_t corr_fstage_in_bytes(const corr_fstage *f) { return f ? f->in_bytes : 0; }
size_t corr_fstage_out_bytes(const corr_fstage *f) { return f ? f->out_bytes : 0; }

}  // extern "C"
