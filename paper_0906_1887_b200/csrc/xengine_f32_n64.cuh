// xengine_f32_n64.cuh -- complex-float32 X-engine for N_I = 64 (the paper's 32 antennas x 2 polarisations,
// PAPER.md:86; config c5), step a4 of DESIGN.md with an 8 x 4 complex register tile.
//
// Why a second kernel: in xengine_f32.cuh (4 x 4 tiles) the shared-memory RETURN path is as busy as the FMA pipe --
// an LDS.128 returns 512 B per warp = 4 cycles of the SM's 128 B/cycle whatever the broadcast, and a 4 x 4 tile needs
// 4 of them per 64 FFMA.  An 8 x 4 tile needs 6 per 128 FFMA (0.75 load cycles per FMA cycle).  The 64-input lower
// triangle is 72 such tiles; 7 ADJACENT channels share a CTA so that 504 threads = 16 warps (4 per scheduler, 128
// registers each) are all busy (3.5 KB contiguous per time row in d_in), and the integration is cut into time slices
// so that the (group, slice) units fill the 148 SMs evenly (c5: 220 groups x 2 slices = 440 units = 2.97 per SM); slices add their partial sums
// with red.global.add.v2.f32 into a zeroed d_vis (FP32 sums in a different order: within the 1e-5 tolerance, reading R8).
//
// V_ij = sum_t x_i conj(x_j), FP32 FMA accumulation; no tensor cores (TF32 cannot meet 1e-5).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ptx_sm100.cuh"    // mbarrier, cp.async.bulk
#include "xengine_f32.cuh"

namespace corr {

constexpr int kN64Chan = 7;                    // channels per CTA
constexpr int kN64Tiles = 72;                  // 8 x 4 tiles of the 64-input lower triangle
constexpr int kN64Threads = kN64Chan * kN64Tiles;  // 504
constexpr int kN64TB = 16;                     // time rows per stage
constexpr int kN64Stages = 3;
constexpr int kN64RowF4 = kN64Chan * 32;       // float4 per time row of a group (3.5 KB)
constexpr int kN64Warps = (kN64Threads + 31) / 32;               // 16
constexpr int kN64Smem = kN64Stages * kN64TB * kN64RowF4 * 16 + 64;  // 168 KB + the stage barriers

struct F32N64Params {
  const float2 *in;  // [T][C][64]
  float2 *vis;       // [C][2080]
  int n_time, n_chan, n_groups, n_slices, slice_len;
  int n_full;        // the first n_full groups are whole integrations (one unit each, plain stores); the other
                     // n_groups - n_full groups are cut into n_slices time slices that reduce-add into zeroed output
  int n_chan_total, chan0;  // d_in is [T][n_chan_total][64]; this handle correlates channels chan0 .. chan0 + n_chan - 1
  int add;           // 1: accumulate mode, every unit reduce-adds into d_vis; 0: only the units of sliced groups do
};

__device__ __forceinline__ void red_add_f32x2(float2 *dst, float re, float im) {
  asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(dst), "f"(re), "f"(im) : "memory");
}

__device__ __forceinline__ void ffma2(float2 &acc, const float2 &a, const float2 &b) {
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(reinterpret_cast<unsigned long long &>(acc))
      : "l"(reinterpret_cast<const unsigned long long &>(a)), "l"(reinterpret_cast<const unsigned long long &>(b)));
}

__global__ void __launch_bounds__(kN64Threads, 1) xengine_f32_n64_kernel(const F32N64Params p) {
  extern __shared__ __align__(16) float4 n64_smem[];
  const int tid = threadIdx.x;
  // units: the whole groups first (they are the long ones), then the slices of the sliced groups
  int grp, t0, t1;
  bool add = p.add != 0;
  if (static_cast<int>(blockIdx.x) < p.n_full) {
    grp = blockIdx.x; t0 = 0; t1 = p.n_time;
  } else {
    const int u = static_cast<int>(blockIdx.x) - p.n_full;
    const int n_cut = p.n_groups - p.n_full;
    grp = p.n_full + u % n_cut;
    t0 = (u / n_cut) * p.slice_len;
    t1 = min(p.n_time, t0 + p.slice_len);
    add = add || p.n_slices > 1;
  }
  const int c0 = grp * kN64Chan;
  const int n_chan_here = min(kN64Chan, p.n_chan - c0);

  // thread -> (channel of the group, 8 x 4 tile): row tile ti (inputs 8 ti ..), column tile tj <= 2 ti + 1 (inputs 4 tj ..)
  const int cg = tid / kN64Tiles;
  const int q = tid - cg * kN64Tiles;
  int ti = 0;
  while ((ti + 1) * (ti + 2) <= q) ++ti;
  const int tj = q - ti * (ti + 1);
  // the two 16-byte column loads are taken in swapped order by every second group of four tj, so that the eight
  // lanes of a quarter warp hit eight different 16-byte banks; `sw` then only renames this thread's accumulators
  const int sw = (tj >> 2) & 1;
  const bool active = cg < n_chan_here;

  const long long row_f4 = static_cast<long long>(p.n_chan_total) * 32;  // float4 per time row of d_in
  const float4 *src0 = reinterpret_cast<const float4 *>(p.in) + static_cast<long long>(p.chan0 + c0) * 32;
  const int valid_f4 = n_chan_here * 32;

  // Stage pipeline: one thread feeds a ring of kN64Stages stages with bulk copies (one contiguous 3.5 KB run per time
  // row) that complete on the stage's `full` mbarrier; every warp arrives on the stage's `empty` mbarrier when it has
  // consumed it.  No CTA-wide barrier in the loop: warps drift up to two stages apart instead of meeting 32 times.
  uint64_t *full_bar = reinterpret_cast<uint64_t *>(n64_smem + kN64Stages * kN64TB * kN64RowF4);
  uint64_t *empty_bar = full_bar + kN64Stages;
  if (tid == 0) {
    for (int s = 0; s < kN64Stages; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], kN64Warps);
    }
    fence_mbar_init();
  }
  __syncthreads();
  const uint32_t row_bytes = static_cast<uint32_t>(valid_f4) * 16;
  auto load_stage = [&](int s) {  // thread 0 only
    const int slot = s % kN64Stages;
    float4 *dst = n64_smem + slot * (kN64TB * kN64RowF4);
    const int tb = t0 + s * kN64TB;
    const int rows = min(kN64TB, t1 - tb);
    mbar_expect_tx(&full_bar[slot], rows * row_bytes);
    for (int r = 0; r < rows; ++r)
      bulk_load(dst + r * kN64RowF4, src0 + static_cast<long long>(tb + r) * row_f4, row_bytes, &full_bar[slot]);
  };

  float2 acc[8][4];  // (Re, Im) of V_ij, i = 8 ti + a, j = this thread's b-th column
#pragma unroll
  for (int a = 0; a < 8; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = make_float2(0.f, 0.f);

  const int n_stages = (t1 - t0 + kN64TB - 1) / kN64TB;
  if (tid == 0)
    for (int s = 0; s < min(kN64Stages, n_stages); ++s) load_stage(s);

  const int off_i = cg * 32 + 4 * ti;
  const int off_j0 = cg * 32 + 2 * tj + sw, off_j1 = cg * 32 + 2 * tj + 1 - sw;
  for (int s = 0; s < n_stages; ++s) {
    const int slot = s % kN64Stages;
    const uint32_t par = (s / kN64Stages) & 1;
    // refill the slot of the PREVIOUS stage (the other warps have had a whole stage's time to leave it, so this wait
    // rarely blocks) with the stage two ahead of this one
    if (tid == 0 && s >= 1 && s - 1 + kN64Stages < n_stages) {
      mbar_wait(&empty_bar[(s - 1) % kN64Stages], ((s - 1) / kN64Stages) & 1);
      load_stage(s - 1 + kN64Stages);
    }
    mbar_wait(&full_bar[slot], par);  // the stage's rows have landed
    const float4 *st = n64_smem + slot * (kN64TB * kN64RowF4);
    const int rows = min(kN64TB, t1 - (t0 + s * kN64TB));
#pragma unroll 2
    for (int r = 0; r < rows; ++r) {
      const float4 *row = st + r * kN64RowF4;
      const float4 a0 = row[off_i], a1 = row[off_i + 1], a2 = row[off_i + 2], a3 = row[off_i + 3];
      const float4 b0 = row[off_j0], b1 = row[off_j1];
      // x_i conj(x_j) = (a_i, b_i) a_j + (b_i, -a_i) b_j: two packed FMAs (fma.rn.f32x2) per product, the x_i
      // operand pairs exactly as they lie in shared memory
      const float2 xi[8] = {make_float2(a0.x, a0.y), make_float2(a0.z, a0.w), make_float2(a1.x, a1.y), make_float2(a1.z, a1.w),
                            make_float2(a2.x, a2.y), make_float2(a2.z, a2.w), make_float2(a3.x, a3.y), make_float2(a3.z, a3.w)};
      const float bre[4] = {b0.x, b0.z, b1.x, b1.z}, bim[4] = {b0.y, b0.w, b1.y, b1.w};
      float2 br2[4], bi2[4];
#pragma unroll
      for (int b = 0; b < 4; ++b) { br2[b] = make_float2(bre[b], bre[b]); bi2[b] = make_float2(bim[b], bim[b]); }
#pragma unroll
      for (int a = 0; a < 8; ++a) {
        const float2 xs = make_float2(xi[a].y, -xi[a].x);
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          ffma2(acc[a][b], xi[a], br2[b]);
          ffma2(acc[a][b], xs, bi2[b]);
        }
      }
    }
    // this warp is done with the stage
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(&empty_bar[slot]);
  }

  if (active) {
    float2 *vis_c = p.vis + static_cast<long long>(c0 + cg) * 2080;
#pragma unroll
    for (int a = 0; a < 8; ++a) {
      const int i = 8 * ti + a;
      float2 *rowp = vis_c + i * (i + 1) / 2;
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const int j = 4 * tj + ((((b >> 1) ^ sw)) << 1) + (b & 1);
        if (j <= i) {
          const float vim = (j == i) ? 0.f : acc[a][b].y;  // Im of an autocorrelation is exactly 0 (reading R9)
          if (add) red_add_f32x2(rowp + j, acc[a][b].x, vim);
          else       rowp[j] = make_float2(acc[a][b].x, vim);
        }
      }
    }
  }
}

}  // namespace corr
