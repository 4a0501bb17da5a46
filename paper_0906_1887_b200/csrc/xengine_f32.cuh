// xengine_f32.cuh -- complex-float32 X-engine on CUDA cores (step a4 of DESIGN.md).
//
// V_ij = sum_t x_i conj(x_j) with FP32 FMA accumulation, the same class of
// computation as the paper's own CMAC kernels but register-tiled: a thread owns a
// 4x4 block of complex accumulators (64 FFMA per 4 shared-memory operand loads) instead of one
// product per thread or G per thread.  No tensor cores: TF32's 10-bit
// mantissa cannot meet the 1e-5 tolerance.
//
// Work item = (channel, 64-input row block I, 64-input column block J <= I).  Samples of TB time
// rows are staged with cp.async (16 B per thread, coalesced along the input axis) into a
// double-buffered shared tile whose row layout is split so that a thread's four inputs are two
// conflict-free 16-byte reads:  row[h][g][2] float2, input = 4g + 2h + {0,1}.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace corr {

constexpr int kF32Block = 64;   // inputs per block edge
constexpr int kF32TB = 16;      // time rows per stage
constexpr int kF32Threads = 256;

struct F32Params {
  const float2 *in;   // [T][C][N]
  float2 *vis;        // [C][nb]
  const int2 *items;  // {chan, I | J << 16}
  int n_items;
  int n_time, n_chan, n_inputs;
  int n_chan_total, chan0;  // d_in is [T][n_chan_total][N]; this handle correlates channels chan0 .. chan0 + n_chan - 1
  long long n_baselines;
  int accumulate;  // 1: d_vis += this integration; every element has exactly one writer
};

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc, bool valid) {
  const uint32_t d = static_cast<uint32_t>(__cvta_generic_to_shared(smem_dst));
  const int sz = valid ? 16 : 0;  // src-size 0 => zero fill
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gsrc), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// One 64-input block of one time row is 512 B = 32 chunks of 16 B (2 inputs each).  Chunk k holds
// inputs 2k, 2k+1 -> g = k >> 1, h = k & 1 -> shared float4 index h*16 + g.
__device__ __forceinline__ void f32_stage_load(float4 *tile, const float2 *in, int t0, int n_time, long long row_stride,
                                               long long col0, int n_valid_chunks, int tid, int nthreads) {
  for (int idx = tid; idx < kF32TB * 32; idx += nthreads) {
    const int r = idx >> 5, k = idx & 31;
    const int t = t0 + r;
    const bool ok = (t < n_time) && (k < n_valid_chunks);
    const float2 *src = in + (ok ? (static_cast<long long>(t) * row_stride + col0 + 2 * k) : 0);
    cp_async16(&tile[r * 32 + (k & 1) * 16 + (k >> 1)], src, ok);
  }
}

__global__ void __launch_bounds__(kF32Threads) xengine_f32_kernel(const F32Params p) {
  __shared__ __align__(16) float4 tile_i[2][kF32TB * 32];
  __shared__ __align__(16) float4 tile_j[2][kF32TB * 32];

  const int2 item = p.items[blockIdx.x];
  const int chan = item.x, I = item.y & 0xFFFF, J = item.y >> 16;
  const bool diag = (I == J);
  const int tid = threadIdx.x;

  // thread -> 4x4 tile (ti, tj) of the 16x16 tile grid; diagonal blocks enumerate ti >= tj only
  int ti, tj;
  bool active;
  if (diag) {
    int r = 0;
    while ((r + 1) * (r + 2) / 2 <= tid) ++r;
    ti = r; tj = tid - r * (r + 1) / 2;
    active = tid < 136;
  } else {
    ti = tid >> 4; tj = tid & 15;
    active = true;
  }

  const long long row_stride = static_cast<long long>(p.n_chan_total) * p.n_inputs;
  const long long col_i = static_cast<long long>(p.chan0 + chan) * p.n_inputs + I * kF32Block;
  const long long col_j = static_cast<long long>(p.chan0 + chan) * p.n_inputs + J * kF32Block;

  const int nvc_i = min(32, (p.n_inputs - I * kF32Block) / 2);
  const int nvc_j = min(32, (p.n_inputs - J * kF32Block) / 2);

  float re[4][4], im[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) { re[a][b] = 0.f; im[a][b] = 0.f; }

  const int n_stages = (p.n_time + kF32TB - 1) / kF32TB;
  f32_stage_load(tile_i[0], p.in, 0, p.n_time, row_stride, col_i, nvc_i, tid, blockDim.x);
  if (!diag) f32_stage_load(tile_j[0], p.in, 0, p.n_time, row_stride, col_j, nvc_j, tid, blockDim.x);
  cp_async_commit();

  for (int s = 0; s < n_stages; ++s) {
    const int buf = s & 1;
    if (s + 1 < n_stages) {
      f32_stage_load(tile_i[buf ^ 1], p.in, (s + 1) * kF32TB, p.n_time, row_stride, col_i, nvc_i, tid, blockDim.x);
      if (!diag) f32_stage_load(tile_j[buf ^ 1], p.in, (s + 1) * kF32TB, p.n_time, row_stride, col_j, nvc_j, tid, blockDim.x);
      cp_async_commit();
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    if (active) {
      const float4 *ri = tile_i[buf];
      const float4 *rj = diag ? tile_i[buf] : tile_j[buf];
#pragma unroll 4
      for (int r = 0; r < kF32TB; ++r) {
        const float4 a01 = ri[r * 32 + ti], a23 = ri[r * 32 + 16 + ti];
        const float4 b01 = rj[r * 32 + tj], b23 = rj[r * 32 + 16 + tj];
        const float ar[4] = {a01.x, a01.z, a23.x, a23.z}, ai[4] = {a01.y, a01.w, a23.y, a23.w};
        const float br[4] = {b01.x, b01.z, b23.x, b23.z}, bi[4] = {b01.y, b01.w, b23.y, b23.w};
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            re[a][b] = fmaf(ar[a], br[b], re[a][b]);
            re[a][b] = fmaf(ai[a], bi[b], re[a][b]);
            im[a][b] = fmaf(ai[a], br[b], im[a][b]);
            im[a][b] = fmaf(-ar[a], bi[b], im[a][b]);
          }
      }
    }
    __syncthreads();
  }

  if (active) {
    float2 *vis_c = p.vis + static_cast<long long>(chan) * p.n_baselines;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      const int i = I * kF32Block + 4 * ti + a;
      if (i >= p.n_inputs) continue;
      float2 *row = vis_c + static_cast<long long>(i) * (i + 1) / 2;
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const int j = J * kF32Block + 4 * tj + b;
        if (j <= i) {
          float2 v = make_float2(re[a][b], j == i ? 0.f : im[a][b]);
          if (p.accumulate) { const float2 old = row[j]; v.x += old.x; v.y += old.y; }
          row[j] = v;
        }
      }
    }
  }
}

}  // namespace corr
