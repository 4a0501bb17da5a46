// corner_turn.cuh -- standalone corner turn (step a1 of DESIGN.md; "unpack").
//
// in  [T][G][W bytes]  ->  out [G][T][W bytes]      (G = channels, or channel pairs when N_I = 32)
// i.e. samples become per-channel, time-major tiles.  Pure byte permutation, no arithmetic: int8
// samples stay int8 (the paper's unpack also converts int -> float; not needed here).
//
// A CTA moves a tile of TT time rows x GG groups through shared memory: 16-byte vectorised loads
// that are contiguous along the group axis (GG*W bytes per time row), 16-byte vectorised stores
// that are contiguous along the time axis (TT*W bytes per group).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace corr {

constexpr int kTurnThreads = 256;
constexpr int kTurnTileBytes = 32768;

struct TurnParams {
  const uint4 *in;
  uint4 *out;
  int n_time;    // T
  int n_groups;  // G
  int wc;        // W / 16: 16-byte chunks per (t, g) row
  int tt, gg;    // tile extents (tt * gg * wc * 16 <= kTurnTileBytes)
  int g_tiles;   // ceil(G / gg): blockIdx.x = time tile * g_tiles + group tile (1-D grid: no 65535 limit on either)
  long long in_row_chunks;  // 16-byte chunks per time row of `in` (the full channel axis of a windowed handle)
  long long in_off_chunks;  // first chunk of group 0 within a time row of `in`
};

__global__ void __launch_bounds__(kTurnThreads) corner_turn_kernel(const TurnParams p) {
  __shared__ uint4 tile[kTurnTileBytes / 16];
  const int t_tile = blockIdx.x / p.g_tiles;
  const int t0 = t_tile * p.tt;
  const int g0 = (blockIdx.x - t_tile * p.g_tiles) * p.gg;
  const int tt = min(p.tt, p.n_time - t0);
  const int gg = min(p.gg, p.n_groups - g0);
  const int row_chunks = gg * p.wc;  // contiguous 16-byte chunks per time row of this tile
  const int n = tt * row_chunks;
  // load: chunk fastest, then group, then time  (global reads contiguous per time row)
  for (int idx = threadIdx.x; idx < n; idx += kTurnThreads) {
    const int t = idx / row_chunks, r = idx - t * row_chunks;
    tile[idx] = __ldg(p.in + static_cast<long long>(t0 + t) * p.in_row_chunks + p.in_off_chunks + static_cast<long long>(g0) * p.wc + r);
  }
  __syncthreads();
  // store: chunk fastest, then time, then group  (global writes contiguous per group)
  const int col_chunks = tt * p.wc;
  for (int idx = threadIdx.x; idx < n; idx += kTurnThreads) {
    const int g = idx / col_chunks, r = idx - g * col_chunks;
    const int t = r / p.wc, k = r - t * p.wc;
    p.out[(static_cast<long long>(g0 + g) * p.n_time + t0) * p.wc + r] = tile[t * row_chunks + g * p.wc + k];
  }
}

}  // namespace corr
