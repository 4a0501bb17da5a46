// xengine_i8.cuh -- int8 complex X-engine on tcgen05 (steps a1-fused, a2, a3, a6 of DESIGN.md).
//
// Per channel c the CMAC is the real Gram matrix G = Y^T Y of the
// (T x 2N) int8 matrix Y whose row t is the raw sample vector [Re x_0, Im x_0, Re x_1, ...]
// exactly as it lies in d_in[t][c][:].  G is cut into 128-row "panels" (64 inputs each).
// A work item = (channel, row panel I, column panels J0..J0+nJ-1 <= I): a 128 x (128*nJ)
// slab of G accumulated over all T in TMEM (int32), then folded to complex visibilities
//   Re V_ij = G[2i][2j] + G[2i+1][2j+1],  Im V_ij = G[2i+1][2j] - G[2i][2j+1]
// and written to the packed lower triangle.
//
// Warp roles (256 threads, 1 CTA/SM, persistent over a static item schedule):
//   warp 0   TMA producer: box {128 B along the chan*input axis, BK time rows}, SWIZZLE_128B.
//            This strided box load IS the corner turn: it lands as the
//            canonical MN-major operand tile, so the input is read from HBM exactly once.
//   warp 1   MMA issuer (one thread): tcgen05.mma.kind::i8, M=128, N=128|256, K=32.
//   warp 2   TMEM allocator.
//   warps 4-7 epilogue: tcgen05.ld, 2x2 fold via shfl.xor 1, masked packed-triangle stores.
#pragma once
#include "ptx_sm100.cuh"

namespace corr {

constexpr int kI8Threads = 256;
constexpr int kPanelBytes = 128;     // bytes of the chan*input axis per panel = 64 complex int8 inputs
constexpr int kAccCols = 256;        // TMEM columns per accumulator ring entry
constexpr int kAccRing = 2;          // 2 x 256 = all 512 TMEM columns
constexpr int kMaxStages = 16;

struct I8Params {
  const int4 *items;   // {chan, I | J0 << 16, nJ, pad}, grouped per CTA
  const int *offsets;  // [grid + 1]: CTA b owns items offsets[b] .. offsets[b+1]-1 (static balanced schedule)
  int n_time;          // T
  int n_inputs;        // N_I
  int n_chan;          // C
  int pair_mode;       // N_I == 32: one panel = two adjacent channels
  int bk;              // time rows per pipeline stage (multiple of 32)
  int slots;           // panels per stage slot array
  int stages;
  int turned;          // 0: d_in is [T][C][2N] (2-D map); 1: scratch is [C][T][2N] (3-D map)
  long long n_baselines;
  int2 *vis;
};

__device__ __forceinline__ void store_vis8(int2 *row_ptr, int i_glob, int j0, int n_inputs, const int (&re)[8],
                                           const int (&im)[8]) {
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    const int j = j0 + u;
    if (j <= i_glob && j < n_inputs) row_ptr[j] = make_int2(re[u], j == i_glob ? 0 : im[u]);
  }
}

__global__ void __launch_bounds__(kI8Threads, 1)
xengine_i8_kernel(const __grid_constant__ CUtensorMap tmap, const I8Params p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ __align__(8) uint64_t full_bar[kMaxStages];
  __shared__ __align__(8) uint64_t empty_bar[kMaxStages];
  __shared__ __align__(8) uint64_t acc_full[kAccRing];
  __shared__ __align__(8) uint64_t acc_empty[kAccRing];
  __shared__ uint32_t tmem_base_smem;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t panel_stage_bytes = static_cast<uint32_t>(p.bk) * kPanelBytes;
  const uint32_t stage_bytes = panel_stage_bytes * p.slots;
  const int n_ksteps = (p.n_time + p.bk - 1) / p.bk;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmap);
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], 1);
    }
    for (int r = 0; r < kAccRing; ++r) {
      mbar_init(&acc_full[r], 1);
      mbar_init(&acc_empty[r], 4);  // one arrive per epilogue warp
    }
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc(&tmem_base_smem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const int it_begin = p.offsets[blockIdx.x], it_end = p.offsets[blockIdx.x + 1];

  if (warp == 0) {
    // ===================================================================== TMA producer
    if (lane == 0) {
      const uint64_t pol = policy_evict_normal();
      int stage = 0;
      uint32_t phase = 0;
      for (int it = it_begin; it < it_end; ++it) {
        const int4 item = p.items[it];
        const int chan = item.x, I = item.y & 0xFFFF, J0 = item.y >> 16, nJ = item.z;
        const bool a_in_b = (I >= J0) && (I < J0 + nJ);
        const int n_load = nJ + (a_in_b ? 0 : 1);
        const int x0 = p.turned ? 0 : chan * p.n_inputs * 2;
        for (int ks = 0; ks < n_ksteps; ++ks) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          mbar_expect_tx(&full_bar[stage], panel_stage_bytes * n_load);
          uint8_t *dst = smem + static_cast<size_t>(stage) * stage_bytes;
          for (int l = 0; l < n_load; ++l) {
            const int panel = (l < nJ) ? (J0 + l) : I;
            if (p.turned)
              tma_load_3d(dst + l * panel_stage_bytes, &tmap, &full_bar[stage], panel * kPanelBytes, ks * p.bk,
                          p.pair_mode ? (chan >> 1) : chan, pol);
            else
              tma_load_2d(dst + l * panel_stage_bytes, &tmap, &full_bar[stage], x0 + panel * kPanelBytes,
                          ks * p.bk, pol);
          }
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      uint32_t ring = 0;  // running count of accumulator ring entries handed out
      for (int it = it_begin; it < it_end; ++it) {
        const int4 item = p.items[it];
        const int I = item.y & 0xFFFF, J0 = item.y >> 16, nJ = item.z;
        const bool a_in_b = (I >= J0) && (I < J0 + nJ);
        const int a_slot = a_in_b ? (I - J0) : nJ;
        const int n_chunks = (nJ + 1) >> 1;
        for (int q = 0; q < n_chunks; ++q) {
          const uint32_t e = ring + q;
          mbar_wait(&acc_empty[e & 1], ((e >> 1) & 1) ^ 1);
        }
        tc_fence_after();
        for (int ks = 0; ks < n_ksteps; ++ks) {
          mbar_wait(&full_bar[stage], phase);
          tc_fence_after();
          const uint32_t sbase = smem_u32(smem + static_cast<size_t>(stage) * stage_bytes);
          const int rows = min(p.bk, p.n_time - ks * p.bk);
          const int nk = (rows + 31) >> 5;  // K = 32 time samples per MMA; TMA zero-fills the tail
          for (int k = 0; k < nk; ++k) {
            const uint32_t koff = static_cast<uint32_t>(k) * 32 * kPanelBytes;
            const uint64_t a_desc = smem_desc_mn_sw128(sbase + a_slot * panel_stage_bytes + koff, panel_stage_bytes, 1024);
            for (int q = 0; q < n_chunks; ++q) {
              const int np = min(2, nJ - 2 * q);
              const uint64_t b_desc =
                  smem_desc_mn_sw128(sbase + (2 * q) * panel_stage_bytes + koff, panel_stage_bytes, 1024);
              const uint32_t d = tmem_base + ((ring + q) & 1) * kAccCols;
              mma_i8_ss(d, a_desc, b_desc, np == 2 ? idesc_i8_mn(128, 256) : idesc_i8_mn(128, 128),
                        (ks | k) != 0);
            }
          }
          mma_commit(&empty_bar[stage]);  // frees the smem stage when these MMAs retire
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
        for (int q = 0; q < n_chunks; ++q) mma_commit(&acc_full[(ring + q) & 1]);
        ring += n_chunks;
      }
    }
  } else if (warp >= 4) {
    // ===================================================================== epilogue
    const int ew = warp - 4;               // TMEM lanes 32*ew .. 32*ew+31
    const int part = lane & 1;             // 0: row 2i (Re row of input i), 1: row 2i+1 (Im row)
    const int li = ew * 16 + (lane >> 1);  // local input index within the row panel
    uint32_t ring = 0;
    for (int it = it_begin; it < it_end; ++it) {
      const int4 item = p.items[it];
      const int chan0 = item.x, I = item.y & 0xFFFF, J0 = item.y >> 16, nJ = item.z;
      const int n_chunks = (nJ + 1) >> 1;
      int chan, i_glob;
      if (p.pair_mode) { chan = chan0 + (li >> 5); i_glob = li & 31; }
      else             { chan = chan0;             i_glob = I * 64 + li; }
      const bool row_ok = (chan < p.n_chan) && (i_glob < p.n_inputs);
      int2 *row_ptr = p.vis + (static_cast<long long>(chan) * p.n_baselines +
                               static_cast<long long>(i_glob) * (i_glob + 1) / 2);
      // highest input index any lane of this warp owns (warp-uniform skip of all-upper batches)
      const int i_warp_max = p.pair_mode ? ((ew & 1) * 16 + 15) : (I * 64 + ew * 16 + 15);
      for (int q = 0; q < n_chunks; ++q) {
        const uint32_t e = ring + q;
        mbar_wait(&acc_full[e & 1], (e >> 1) & 1);
        tc_fence_after();
        const int np = min(2, nJ - 2 * q);
        const uint32_t tchunk = tmem_base + (static_cast<uint32_t>(ew * 32) << 16) + (e & 1) * kAccCols;
        for (int cb = 0; cb < np * 4; ++cb) {  // 32 TMEM columns = 16 inputs j per batch
          int j_base;                           // global input index of the batch's first column pair
          bool batch_ok;
          if (p.pair_mode) {
            j_base = (cb & 1) * 16;
            batch_ok = ((cb >> 1) == (ew >> 1)) && (j_base <= i_warp_max);
          } else {
            j_base = (J0 + 2 * q + (cb >> 2)) * 64 + (cb & 3) * 16;
            batch_ok = (j_base <= i_warp_max) && (j_base < p.n_inputs);
          }
          if (!batch_ok) continue;  // warp-uniform
          uint32_t v[32];
          tmem_ld_32x32(tchunk + cb * 32, v);
          tmem_ld_wait();
          int r[16];
#pragma unroll
          for (int jj = 0; jj < 16; ++jj) {
            const int other = __shfl_xor_sync(0xffffffffu, static_cast<int>(v[2 * jj + 1]), 1);
            r[jj] = part ? (static_cast<int>(v[2 * jj]) - other) : (static_cast<int>(v[2 * jj]) + other);
          }
          // even lane keeps columns 0..7 (has Re, needs Im); odd lane keeps 8..15 (has Im, needs Re)
          int re[8], im[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            const int send = part ? r[u] : r[u + 8];
            const int recv = __shfl_xor_sync(0xffffffffu, send, 1);
            re[u] = part ? recv : r[u];
            im[u] = part ? r[u + 8] : recv;
          }
          if (row_ok) store_vis8(row_ptr, i_glob, j_base + part * 8, p.n_inputs, re, im);
        }
        // all tcgen05.ld of this ring entry have completed (wait::ld above): hand it back
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&acc_empty[e & 1]);
      }
      ring += n_chunks;
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

}  // namespace corr
