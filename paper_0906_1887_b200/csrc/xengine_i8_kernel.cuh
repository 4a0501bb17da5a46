// xengine_i8_kernel.cuh -- the kernel body of xengine_i8.cuh (included from there).
#pragma once

namespace corr {

__global__ void __launch_bounds__(kI8Threads, 1)
xengine_i8_kernel(const __grid_constant__ CUtensorMap tmap256, const __grid_constant__ CUtensorMap tmap128,
                  const __grid_constant__ CUtensorMap tmap64, const __grid_constant__ I8Params p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ __align__(8) uint64_t full_bar[kMaxStages];
  __shared__ __align__(8) uint64_t empty_bar[kMaxStages];
  __shared__ __align__(8) uint64_t acc_full[2];
  __shared__ __align__(8) uint64_t acc_empty[2];
  __shared__ uint32_t tmem_base_smem;

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int n_rounds = (p.n_items + gridDim.x - 1) / gridDim.x;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmap256);
    tma_prefetch_desc(&tmap128);
    tma_prefetch_desc(&tmap64);
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], 1);
    }
    for (int r = 0; r < 2; ++r) {
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

  if (warp == 0) {
    // ===================================================================== TMA producer
    if (lane == 0 && !(p.probe & 8)) {
      const uint64_t pol = policy_evict_normal();
      int stage = 0;
      uint32_t phase = 0;
      for (int r = 0; r < n_rounds; ++r) {
        const int g = item_of_round(p, r);
        if (g >= p.n_items) continue;
        const I8Item it = decode_item(p, g);
        const CUtensorMap *map = it.map == 0 ? &tmap256 : (it.map == 1 ? &tmap128 : &tmap64);
        const uint32_t panel_bytes = static_cast<uint32_t>(it.bk) * kPanelBytes;
        for (int t = it.t0; t < it.t1; t += it.bk) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          if (p.probe & 2) {
            mbar_arrive(&full_bar[stage]);
          } else {
            mbar_expect_tx(&full_bar[stage], panel_bytes * it.n_load);
            uint8_t *dst = smem + static_cast<size_t>(stage) * p.stage_bytes;
            for (int l = 0; l < it.n_load; ++l) {
              const bool is_a = l >= it.nblk;
              const int x = is_a ? it.xa : it.x0 + l * it.dx;
              const int z = is_a ? it.za : it.z0 + l * it.dz;
              if (p.turned) tma_load_3d(dst + l * panel_bytes, map, &full_bar[stage], x, t, z, pol);
              else          tma_load_2d(dst + l * panel_bytes, map, &full_bar[stage], x, t, pol);
            }
          }
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer
    // The whole warp walks the (uniform) schedule so that loop state lives in uniform registers;
    // one lane issues.  Descriptor low words are advanced by plain adds (all offsets are multiples
    // of 16 B and the address field cannot carry into the LBO field below 256 KB).
    {
      const bool leader = lane == 0;
      int stage = 0;
      uint32_t phase = 0;
      uint32_t ring = 0;  // accumulator ring entries handed out so far
      constexpr uint32_t kIdesc128 = idesc_i8_mn(128, 128), kIdesc256 = idesc_i8_mn(128, 256);
      constexpr uint32_t kDescHi = static_cast<uint32_t>(((1024ull >> 4) | (1ull << 14) | (2ull << 29)));
      const uint32_t smem_lo = __reduce_or_sync(0xffffffffu, (smem_u32(smem) & 0x3FFFFu) >> 4);
      // REDUX lands in a uniform register: keeps the TMEM addresses out of the vector file (no R2UR per MMA)
      const uint32_t tmem_u = __reduce_or_sync(0xffffffffu, tmem_base);
      const long long dbg_t0 = clock64();
      int dbg_n = 0;
      for (int r = 0; r < n_rounds; ++r) {
        const int g = item_of_round(p, r);
        if (g >= p.n_items) continue;
        const I8Item it = decode_item(p, g);
        const uint32_t panel16 = static_cast<uint32_t>(it.bk) * (kPanelBytes / 16);  // panel bytes / 16
        const uint32_t lbo_field = (panel16 & 0x3FFFu) << 16;
        const int n_chunks = (it.nblk + 1) >> 1;
        if (!(p.probe & 4))
          for (int q = 0; q < n_chunks; ++q) mbar_wait(&acc_empty[(ring + q) & 1], (((ring + q) >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t d0 = tmem_u + (ring & 1) * kAccCols;        // chunk 0
        uint32_t d1 = tmem_u + ((ring + 1) & 1) * kAccCols;  // chunk 1
        if (p.probe & 64) d1 = d0;
        for (int t = it.t0; t < it.t1; t += it.bk) {
          if (!(p.probe & 8)) mbar_wait(&full_bar[stage], phase);
          if (!(p.probe & 32)) tc_fence_after();
          const uint32_t lo_stage = (smem_lo + static_cast<uint32_t>(stage) * (p.stage_bytes >> 4)) | lbo_field;
          const int nk = (min(it.bk, it.t1 - t) + 31) >> 5;  // K = 32 samples per MMA; TMA zero-fills past T
          if (leader) {
            for (int k = 0; k < ((p.probe & 1) ? 0 : nk); ++k) {
              const uint32_t lo_k = lo_stage + static_cast<uint32_t>(k) * (32 * kPanelBytes / 16);
              const uint32_t acc = (t != it.t0 || k != 0) ? 1u : 0u;  // uniform: first MMA of the slice overwrites
              if (p.diag) {
                for (int b = 0; b < it.nblk; ++b) {
                  const uint64_t d = (static_cast<uint64_t>(kDescHi) << 32) | (lo_k + b * panel16);
                  mma_i8_ss(((b & 2) ? d1 : d0) + (b & 1) * 128, d, d, kIdesc128, acc);
                }
              } else {
                const uint64_t a_desc = (static_cast<uint64_t>(kDescHi) << 32) | (lo_k + it.a_slot * panel16);
                const uint64_t b_desc0 = (static_cast<uint64_t>(kDescHi) << 32) | lo_k;
                mma_i8_ss(d0, a_desc, b_desc0, it.nblk >= 2 ? kIdesc256 : kIdesc128, acc);
                if (it.nblk > 2) {
                  const uint64_t b_desc1 = (static_cast<uint64_t>(kDescHi) << 32) | (lo_k + 2 * panel16);
                  mma_i8_ss(d1, a_desc, b_desc1, it.nblk == 4 ? kIdesc256 : kIdesc128, acc);
                }
              }
              ++dbg_n;
            }
            if (!(p.probe & 8)) mma_commit(&empty_bar[stage]);  // frees the smem stage when these MMAs retire
          }
          __syncwarp();
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
        if (leader)
          for (int q = 0; q < n_chunks; ++q) mma_commit(&acc_full[(ring + q) & 1]);
        __syncwarp();
        ring += n_chunks;
      }
      if ((p.probe & 128) && leader && blockIdx.x < 8)
        p.vis[blockIdx.x] = make_int2(static_cast<int>(clock64() - dbg_t0), dbg_n);
    }
  } else if (warp >= 4 && !(p.probe & 4)) {
    // ===================================================================== epilogue
    const int ew = warp - 4;               // TMEM lanes 32*ew .. 32*ew+31
    const int part = lane & 1;             // 0: row 2i (Re row of input i), 1: row 2i+1 (Im row)
    const int li = ew * 16 + (lane >> 1);  // local input index within the row panel
    const bool atomic = p.n_slices > 1;
    uint32_t ring = 0;
    for (int r = 0; r < n_rounds; ++r) {
      const int g = item_of_round(p, r);
      if (g >= p.n_items) continue;
      const I8Item it = decode_item(p, g);
      const int n_chunks = (it.nblk + 1) >> 1;
      for (int q = 0; q < n_chunks; ++q) {
        const uint32_t e = ring + q;
        mbar_wait(&acc_full[e & 1], (e >> 1) & 1);
        tc_fence_after();
        const uint32_t tchunk = tmem_base + (static_cast<uint32_t>(ew * 32) << 16) + (e & 1) * kAccCols;
        const int nb_here = min(2, it.nblk - 2 * q);
        for (int bb = 0; bb < nb_here; ++bb) {
          const int b = 2 * q + bb;
          // block b: which channel / inputs do its 128 rows x 128 columns hold?
          int chan, i_glob, j_blk0;  // this lane's channel and input i; first input j of the block
          bool diag_blk;
          if (p.diag) {
            const int panel = it.J0 + b;
            chan = p.pair_mode ? 2 * panel + (li >> 5) : panel;
            i_glob = p.pair_mode ? (li & 31) : li;
            j_blk0 = 0;
            diag_blk = true;
          } else {
            chan = it.chan;
            i_glob = it.I * 64 + li;
            j_blk0 = (it.J0 + b) * 64;
            diag_blk = (it.J0 + b) == it.I;
          }
          const bool row_ok = (chan < p.n_chan) && (i_glob < p.n_inputs);
          int2 *row_ptr = p.vis + (static_cast<long long>(chan) * p.n_baselines +
                                   static_cast<long long>(i_glob) * (i_glob + 1) / 2);
          for (int cb = 0; cb < 4; ++cb) {  // 32 TMEM columns = 16 inputs j per batch
            // warp-uniform skips: batches entirely above the diagonal / in the other channel / past N_I
            int j_base;
            bool batch_ok;
            if (p.pair_mode) {
              j_base = (cb & 1) * 16;
              batch_ok = ((cb >> 1) == (ew >> 1)) && (j_base <= (ew & 1) * 16 + 15);
            } else {
              j_base = j_blk0 + cb * 16;
              batch_ok = (j_base < p.n_inputs) && (!diag_blk || cb * 16 <= ew * 16 + 15);
            }
            if (!batch_ok) continue;
            uint32_t v[32];
            tmem_ld_32x32(tchunk + bb * 128 + cb * 32, v);
            tmem_ld_wait();
            int rr[16];
#pragma unroll
            for (int jj = 0; jj < 16; ++jj) {
              const int other = __shfl_xor_sync(0xffffffffu, static_cast<int>(v[2 * jj + 1]), 1);
              rr[jj] = part ? (static_cast<int>(v[2 * jj]) - other) : (static_cast<int>(v[2 * jj]) + other);
            }
            // even lane keeps columns 0..7 (has Re, needs Im); odd lane keeps 8..15 (has Im, needs Re)
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const int send = part ? rr[u] : rr[u + 8];
              const int recv = __shfl_xor_sync(0xffffffffu, send, 1);
              const int re = part ? recv : rr[u];
              const int im = part ? rr[u + 8] : recv;
              const int j = j_base + part * 8 + u;
              if (row_ok && j <= i_glob && j < p.n_inputs) {
                if (atomic) put_vis<true>(row_ptr + j, re, j == i_glob ? 0 : im);
                else        put_vis<false>(row_ptr + j, re, j == i_glob ? 0 : im);
              }
            }
          }
        }
        // every tcgen05.ld of this ring entry has completed (wait::ld above): hand it back
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
