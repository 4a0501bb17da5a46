// xengine_i8_kernel.cuh -- the kernel body of xengine_i8.cuh (included from there).
#pragma once
#include "xengine_i8_epilogue.cuh"

namespace corr {

// NK back-to-back MMAs over the NK k-steps (32 time samples = 4096 B of a panel each) of one stage.
// Straight-line code: the descriptor words of all NK issues are independent of one another.
template <int NK, bool kPair>
__device__ __forceinline__ void issue_k(uint32_t d, uint32_t lo_a, uint32_t lo_b, uint32_t hi, uint32_t idesc,
                                        uint32_t acc0) {
#pragma unroll
  for (int k = 0; k < NK; ++k) {
    const uint64_t da = (static_cast<uint64_t>(hi) << 32) | (lo_a + k * (32 * kPanelBytes / 16));
    const uint64_t db = (static_cast<uint64_t>(hi) << 32) | (lo_b + k * (32 * kPanelBytes / 16));
    if (kPair) mma_i8_ss_2sm(d, da, db, idesc, k == 0 ? acc0 : 1u);
    else       mma_i8_ss(d, da, db, idesc, k == 0 ? acc0 : 1u);
  }
}
// 512-wide pair tiles: per k-step the same A tile multiplies two B tiles (column halves d0, d1).  Issued back to
// back with collector hints, so that the tensor core reads A from shared memory once per k-step instead of twice.
template <int NK>
__device__ __forceinline__ void issue_k_wide(uint32_t d0, uint32_t d1, uint32_t lo_a, uint32_t lo_b0, uint32_t lo_b1,
                                             uint32_t hi, uint32_t idesc, uint32_t acc0) {
#pragma unroll
  for (int k = 0; k < NK; ++k) {
    const uint64_t da = (static_cast<uint64_t>(hi) << 32) | (lo_a + k * (32 * kPanelBytes / 16));
    const uint64_t db0 = (static_cast<uint64_t>(hi) << 32) | (lo_b0 + k * (32 * kPanelBytes / 16));
    const uint64_t db1 = (static_cast<uint64_t>(hi) << 32) | (lo_b1 + k * (32 * kPanelBytes / 16));
    mma_i8_ss_2sm_collect<1>(d0, da, db0, idesc, k == 0 ? acc0 : 1u);
    mma_i8_ss_2sm_collect<2>(d1, da, db1, idesc, k == 0 ? acc0 : 1u);
  }
}
__device__ __forceinline__ void issue_kn_wide(uint32_t d0, uint32_t d1, uint32_t lo_a, uint32_t lo_b0, uint32_t lo_b1,
                                              uint32_t hi, uint32_t idesc, uint32_t acc0, int nk) {
  for (int k = 0; k < nk; ++k) {
    const uint64_t da = (static_cast<uint64_t>(hi) << 32) | (lo_a + k * (32 * kPanelBytes / 16));
    const uint64_t db0 = (static_cast<uint64_t>(hi) << 32) | (lo_b0 + k * (32 * kPanelBytes / 16));
    const uint64_t db1 = (static_cast<uint64_t>(hi) << 32) | (lo_b1 + k * (32 * kPanelBytes / 16));
    mma_i8_ss_2sm_collect<1>(d0, da, db0, idesc, k == 0 ? acc0 : 1u);
    mma_i8_ss_2sm_collect<2>(d1, da, db1, idesc, k == 0 ? acc0 : 1u);
  }
}

template <bool kPair>
__device__ __forceinline__ void issue_kn(uint32_t d, uint32_t lo_a, uint32_t lo_b, uint32_t hi, uint32_t idesc,
                                         uint32_t acc0, int nk) {
  for (int k = 0; k < nk; ++k) {
    const uint64_t da = (static_cast<uint64_t>(hi) << 32) | (lo_a + k * (32 * kPanelBytes / 16));
    const uint64_t db = (static_cast<uint64_t>(hi) << 32) | (lo_b + k * (32 * kPanelBytes / 16));
    if (kPair) mma_i8_ss_2sm(d, da, db, idesc, k == 0 ? acc0 : 1u);
    else       mma_i8_ss(d, da, db, idesc, k == 0 ? acc0 : 1u);
  }
}

// maps: the tensor maps of the input(s), [n_batch][3] (box heights 256 / 128 / 64 time rows); vis_list: the output of
// every integration of a batched launch (kBatch), else unused (p.vis).
}  // namespace corr
#include "xengine_i8_resident.cuh"
namespace corr {

template <bool kPair, bool kProbe, bool kPacked = false, bool kBatch = false>
__device__ __forceinline__ void xengine_i8_body(const CUtensorMap *maps, int2 *const *vis_list, const I8Params &p) {
  // All shared memory is dynamic (no static variables), so the window starts 1024-byte aligned as the
  // 128-byte swizzle needs: [stage ring][epilogue staging][mbarriers + TMEM base].
  extern __shared__ __align__(1024) uint8_t smem[];
  // 4-bit packed input (kPacked): TMA lands the packed boxes in a second ring (half the bytes) behind the
  // int8 ring; eight expand warps sign-extend the nibbles into the int8 ring in the MN-major SW128 layout.
  // Resident-A plans (CTA pairs, T <= 1152) put the A panel of the whole integration in front of the ring.
  const uint32_t a_bytes = (kPair && p.resident) ? static_cast<uint32_t>(p.a_sub) * kResSubBytes : 0;
  uint8_t *ring_base = smem + a_bytes;
  const uint32_t raw_stage_bytes = kPacked ? static_cast<uint32_t>(p.stage_bytes) / 2 : 0;
  uint8_t *raw = ring_base + static_cast<size_t>(p.stages) * p.stage_bytes;
  uint8_t *epi_stage = raw + static_cast<size_t>(p.stages) * raw_stage_bytes;
  uint64_t *full_bar = reinterpret_cast<uint64_t *>(epi_stage + kEpiWarps * kEpiWarpBytes);
  uint64_t *empty_bar = full_bar + kMaxStages;
  uint64_t *acc_full = empty_bar + kMaxStages;
  uint64_t *acc_empty = acc_full + 2;
  uint64_t *raw_full = acc_empty + 2;
  uint64_t *raw_empty = raw_full + kMaxStages;
  uint64_t *a_full = raw_empty + kMaxStages;  // resident-A plans: one pair of barriers per 128-row sub-stage of the A region
  uint64_t *a_empty = a_full + kResMaxSub;
  uint32_t &tmem_base_smem = *reinterpret_cast<uint32_t *>(a_empty + kResMaxSub);

  // programmatic dependent launch (single-CTA kernels): the next call's launch, barrier set-up and TMEM allocation may
  // overlap this call's tail; every role that touches global memory waits for the preceding grid first
  if (!kPair && !kBatch) griddep_launch_dependents();
  const int probe = kProbe ? p.probe : 0;  // diagnostics (-DCORR_DIAG builds only) compile away in the product
  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int n_rounds = (p.n_items + p.units - 1) / p.units;
  const int rank = kPair ? static_cast<int>(cluster_ctarank()) : 0;  // CTA within the pair; 0 issues the MMAs

  // Warp roles: epilogue = warps 0-7, TMA producers = 8 and 11, MMA issuer = 9, TMEM allocator = 10.  The single-thread
  // roles sit in the HIGHEST warps because the SMSP arbiter favours higher warp ids: they are the critical
  // path and must not queue behind eight busy epilogue warps.
  if (warp == kProducerWarp && lane == 0) {
    tma_prefetch_desc(&maps[0]);
    tma_prefetch_desc(&maps[1]);
    tma_prefetch_desc(&maps[2]);
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(&full_bar[s], kPacked ? kExpandWarps : 1);  // packed: the expand warps publish the int8 stage
      mbar_init(&empty_bar[s], 1);
      if (kPacked) {
        mbar_init(&raw_full[s], 1);
        mbar_init(&raw_empty[s], kExpandWarps);
      }
    }
    if (kPair)
      for (int g = 0; g < kResMaxSub; ++g) {
        mbar_init(&a_full[g], 1);
        mbar_init(&a_empty[g], 1);
      }
    for (int r = 0; r < 2; ++r) {
      mbar_init(&acc_full[r], 1);
      mbar_init(&acc_empty[r], kEpiWarps * (kPair ? 2 : 1));  // one arrive per epilogue warp (of both CTAs)
    }
    fence_mbar_init();
  }
  if (warp == kAllocWarp) { if (kPair) tmem_alloc_2sm(&tmem_base_smem, 512); else tmem_alloc(&tmem_base_smem, 512); }
  tc_fence_before();
  if (kPair) cluster_sync_all(); else __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;

  if (kPair && p.resident && (warp == kProducerWarp || warp == kProducerWarp2 || warp == kMmaWarp)) {
    // ===================================================================== resident-A plans: their own producers and issuer
    if (warp == kMmaWarp) resident_mma<kProbe>(p, smem, a_bytes, full_bar, empty_bar, acc_full, acc_empty, a_full, a_empty, tmem_base, n_rounds, rank);
    else resident_producer(p, maps, smem, a_bytes, full_bar, empty_bar, a_full, a_empty, n_rounds, rank, warp == kProducerWarp2);
  } else if (warp == kProducerWarp || warp == kProducerWarp2) {
    // ===================================================================== TMA producers
    // two warps walk the same schedule and take alternate stages: one thread cannot issue the boxes of a
    // stage (wait, expect_tx, up to 4 TMA instructions) as fast as the tensor pipe drains it
    const int pw = (warp == kProducerWarp) ? 0 : 1;
    int iter = 0;
    if (elect_one() && !(probe & 8)) {
      if (!kPair && !kBatch) griddep_wait();  // d_in may have been written by the preceding kernel of the stream
      const uint64_t pol = policy_evict_normal();
      const uint32_t full_leader = kPair ? mapa_u32(&full_bar[0], 0) : 0;
      int stage = 0;
      uint32_t phase = 0;
      long long w_empty = 0;  // diagnostics (probe bit 128): cycles this producer waited for a free stage
      I8Iter cur = iter_init(p);
      for (int r = 0; r < n_rounds; ++r, iter_next(p, cur)) {
        if (!iter_valid(p, cur)) continue;
        const I8Item it = decode_item(p, cur, rank);
        const CUtensorMap *map = maps + (kBatch ? 3 * cur.bi : 0) + it.map;
        const uint32_t panel_bytes = static_cast<uint32_t>(it.bk) * kPanelBytes;
        for (int t = it.t0; t < it.t1; t += it.bk, ++iter) {
          if ((iter & 1) != pw) {
            if (++stage == p.stages) { stage = 0; phase ^= 1; }
            continue;
          }
          if (kPacked) {
            // packed boxes {64 B, bk rows} land in the raw ring; the expand warps own the int8 ring
            mbar_wait(&raw_empty[stage], phase ^ 1);
            const uint32_t raw_panel = static_cast<uint32_t>(it.bk) * (kPanelBytes / 2);
            mbar_expect_tx(&raw_full[stage], raw_panel * it.n_load);
            uint8_t *rdst = raw + static_cast<size_t>(stage) * raw_stage_bytes;
            for (int l = 0; l < it.n_load; ++l) {
              const bool is_a = l >= it.nblk_load;
              const int x = (is_a ? it.xa : it.x0 + l * it.dx) >> 1;  // one byte per sample: half the offset
              tma_load_2d(rdst + l * raw_panel, map, &raw_full[stage], x, t, pol);
            }
            if (++stage == p.stages) { stage = 0; phase ^= 1; }
            continue;
          }
          long long tw = 0;
          if (kProbe && (probe & 128)) tw = clock64();
          mbar_wait(&empty_bar[stage], phase ^ 1);
          if (kProbe && (probe & 128)) w_empty += clock64() - tw;
          if (probe & 2) {
            if (rank == 0) mbar_arrive(&full_bar[stage]);
          } else {
            // pair mode: both CTAs' boxes complete on the LEADER's barrier, which expects the bytes of both
            if (rank == 0) mbar_expect_tx(&full_bar[stage], panel_bytes * it.n_load * (kPair ? 2 : 1));
            uint8_t *dst = ring_base + static_cast<size_t>(stage) * p.stage_bytes;
            const uint32_t bar2 = kPair ? full_leader + stage * 8 : 0;
            for (int l = 0; l < it.n_load; ++l) {
              const bool is_a = l >= it.nblk_load;
              const int x = is_a ? it.xa : it.x0 + l * it.dx;
              const int z = is_a ? it.za : it.z0 + l * it.dz;
              if (kPair) {
                if (p.turned) tma_load_3d_2sm(dst + l * panel_bytes, map, bar2, x, t, z, pol);
                else          tma_load_2d_2sm(dst + l * panel_bytes, map, bar2, x, t, pol);
              } else {
                if (p.turned) tma_load_3d(dst + l * panel_bytes, map, &full_bar[stage], x, t, z, pol);
                else          tma_load_2d(dst + l * panel_bytes, map, &full_bar[stage], x, t, pol);
              }
            }
          }
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
      }
      if (kProbe && (probe & 128) && p.diag_stats && rank == 0 && pw == 0)
        p.diag_stats[4 * (blockIdx.x >> (kPair ? 1 : 0)) + 3] = static_cast<unsigned long long>(w_empty);
    }
  } else if (warp == kMmaWarp) {
    // ===================================================================== MMA issuer
    // One elected thread (elect.sync, so that ptxas emits plain uniform-datapath code without a waterfall
    // loop around every UTCIMMA) walks the schedule.  Descriptor low words are advanced by plain adds
    // (all offsets are multiples of 16 B and the address field cannot carry into the LBO field below 256 KB).
    if (rank == 0 && elect_one()) {
      constexpr bool leader = true;
      int stage = 0;
      uint32_t phase = 0;
      uint32_t ring = 0;  // accumulator ring entries handed out so far
      constexpr uint32_t kIdesc128 = idesc_i8_mn(128, 128);
      constexpr uint32_t kIdesc256 = kPair ? idesc_i8_mn(256, 256) : idesc_i8_mn(128, 256);
      constexpr uint32_t kDescHi = static_cast<uint32_t>(((1024ull >> 4) | (1ull << 14) | (2ull << 29)));
      const uint32_t smem_lo = (smem_u32(ring_base) & 0x3FFFFu) >> 4;
      const uint32_t tmem_u = tmem_base;
      long long w_full = 0, w_acc = 0, t_begin = 0;  // diagnostics (probe bit 128): cycles spent waiting for loads / for TMEM
      if (kProbe && (probe & 128)) t_begin = clock64();
      I8Iter cur = iter_init(p);
      for (int r = 0; r < n_rounds; ++r, iter_next(p, cur)) {
        if (!iter_valid(p, cur)) continue;
        const I8Item it = decode_item(p, cur, 0);
        const int u_bk = it.bk;
        const int u_t0 = it.t0;
        const int u_t1 = it.t1;
        const int u_nblk = it.nblk;
        const uint32_t panel16 = static_cast<uint32_t>(u_bk) * (kPanelBytes / 16);  // panel bytes / 16
        const uint32_t a_off = static_cast<uint32_t>(it.a_slot) * panel16;
        const uint32_t lbo_field = (panel16 & 0x3FFFu) << 16;
        const int n_chunks = (u_nblk + 1) >> 1;
        long long tw = 0;
        if (kProbe && (probe & 128)) tw = clock64();
        if (!(probe & 4))
          for (int q = 0; q < n_chunks; ++q) mbar_wait(&acc_empty[(ring + q) & 1], (((ring + q) >> 1) & 1) ^ 1);
        if (kProbe && (probe & 128)) w_acc += clock64() - tw;
        tc_fence_after();
        const uint32_t d0 = tmem_u + (ring & 1) * kAccCols;        // chunk 0
        const uint32_t d1 = tmem_u + ((ring + 1) & 1) * kAccCols;  // chunk 1
        const uint32_t idesc0 = u_nblk >= 2 ? kIdesc256 : kIdesc128;
        for (int t = u_t0; t < u_t1; t += u_bk) {
          if (kProbe && (probe & 128)) tw = clock64();
          if (!(probe & 8)) mbar_wait(&full_bar[stage], phase);
          if (kProbe && (probe & 128)) w_full += clock64() - tw;
          if (!(kProbe && (probe & 64))) tc_fence_after();
          const uint32_t lo_stage = (smem_lo + static_cast<uint32_t>(stage) * (p.stage_bytes >> 4)) | lbo_field;
          const int nk = (min(u_bk, u_t1 - t) + 31) >> 5;  // K = 32 samples per MMA; TMA zero-fills past T
          const uint32_t acc0 = (t != u_t0) ? 1u : 0u;  // the first MMA of the slice overwrites the accumulator
          if (!(probe & 1)) {
            if (p.diag) {
              for (int b = 0; b < u_nblk; ++b) {
                const uint32_t dcol = ((b & 2) ? d1 : d0) + (b & 1) * 128;
                const uint32_t lo_b = lo_stage + b * panel16;
                if (nk == 2)      issue_k<2, false>(dcol, lo_b, lo_b, kDescHi, kIdesc128, acc0);
                else              issue_kn<false>(dcol, lo_b, lo_b, kDescHi, kIdesc128, acc0, nk);
              }
            } else {
              const uint32_t lo_a = lo_stage + a_off;
              if (kPair && u_nblk > 2 && p.collect) {  // 512-wide pair tile, A read once per k-step (collector reuse)
                const uint32_t lo_b1 = lo_stage + panel16;
                if (nk == 4) issue_k_wide<4>(d0, d1, lo_a, lo_stage, lo_b1, kDescHi, idesc0, acc0);
                else         issue_kn_wide(d0, d1, lo_a, lo_stage, lo_b1, kDescHi, idesc0, acc0, nk);
              } else {
              if (nk == 2)      issue_k<2, kPair>(d0, lo_a, lo_stage, kDescHi, idesc0, acc0);
              else if (nk == 4) issue_k<4, kPair>(d0, lo_a, lo_stage, kDescHi, idesc0, acc0);
              else if (nk == 8) issue_k<8, kPair>(d0, lo_a, lo_stage, kDescHi, idesc0, acc0);
              else              issue_kn<kPair>(d0, lo_a, lo_stage, kDescHi, idesc0, acc0, nk);
              if (kPair && u_nblk > 2) {  // 512-wide pair tile: second column half from smem slot 1 into chunk 1
                const uint32_t lo_b1 = lo_stage + panel16;
                if (nk == 4) issue_k<4, kPair>(d1, lo_a, lo_b1, kDescHi, idesc0, acc0);
                else         issue_kn<kPair>(d1, lo_a, lo_b1, kDescHi, idesc0, acc0, nk);
              }
              }
            }
          }
          if (leader && !(probe & 8)) {  // frees the stage (in both CTAs of a pair) when these MMAs retire
            if (kPair) mma_commit_2sm(&empty_bar[stage], 3); else mma_commit(&empty_bar[stage]);
          }
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
        if (leader)
          for (int q = 0; q < n_chunks; ++q) {
            if (kPair) mma_commit_2sm(&acc_full[(ring + q) & 1], 3); else mma_commit(&acc_full[(ring + q) & 1]);
          }
        ring += n_chunks;
      }
      if (kProbe && (probe & 128) && p.diag_stats) {
        unsigned long long *st = p.diag_stats + 4 * (blockIdx.x >> (kPair ? 1 : 0));
        st[0] = static_cast<unsigned long long>(clock64() - t_begin);
        st[1] = static_cast<unsigned long long>(w_full);
        st[2] = static_cast<unsigned long long>(w_acc);
      }
    }
  } else if (kPacked && warp >= kExpandWarp0) {
    // ===================================================================== expand warps (4-bit input)
    // raw ring -> int8 ring: each byte (low nibble Re, high nibble Im, two's complement, DESIGN
    // reading R18) becomes the int8 pair (16 Re, 16 Im), written in the MN-major 128-byte-swizzled operand
    // layout the TMA would have produced for int8 input.  A nibble moved to the top of its byte IS 16 x its
    // two's-complement value, so no sign extension is needed: the Gram sums come out 256 x too large, exactly,
    // and the epilogue shifts them right by 8 (p.out_shift).  |256 V| <= T * 2 * 128^2 still fits int32.
    const int et = threadIdx.x - kExpandWarp0 * 32;  // 0 .. 127
    int stage = 0;
    uint32_t phase = 0;
    I8Iter cur = iter_init(p);
    for (int r = 0; r < n_rounds; ++r, iter_next(p, cur)) {
      if (!iter_valid(p, cur)) continue;
      const I8Item it = decode_item(p, cur, rank);
      const uint32_t panel_bytes = static_cast<uint32_t>(it.bk) * kPanelBytes;
      const int n_chunks = it.n_load * it.bk * 4;  // 16-byte packed chunks of this stage
      const int sh = 31 - __clz(it.bk * 4);
      for (int t = it.t0; t < it.t1; t += it.bk) {
        mbar_wait(&raw_full[stage], phase);       // packed bytes have landed
        mbar_wait(&empty_bar[stage], phase ^ 1);  // the int8 slot has been consumed by the MMAs
        const uint8_t *src = raw + static_cast<size_t>(stage) * raw_stage_bytes;
        uint8_t *dst = ring_base + static_cast<size_t>(stage) * p.stage_bytes;
        for (int idx = et; idx < n_chunks; idx += kExpandWarps * 32) {
          const int l = idx >> sh;            // panel (bk * 4 chunks each, a power of two)
          const int rem = idx & ((1 << sh) - 1);
          const int k = rem >> 2, q = rem & 3;
          const uint4 w = *reinterpret_cast<const uint4 *>(src + l * (panel_bytes / 2) + k * 64 + q * 16);
          const uint32_t in[4] = {w.x, w.y, w.z, w.w};
          uint32_t out[8];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const uint32_t re = (in[u] << 4) & 0xF0F0F0F0u;  // 16 * Re in every byte
            const uint32_t im = in[u] & 0xF0F0F0F0u;         // 16 * Im in every byte
            out[2 * u] = __byte_perm(re, im, 0x5140);      // re0 im0 re1 im1
            out[2 * u + 1] = __byte_perm(re, im, 0x7362);  // re2 im2 re3 im3
          }
          uint8_t *row = dst + l * panel_bytes + k * kPanelBytes;
          const int sw = k & 7;  // 128-byte swizzle: 16-byte chunk index XOR (row mod 8)
          *reinterpret_cast<uint4 *>(row + (((2 * q) ^ sw) << 4)) = make_uint4(out[0], out[1], out[2], out[3]);
          *reinterpret_cast<uint4 *>(row + (((2 * q + 1) ^ sw) << 4)) = make_uint4(out[4], out[5], out[6], out[7]);
        }
        fence_proxy_async();  // generic-proxy writes -> visible to the tensor core's (async-proxy) reads
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(&full_bar[stage]);
          mbar_arrive(&raw_empty[stage]);
        }
        if (++stage == p.stages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp < kEpiWarps && !(probe & 4)) {
    // ===================================================================== epilogue
    if (!kPair && !kBatch) griddep_wait();  // d_vis may still be written (or read) by the preceding kernel of the stream
    const int ew = warp & 3;         // TMEM lanes 32*ew .. 32*ew+31 (a warp may only touch its own quadrant)
    const int hsel = warp >> 2;        // which half (64 TMEM columns) of every block this warp folds
    constexpr int kShift = kPacked ? 8 : 0;
    if (p.n_slices > 1 || p.accumulate || ((kPair || kBatch || kPacked) && p.mix_cut))
      i8_epilogue<1, kShift, kBatch, !kPacked, kPair>(p, vis_list, tmem_base, epi_stage + warp * kEpiWarpBytes,
                                                      acc_full, acc_empty, n_rounds, ew, hsel, lane, rank, kPair, probe);
    else if (!kPair && !kBatch && !kPacked && p.mix_cut)  // mixed plan: whole groups store, their sliced neighbours reduce-add
      i8_epilogue<2, kShift, kBatch, !kPacked, kPair>(p, vis_list, tmem_base, epi_stage + warp * kEpiWarpBytes,
                                                      acc_full, acc_empty, n_rounds, ew, hsel, lane, rank, kPair, probe);
    else
      i8_epilogue<0, kShift, kBatch, !kPacked, kPair>(p, vis_list, tmem_base, epi_stage + warp * kEpiWarpBytes,
                                                      acc_full, acc_empty, n_rounds, ew, hsel, lane, rank, kPair, probe);
  }

  tc_fence_before();
  if (kPair) cluster_sync_all(); else __syncthreads();
  if (warp == kAllocWarp) {
    tc_fence_after();
    if (kPair) tmem_dealloc_2sm(tmem_base, 512); else tmem_dealloc(tmem_base, 512);
  }
}

__global__ void __launch_bounds__(kI8Threads, 1)
xengine_i8_kernel(const __grid_constant__ I8Maps tm, const __grid_constant__ I8Params p) {
#ifdef CORR_DIAG
  if (p.probe) { xengine_i8_body<false, true>(tm.m, nullptr, p); return; }
#endif
  xengine_i8_body<false, false>(tm.m, nullptr, p);
}

// One launch over n_batch integrations (corr_xengine_batch; "process large batches of data per call",
// 32 blocks of spectra per GPU call): the schedule walk carries the integration index, which selects
// the tensor maps and the output of the item.  All SMs stay busy on inputs too small to fill the chip alone (c1).
__global__ void __launch_bounds__(kI8Threads, 1)
xengine_i8_batch_kernel(const __grid_constant__ I8Batch bt, const __grid_constant__ I8Params p) {
  xengine_i8_body<false, false, false, true>(&bt.m[0][0], bt.vis, p);
}

// 4-bit packed input (the paper's "1-byte mode"): 20 warps, the last eight expand nibbles to int8.
__global__ void __launch_bounds__(kI4Threads, 1)
xengine_i4_kernel(const __grid_constant__ I8Maps tm, const __grid_constant__ I8Params p) {
  xengine_i8_body<false, false, true>(tm.m, nullptr, p);
}

// CTA pairs: tcgen05.mma.cta_group::2, M = 256 (one 128-row panel per CTA), each CTA stages half of B.
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kI8Threads, 1)
xengine_i8_pair_kernel(const __grid_constant__ I8Maps tm, const __grid_constant__ I8Params p) {
#ifdef CORR_DIAG
  if (p.probe) { xengine_i8_body<true, true>(tm.m, nullptr, p); return; }
#endif
  xengine_i8_body<true, false>(tm.m, nullptr, p);
}

}  // namespace corr
