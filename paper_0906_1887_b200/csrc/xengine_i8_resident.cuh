// xengine_i8_resident.cuh -- "resident A" plans of the CTA-pair kernel (included from xengine_i8_kernel.cuh).
//
// Short integrations with many inputs (config c4: N_I = 1024, T = 1000) are bound by the SM's 128 B/cycle
// shared-memory datapath, not by the tensor pipe: per 256 x 256 tile and k-step a CTA's MMA reads 8 KB of
// operands, TMA writes 8 KB of new operands, and the epilogue moves another 3.5 x its 64 KB of output per tile
// (DESIGN.md section 7).  The A operand of a CTA -- its 128-row panel over the WHOLE integration, 128 B x T
// <= 128 KB -- fits in shared memory when T <= 1152 (144 KB, beside a 3-stage B ring; 4 stages up to T = 1024), so a pair keeps it there and walks every column tile of its
// row pair with it: A is written to shared memory once per ROW (R + 1 tiles) instead of once per tile, the
// diagonal tile (whose B operand is the A panel itself) loads nothing at all, and the L2 -> SM traffic of c4
// drops from 2 x 128 KB to (128 + 128 / 4.5) KB per tile on average.
//
//   schedule item = unit (channel, u): row pairs R1 = pp - 1 - u and R2 = u, pp + 1 tiles in every unit
//   A region      = a_sub sub-stages of 128 time rows (16 KB), barriers a_full[g] / a_empty[g]:
//                   loaded before the first tile of a row, released by the MMAs of the row's LAST (diagonal)
//                   tile sub-stage by sub-stage, so the next row's A streams in under that tile
//   B ring        = stages x 16 KB (one 128-row box of the CTA's half of B per stage), as in the other plans
// Warp kProducerWarp feeds the B ring, warp kProducerWarp2 the A region, warp kMmaWarp issues; the epilogue is the
// common one (it walks the same tiles through res_tile / res_item).
#pragma once

namespace corr {

constexpr int kResMaxSub = 9;            // 9 x 128 = 1152 time rows at most (a 3-stage B ring fits beside them)
constexpr int kResSubBytes = 128 * 128;  // one sub-stage / one ring stage: 128 time rows of a 128-byte panel

__device__ __forceinline__ void resident_producer(const I8Params &p, const CUtensorMap *maps, uint8_t *smem, uint32_t a_bytes,
                                                  uint64_t *full_bar, uint64_t *empty_bar, uint64_t *a_full,
                                                  uint64_t *a_empty, int n_rounds, int rank, bool a_side) {
  if (!elect_one()) return;
  const uint64_t pol = policy_evict_normal();
  const CUtensorMap *map = maps + 1;  // box {128 B, 128 time rows}
  const uint32_t full_leader = mapa_u32(&full_bar[0], 0);
  const uint32_t a_full_leader = mapa_u32(&a_full[0], 0);
  uint8_t *ring = smem + a_bytes;
  int stage = 0;
  uint32_t phase = 0;
  uint32_t rows_done = 0;  // rows this pair has started: the phase of the A sub-stage barriers
  I8Iter cur = iter_init(p);
  for (int r = 0; r < n_rounds; ++r, iter_next(p, cur)) {
    if (!iter_valid(p, cur)) continue;
    const int n_sub = res_n_tiles(p, cur);
    for (int sub = 0; sub < n_sub; ++sub) {
      const ResTile tl = res_tile(p, cur, sub);
      const I8Item it = res_item(p, cur, tl, rank);
      if (a_side) {
        if (!tl.first) continue;
        // the row's A panel: sub-stage g is free once the previous row's diagonal tile has consumed it
        for (int g = 0; g < p.a_sub; ++g) {
          mbar_wait(&a_empty[g], (rows_done & 1) ^ 1);
          if (rank == 0) mbar_expect_tx(&a_full[g], 2 * kResSubBytes);  // both CTAs' boxes complete on the leader's barrier
          tma_load_2d_2sm(smem + g * kResSubBytes, map, a_full_leader + g * 8, it.xa, g * 128, pol);
        }
        ++rows_done;
      } else {
        if (tl.diag) continue;  // the diagonal tile multiplies the resident panel by itself
        for (int g = 0; g < p.a_sub; ++g) {
          mbar_wait(&empty_bar[stage], phase ^ 1);
          if (rank == 0) mbar_expect_tx(&full_bar[stage], 2 * kResSubBytes);
          tma_load_2d_2sm(ring + stage * kResSubBytes, map, full_leader + stage * 8, it.x0, g * 128, pol);
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
      }
    }
  }
}

template <bool kProbe>
__device__ __forceinline__ void resident_mma(const I8Params &p, uint8_t *smem, uint32_t a_bytes, uint64_t *full_bar,
                                             uint64_t *empty_bar, uint64_t *acc_full, uint64_t *acc_empty,
                                             uint64_t *a_full, uint64_t *a_empty, uint32_t tmem_base, int n_rounds,
                                             int rank) {
  if (rank != 0 || !elect_one()) return;
  constexpr uint32_t kIdesc = idesc_i8_mn(256, 256);
  constexpr uint32_t kDescHi = static_cast<uint32_t>(((1024ull >> 4) | (1ull << 14) | (2ull << 29)));
  constexpr uint32_t kSub16 = kResSubBytes / 16;
  const uint32_t lbo_field = (kSub16 & 0x3FFFu) << 16;
  const uint32_t a_lo0 = ((smem_u32(smem) & 0x3FFFFu) >> 4) | lbo_field;
  const uint32_t ring_lo0 = ((smem_u32(smem + a_bytes) & 0x3FFFFu) >> 4) | lbo_field;
  int stage = 0;
  uint32_t phase = 0, ring = 0, rows_done = 0;
  long long w_full = 0, w_acc = 0, t_begin = 0, tw = 0;
  if (kProbe && (p.probe & 128)) t_begin = clock64();
  I8Iter cur = iter_init(p);
  for (int r = 0; r < n_rounds; ++r, iter_next(p, cur)) {
    if (!iter_valid(p, cur)) continue;
    const int n_sub = res_n_tiles(p, cur);
    for (int sub = 0; sub < n_sub; ++sub) {
      const ResTile tl = res_tile(p, cur, sub);
      if (kProbe && (p.probe & 128)) tw = clock64();
      mbar_wait(&acc_empty[ring & 1], ((ring >> 1) & 1) ^ 1);
      if (kProbe && (p.probe & 128)) w_acc += clock64() - tw;
      tc_fence_after();
      const uint32_t d = tmem_base + (ring & 1) * kAccCols;
      for (int g = 0; g < p.a_sub; ++g) {
        if (kProbe && (p.probe & 128)) tw = clock64();
        if (tl.first) mbar_wait(&a_full[g], rows_done & 1);
        if (!tl.diag) mbar_wait(&full_bar[stage], phase);
        if (kProbe && (p.probe & 128)) w_full += clock64() - tw;
        tc_fence_after();
        const uint32_t lo_a = a_lo0 + g * kSub16;
        const uint32_t lo_b = tl.diag ? lo_a : ring_lo0 + stage * kSub16;
        const int nk = (min(128, p.n_time - g * 128) + 31) >> 5;  // K = 32 samples per MMA; TMA zero-fills past T
        const uint32_t acc0 = g ? 1u : 0u;
        if (nk == 4) issue_k<4, true>(d, lo_a, lo_b, kDescHi, kIdesc, acc0);
        else         issue_kn<true>(d, lo_a, lo_b, kDescHi, kIdesc, acc0, nk);
        if (!tl.diag) {  // frees the B stage in both CTAs when these MMAs retire
          mma_commit_2sm(&empty_bar[stage], 3);
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        } else {         // last tile of the row: the A sub-stage may be refilled with the next row's panel
          mma_commit_2sm(&a_empty[g], 3);
        }
      }
      mma_commit_2sm(&acc_full[ring & 1], 3);
      ++ring;
      if (tl.diag) ++rows_done;
    }
  }
  if (kProbe && (p.probe & 128) && p.diag_stats) {
    unsigned long long *st = p.diag_stats + 4 * (blockIdx.x >> 1);
    st[0] = static_cast<unsigned long long>(clock64() - t_begin);
    st[1] = static_cast<unsigned long long>(w_full);
    st[2] = static_cast<unsigned long long>(w_acc);
    st[3] = 0;
  }
}

}  // namespace corr
