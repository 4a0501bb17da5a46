// xengine_i8_epilogue.cuh -- step a3: fold the real Gram blocks in TMEM into packed complex
// visibilities (included from xengine_i8_kernel.cuh).
//
// One epilogue warp owns 32 TMEM lanes = 16 inputs i (lane 2r holds the Re row of input r, lane
// 2r+1 the Im row) and one half (64 TMEM columns = 32 inputs j) of every block:
//   tcgen05.ld 32 columns -> one shfl.xor 1 per column pair gives Re V_ij on the even lane and
//   Im V_ij on the odd lane -> staged in shared memory as [16 rows][32 complex] (row stride 264 / 272 B)
//   -> shipped one packed-triangle ROW at a time:
//        whole integrations : 32 lanes x 8 B = 256 contiguous bytes per store instruction;
//        time-sliced items  : one cp.reduce.async.bulk.add.s32 per row (integer reduce-add in L2)
//                             for the 16-byte aligned body + <= 2 scalar atomics for the edges.
// Software pipeline inside the warp: the TMEM load of the warp's NEXT half block of the same accumulator is
// issued as soon as the fold of the current one has consumed the registers, so it runs under the current half
// block's shared-memory round trip and global stores; and the accumulator is handed back to the MMA issuer
// right after the warp's LAST tcgen05.ld of it has completed, before that half block is folded and stored.
// The accumulator is therefore held for two loads and one fold + store instead of two of each (T = 1000 tiles
// are only 4096 tensor cycles long: the epilogue of tile n must be out of TMEM before tile n + 2 starts).
// The TMEM buffer is handed back with a RELAXED mbarrier arrive: a releasing arrive made the warp
// wait (MEMBAR) for all of its visibility stores to land, which serialised epilogue and DRAM writes.
#pragma once

namespace corr {

constexpr int kEpiRowBytes = 272;  // 32 complex int32 + one alignment slot, 16-byte multiple
constexpr int kEpiRowBytesPlain = 264;  // plain-store path: 66-word stride, conflict-free staging writes
constexpr int kEpiWarpBytes = 16 * kEpiRowBytes;  // 4352 B per epilogue warp

// What one warp does with one 128-column block of an accumulator (all fields warp-uniform).
struct EpiTask {
  bool valid;     // this warp has visibilities in the block (not above the diagonal / another channel / past N_I)
  bool diag_blk;  // diagonal block: keep j <= i only
  int chan_w;     // channel of the warp's rows
  int i0_w;       // first of the warp's 16 inputs i
  int j0;         // first of the 32 inputs j of the warp's half block
};

__device__ __forceinline__ EpiTask epi_task(const I8Params &p, const I8Item &it, int b, int ew, int hsel) {
  EpiTask t;
  t.valid = false; t.diag_blk = true; t.chan_w = 0; t.i0_w = 0; t.j0 = 0;
  const int Jb = it.J0 + (it.jperm ? (((b & 1) << 1) | (b >> 1)) : b);  // column panel held by block b
  if (!p.diag && Jb > it.I) return t;  // block above the diagonal (pair tiles on the diagonal)
  int j_blk0;
  if (p.diag) {
    const int panel = it.J0 + b;
    t.chan_w = p.pair_mode ? 2 * panel + (ew >> 1) : panel;
    t.i0_w = p.pair_mode ? (ew & 1) * 16 : ew * 16;
    j_blk0 = 0;
    t.diag_blk = true;
  } else {
    t.chan_w = it.chan;
    t.i0_w = it.I * 64 + ew * 16;
    j_blk0 = Jb * 64;
    t.diag_blk = Jb == it.I;
  }
  const bool warp_ok = (t.chan_w < p.n_chan) && (t.i0_w < p.n_inputs);
  bool ok;
  if (p.pair_mode) { t.j0 = 0; ok = (hsel == (ew >> 1)); }
  else { t.j0 = j_blk0 + hsel * 32; ok = (t.j0 < p.n_inputs) && (!t.diag_blk || hsel * 32 <= ew * 16 + 15); }
  t.valid = ok && warp_ok;
  return t;
}

// kAtomic: reduce-add into d_vis (time-sliced or accumulating items) instead of plain stores.  kShift: 8 for
// 4-bit input (operands are 16 x the samples), else 0.  Both are compile-time so that the plain-store path is
// the bare minimum per value: one SHFL, one IMAD (v + sgn * partner), one conflict-free STS.
// kPipe: software-pipelined TMEM loads (needs ~50 more registers; off in the 640-thread 4-bit kernel).
// kAtomic: 0 = plain stores, 1 = every item reduce-adds (time slices, accumulate mode), 2 = mixed plan: only the items
// that are time slices reduce-add (I8Item::sliced), whole-integration items store.
template <int kAtomic, int kShift, bool kBatch, bool kPipe, bool kResident>
__device__ __forceinline__ void i8_epilogue(const I8Params &p, int2 *const *vis_list, uint32_t tmem_base, uint8_t *stage_buf,
                                            uint64_t *acc_full, uint64_t *acc_empty, int n_rounds, int ew,
                                            int hsel, int lane, int rank, bool pair, int probe) {
  const int part = lane & 1;  // 0: row 2i (Re row of input i), 1: row 2i+1 (Im row)
  const int rl = lane >> 1;   // which of the warp's 16 inputs this lane pair holds
  const int sgn = part ? -1 : 1;  // Re = G[2i][2j] + G[2i+1][2j+1], Im = G[2i+1][2j] - G[2i][2j+1]
  // staging row stride: 272 B keeps rows 16-byte aligned for the bulk reduce-add; 264 B (66 words) makes the
  // 4-byte staging writes of the 32 lanes hit 32 different banks on the plain-store path
  constexpr int kRowB = kAtomic ? kEpiRowBytes : kEpiRowBytesPlain;
  bool any_atomic = false;
  int *st_w = reinterpret_cast<int *>(stage_buf) + rl * (kRowB / 4) + part;
  uint32_t ring = 0;
  I8Iter cur = iter_init(p);
  for (int r = 0; r < n_rounds; ++r, iter_next(p, cur)) {
    if (!iter_valid(p, cur)) continue;
    const int n_sub = (kResident && p.resident) ? res_n_tiles(p, cur) : 1;  // resident-A plans: an item is a unit of tiles
    for (int sub = 0; sub < n_sub; ++sub) {
    const I8Item it = (kResident && p.resident) ? res_item(p, cur, res_tile(p, cur, sub), rank) : decode_item(p, cur, rank);
    int2 *const vis = kBatch ? vis_list[cur.bi] : p.vis;  // output of this item's integration
    const bool atomic = kAtomic == 1 || (kAtomic == 2 && it.sliced);
    any_atomic = any_atomic || atomic;
    const int n_chunks = (it.nblk + 1) >> 1;
    for (int q = 0; q < n_chunks; ++q) {
      const uint32_t e = ring + q;
      // the (at most two) blocks of this accumulator in which the warp has work
      const int nb_here = min(2, it.nblk - 2 * q);
      const EpiTask tk0 = epi_task(p, it, 2 * q, ew, hsel);
      EpiTask tk1 = tk0;
      tk1.valid = false;
      if (nb_here > 1) tk1 = epi_task(p, it, 2 * q + 1, ew, hsel);
      mbar_wait(&acc_full[e & 1], (e >> 1) & 1);
      tc_fence_after();
      const uint32_t tchunk = tmem_base + (static_cast<uint32_t>(ew * 32) << 16) + (e & 1) * kAccCols + hsel * 64;
      bool released = false;
      auto release = [&]() {  // every tcgen05.ld of this ring entry by this warp has completed (wait::ld): hand it back
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          if (pair) mbar_arrive_cluster(mapa_u32(&acc_empty[e & 1], 0));  // the leader's MMA thread owns the wait
          else      mbar_arrive_relaxed(&acc_empty[e & 1]);
        }
        released = true;
      };
      // both 32-column loads of a half block are in flight before the single wait
      uint32_t v0[32], v1[32];
      auto load = [&](int bb) {
        tmem_ld_32x32(tchunk + bb * 128, v0);
        tmem_ld_32x32(tchunk + bb * 128 + 32, v1);
      };
      // one half block: fold, stage, ship.  `next`: the block whose load is issued once the registers are free
      // (-1: none, the accumulator is handed back instead).
      auto half_block = [&](const EpiTask &tk, int next) {
        // this lane pair's row: input i_row, its first packed element and how many columns it keeps
        const int i_row = tk.i0_w + rl;
        // sliced (accumulating) items ship rows with bulk reduce-add: 16-byte aligned pairs in global memory must
        // be 16-byte aligned in shared memory too, so a row is shifted by one slot when its first element is odd
        const int par = atomic ? static_cast<int>((static_cast<long long>(tk.chan_w) * p.n_baselines +
                                                    i_row * (i_row + 1) / 2 + tk.j0) & 1) : 0;
        int *st_row = st_w + par * 2;
        if (kAtomic && lane < 16) bulk_wait_read_all();  // earlier bulk reduces have read the staging buffer
        __syncwarp();  // the previous half block has been read out of the staging buffer
        tmem_ld_wait_regs(v0);
        tmem_ld_wait_regs(v1);
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) {
          const int o0 = __shfl_xor_sync(0xffffffffu, static_cast<int>(v0[2 * jj + 1]), 1);
          const int o1 = __shfl_xor_sync(0xffffffffu, static_cast<int>(v1[2 * jj + 1]), 1);
          int a0 = o0 * sgn + static_cast<int>(v0[2 * jj]);
          int a1 = o1 * sgn + static_cast<int>(v1[2 * jj]);
          if (kShift) { a0 >>= kShift; a1 >>= kShift; }  // 4-bit input: sums are exact multiples of 256
          // (Im of an autocorrelation needs no special case: G is computed in exact integers and is
          //  symmetric, so G[2i+1][2i] - G[2i][2i+1] is exactly 0)
          st_row[jj * 2] = a0;                          // even lane: Re -> .x, odd lane: Im -> .y
          st_row[(16 + jj) * 2] = a1;
        }
        // the registers are free again: start the load of the warp's next half block of this accumulator, or, if
        // this was the last one, give the accumulator back before the shared-memory round trip and the stores
        if (next < 0) release();
        else if (kPipe) load(next);
        if (atomic) fence_proxy_async();  // generic-proxy writes -> visible to the bulk (async) proxy
        __syncwarp();
        if (atomic) {
          if (lane < 16 && !(probe & 16)) {
            // lane r ships row r: elements j0 .. j0+cnt-1 of input i = i0_w + r
            const int i = tk.i0_w + lane;
            const int cnt = (i < p.n_inputs) ? min(32, min(i, p.n_inputs - 1) - tk.j0 + 1) : 0;
            if (cnt > 0) {
              const long long e0 = static_cast<long long>(tk.chan_w) * p.n_baselines + i * (i + 1) / 2 + tk.j0;
              const int sh = static_cast<int>(e0 & 1);
              const int2 *srow = reinterpret_cast<const int2 *>(stage_buf + lane * kRowB) + sh;  // element 0
              int2 *grow = vis + e0;
              int head = sh;                         // one leading element if e0 is odd
              int body = (cnt - head) & ~1;          // aligned pairs
              if (cnt < head) { head = cnt; body = 0; }
              const int tail = cnt - head - body;    // one trailing element
              if (head) {
                const int2 x = srow[0];
                put_vis<true>(grow, x.x, x.y);
              }
              if (body) {
                bulk_reduce_add_s32(grow + head, srow + head, body * 8);
              }
              if (tail) {
                const int2 x = srow[cnt - 1];
                put_vis<true>(grow + cnt - 1, x.x, x.y);
              }
            }
            bulk_commit();
          }
        } else if (!(probe & 16)) {
          // one packed-triangle row per instruction: 32 lanes x 8 B = 256 contiguous bytes.  N_I is a multiple
          // of 32, so every row and column of the half block exists; only diagonal blocks need the j <= i test.
          const int j = tk.j0 + lane;
          const int i = tk.i0_w;
          int2 *row = vis + (static_cast<long long>(tk.chan_w) * p.n_baselines + i * (i + 1) / 2 + j);
          const int2 *src = reinterpret_cast<const int2 *>(stage_buf) + lane;
          int2 val[16];
#pragma unroll
          for (int rr = 0; rr < 16; ++rr) val[rr] = src[rr * (kRowB / 8)];  // 16 independent loads
          if (!tk.diag_blk) {
#pragma unroll
            for (int rr = 0; rr < 16; ++rr) {
              *row = val[rr];
              row += i + rr + 1;  // next row of the triangle starts i+1 elements further on
            }
          } else {
#pragma unroll
            for (int rr = 0; rr < 16; ++rr) {
              if (j <= i + rr) *row = val[rr];
              row += i + rr + 1;
            }
          }
        }
        if (!kPipe && next >= 0) load(next);
      };
      if (tk0.valid) {
        load(0);
        half_block(tk0, tk1.valid ? 1 : -1);
      } else if (tk1.valid) {
        load(1);
      }
      if (tk1.valid) half_block(tk1, -1);
      if (!released) release();  // the warp had nothing to read in this accumulator
    }
    ring += n_chunks;
    }
  }
  if (kAtomic && any_atomic && lane < 16) bulk_wait_all();  // all reduce-adds performed before the CTA retires
}

}  // namespace corr
