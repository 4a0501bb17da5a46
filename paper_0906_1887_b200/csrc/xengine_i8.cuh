// xengine_i8.cuh -- int8 complex X-engine on tcgen05 (steps a1-fused, a2, a3, a6 of DESIGN.md).
//
// Per channel c the CMAC is the real Gram matrix G = Y^T Y of the
// (T x 2N) int8 matrix Y whose row t is the raw sample vector [Re x_0, Im x_0, Re x_1, ...]
// exactly as it lies in d_in[t][c][:].  G is cut into 128-row "panels" (64 inputs each; for
// N_I = 32 one panel is two adjacent channels).  A work item accumulates up to four 128x128
// blocks of G over a time slice in TMEM (int32) and folds them to complex visibilities
//   Re V_ij = G[2i][2j] + G[2i+1][2j+1],  Im V_ij = G[2i+1][2j] - G[2i][2j+1].
// Two item kinds:
//   slab  (N_I >= 128): row panel I x column panels J0, J0+1 (<= I) of one channel: one 128x256
//                       accumulator, so the two TMEM halves double-buffer items (epilogue overlaps MMA);
//   diag  (N_I <= 64) : the diagonal blocks of up to four ADJACENT channels (or channel pairs), so
//                       that each time row is fetched as one 512-byte contiguous run (HBM-friendly).
// The schedule (descendant of the paper's constant-memory pair table) lives in the
// kernel-parameter constant bank and is decoded with uniform arithmetic: everything the MMA issuer
// touches stays in uniform registers, which is what lets one thread issue at the tensor-pipe rate.
//
// Warp roles (384 threads, 1 CTA/SM, persistent):
//   warps 8, 11  TMA producers (one thread each, alternate stages): box {128 B along the chan*input
//            axis, bk time rows}, SWIZZLE_128B.
//            This strided box load IS the corner turn: it lands as the
//            canonical MN-major operand tile, so the input is read from HBM exactly once.
//   warp 9   MMA issuer (one thread): tcgen05.mma.kind::i8, M=128, N=128|256, K=32.
//   warp 10  TMEM allocator.
//   warps 0-7 epilogue (two per TMEM lane quadrant, one per half block): tcgen05.ld, 2x2 fold via
//            shfl.xor 1, packed-triangle stores (or integer
//            red.add when an integration is split into time slices; integer sums are exact and
//            order-independent, so the result stays bit-exact).
#pragma once
#include "ptx_sm100.cuh"

namespace corr {

constexpr int kI8Threads = 384;    // 4 control warps + 8 epilogue warps
constexpr int kEpiWarps = 8;
constexpr int kExpandWarp0 = 12, kExpandWarps = 8;  // 4-bit input only (640-thread launch)
constexpr int kI4Threads = 640;
constexpr int kProducerWarp = 8, kMmaWarp = 9, kAllocWarp = 10, kProducerWarp2 = 11;
constexpr int kPanelBytes = 128;  // bytes of the chan*input axis per panel = 64 complex int8 samples
constexpr int kAccCols = 256;     // TMEM columns per accumulator ring entry (two 128-column blocks)
constexpr int kMaxStages = 8;
constexpr int kMaxKinds = 1056;   // slab kinds per channel at N_I = 4096 (64 panels, column pairs)
constexpr int kMaxBatch = 64;     // integrations per launch of the batched entry point (corr_xengine_batch)

struct I8Params {
  // ---- schedule (uniform) ----
  int n_groups;      // diag: groups of gsize panels; slab: channels
  int gsize;         // diag: adjacent panels per item (4, or 2 / 1 for small problems)
  int n_kinds;       // items per group (diag: 1)
  int n_slices;      // time slices per integration (> 1 => results are accumulated with red.add)
  int slice_len;     // samples per slice (multiple of 64 when n_slices > 1)
  int n_batch;       // integrations per launch (1 except for xengine_i8_batch_kernel)
  int n_items;       // n_groups * n_kinds * n_slices * n_batch
  int rot;           // per-round rotation of the CTA -> item map (spreads the kinds over the CTAs)
  int dq[2], dr[2];  // (grid + rot) and rot, each split as quotient / remainder by n_kinds (host-computed)
  int diag;          // item kind
  int pair2;         // 1: CTA pairs (cta_group::2): an item is a 256 x 256 tile, 128 rows per CTA
  int units;         // schedule walkers: CTAs, or CTA pairs when pair2
  int n_panels;      // diag: total panels along the chan*input axis; slab: panels per channel
  // ---- problem ----
  int n_time, n_inputs, n_chan;
  int pair_mode;     // N_I == 32: one panel = two adjacent channels
  int stages, stage_bytes;
  int turned;        // 0: d_in is [T][C][2N] (2-D maps); 1: scratch is [G][T][W] (3-D maps)
  int probe;         // diagnostics only (corr_set_probe)
  unsigned long long *diag_stats;  // diagnostics only (probe bit 128): [unit][4] = kernel cycles, MMA waits for loads, MMA waits for TMEM, producer waits for a stage
  int out_shift;     // 8 for 4-bit input (operands are 16 x the samples), else 0
  int accumulate;    // 1: add this integration into d_vis instead of overwriting it
  int mix_full, mix_cut, mix_len;  // diag plans with more groups than CTAs: whole groups + sliced left-over groups (decode_item)
  int resident;      // 1: CTA pairs keep their A panel of the WHOLE integration in shared memory (T <= 1152) and walk all
                     //    column tiles of a row pair with it; an item is then a unit of two row pairs (xengine_i8_resident.cuh)
  int a_sub;         // resident: 128-row sub-stages of the A region (ceil(T / 128))
  int collect;       // 1: 512-wide pair tiles issue their two MMAs per k-step with A-collector reuse
  long long n_baselines;
  int2 *vis;
  unsigned short kinds[kMaxKinds];  // slab: I | (J0 / 2) << 6 | (nblk - 1) << 11; pair: Ip | (J0 / 2) << 6 | wide << 11
};

struct I8Item {
  int t0, t1;        // time slice
  int nblk;          // 128-column blocks (1..4)
  int nblk_load;     // B panels this CTA fetches (= nblk, except in pair mode)
  int jperm;         // 1: TMEM column block b holds column panel J0 + {0, 2, 1, 3}[b] (512-wide pair tiles)
  int n_load;        // panels fetched per k-step (nblk, +1 when A is not one of the B panels)
  int a_slot;        // slab: smem slot of the A panel; diag: unused (A = B = slot b)
  int x0, z0;        // TMA coordinates of block 0 (block b at x0 + b*dx, z0 + b*dz)
  int dx, dz;
  int xa, za;        // TMA coordinates of a separate A panel
  int bk, map;       // time rows per stage and the tensor map (box height) that goes with it
  int chan, I, J0;   // slab: channel, row panel, first column panel; diag: first panel in J0
  bool sliced;       // mixed plans: this item is a time slice (reduce-add) and not a whole integration (plain stores)
};

// Tensor maps of one input buffer (box heights 256 / 128 / 64 time rows) and the per-integration arguments of a
// batched launch: one launch walks a schedule that spans n_batch integrations (the paper's remedy for small
// transfers: "process large batches of data per call"; 32 blocks per call).
struct I8Maps { CUtensorMap m[3]; };
struct I8Batch {
  CUtensorMap m[kMaxBatch][3];
  int2 *vis[kMaxBatch];
};

// Position of a CTA in the schedule: item g = ((bi * n_slices + s) * n_groups + grp) * n_kinds + k, walked WITHOUT
// divisions (additions, compares and constant-bank reads only), so that ptxas keeps the whole walk
// and everything decoded from it in uniform registers.  Round r of CTA b takes item
// r * grid + (b + r * rot) mod grid.
struct I8Iter {
  int bi, s, grp, k, b;
};
__device__ __forceinline__ void iter_carry(const I8Params &p, I8Iter &c) {
  if (c.k >= p.n_kinds) { c.k -= p.n_kinds; ++c.grp; }
  while (c.grp >= p.n_groups) { c.grp -= p.n_groups; ++c.s; }
  while (c.s >= p.n_slices && c.bi < p.n_batch) { c.s -= p.n_slices; ++c.bi; }
}
__device__ __forceinline__ I8Iter iter_init(const I8Params &p) {
  I8Iter c;
  c.b = static_cast<int>(blockIdx.x) >> p.pair2;
  c.bi = 0; c.s = 0; c.grp = 0; c.k = c.b;
  while (c.k >= p.n_kinds) { c.k -= p.n_kinds; ++c.grp; }
  iter_carry(p, c);
  return c;
}
__device__ __forceinline__ void iter_next(const I8Params &p, I8Iter &c) {
  c.b += p.rot;
  int w = 0;
  if (c.b >= p.units) { c.b -= p.units; w = 1; }  // wrapped: g advances by rot only
  c.k += p.dr[w];
  c.grp += p.dq[w];
  iter_carry(p, c);
}
__device__ __forceinline__ bool iter_valid(const I8Params &p, const I8Iter &c) { return c.bi < p.n_batch; }

// Decode of a schedule position (all inputs are kernel parameters / uniform counters).
__device__ __forceinline__ I8Item decode_item(const I8Params &p, const I8Iter &c, int rank = 0) {
  I8Item it;
  it.sliced = false;
  const int s = c.s, grp = c.grp, k = c.k;
  it.t0 = s * p.slice_len;
  it.t1 = min(p.n_time, it.t0 + p.slice_len);
  const int row = 2 * p.n_inputs;  // bytes per (t, c)
  if (p.diag) {
    // mixed plans (more groups than CTAs): the first mix_full group slots are whole integrations, the rest are the
    // mix_slices time slices of the mix_cut left-over groups, slice-major (the walk itself has n_slices = 1)
    int g = grp;
    if (p.mix_cut && g >= p.mix_full) {
      int u = g - p.mix_full, sl = 0;
      while (u >= p.mix_cut) { u -= p.mix_cut; ++sl; }
      g = p.mix_full + u;
      it.sliced = true;
      it.t0 = sl * p.mix_len;
      it.t1 = min(p.n_time, it.t0 + p.mix_len);
    }
    const int panel0 = g * p.gsize;
    it.nblk = min(p.gsize, p.n_panels - panel0);
    it.n_load = it.nblk;
    it.a_slot = 0;
    it.chan = 0; it.I = 0; it.J0 = panel0;
    if (p.turned) { it.x0 = 0; it.z0 = panel0; it.dx = 0; it.dz = 1; }
    else          { it.x0 = panel0 * kPanelBytes; it.z0 = 0; it.dx = kPanelBytes; it.dz = 0; }
    it.xa = 0; it.za = 0;
  } else if (p.pair2) {
    // CTA `rank` of the pair owns row panel 2*Ip + rank.  A 256-wide tile (wide = 0) puts column panel
    // J0 + rank in this CTA (its half of B).  A 512-wide tile (wide = 1: two M=256,N=256 MMAs per k-step,
    // all 512 TMEM columns) puts panels J0 + 2*rank, J0 + 2*rank + 1 here -- ADJACENT panels, so each
    // time row is one 256..384-byte run in HBM -- which makes the TMEM column blocks hold the panels
    // J0 + {0, 2, 1, 3}.  The A panel always gets its own slot so that both CTAs use the same offsets.
    const unsigned kd = p.kinds[k];
    const int Ip = kd & 63;
    const int wide = (kd >> 11) & 1;
    it.I = 2 * Ip + rank; it.J0 = ((kd >> 6) & 31) * 2; it.nblk = wide ? 4 : 2;
    it.jperm = wide;
    it.chan = grp;
    const int xc = p.turned ? 0 : grp * row;
    it.z0 = p.turned ? grp : 0; it.dx = kPanelBytes; it.dz = 0;
    it.xa = xc + it.I * kPanelBytes; it.za = it.z0;
    if (wide) {
      it.nblk_load = 2; it.n_load = 3; it.a_slot = 2;
      it.x0 = xc + (it.J0 + 2 * rank) * kPanelBytes;
    } else {
      const bool same = (2 * Ip == it.J0);  // diagonal tile: the CTA's A panel is its B half
      it.nblk_load = 1; it.n_load = same ? 1 : 2; it.a_slot = same ? 0 : 1;
      it.x0 = xc + (it.J0 + rank) * kPanelBytes;
    }
  } else {
    const unsigned kd = p.kinds[k];
    it.I = kd & 63; it.J0 = ((kd >> 6) & 31) * 2; it.nblk = ((kd >> 11) & 1) + 1;
    it.chan = grp;
    const bool a_in_b = it.I < it.J0 + it.nblk;
    it.n_load = it.nblk + (a_in_b ? 0 : 1);
    it.a_slot = a_in_b ? (it.I - it.J0) : it.nblk;
    const int xc = p.turned ? 0 : grp * row;
    it.x0 = xc + it.J0 * kPanelBytes; it.z0 = p.turned ? grp : 0; it.dx = kPanelBytes; it.dz = 0;
    it.xa = xc + it.I * kPanelBytes; it.za = it.z0;
  }
  if (!p.pair2) { it.nblk_load = it.nblk; it.jperm = 0; }
  // the tallest box (256 / 128 / 64 time rows) whose n_load panels fit one stage
  if (it.n_load * 256 * kPanelBytes <= p.stage_bytes)      { it.bk = 256; it.map = 0; }
  else if (it.n_load * 128 * kPanelBytes <= p.stage_bytes) { it.bk = 128; it.map = 1; }
  else                                                     { it.bk = 64;  it.map = 2; }
  return it;
}

// Resident-A plans: the tiles of one schedule item (a unit = row pairs R1 = pp-1-u and R2 = u of one channel, so that
// every unit has pp + 1 tiles), in the order every role walks them: row R1 first, each row's column tiles J0 = 0, 2, ...
// with the diagonal tile (J0 = 2R, whose B operand IS the resident A panel) last.
struct ResTile {
  int R, J0;
  bool first, diag;  // first / last (diagonal) tile of its row
};
__device__ __forceinline__ int res_n_tiles(const I8Params &p, const I8Iter &c) {
  const int pp = (p.n_panels + 1) >> 1, u = c.k, r1 = pp - 1 - u;
  return (r1 + 1) + (r1 != u ? u + 1 : 0);
}
__device__ __forceinline__ ResTile res_tile(const I8Params &p, const I8Iter &c, int sub) {
  const int pp = (p.n_panels + 1) >> 1, u = c.k, r1 = pp - 1 - u;
  ResTile t;
  if (sub <= r1) { t.R = r1; t.J0 = 2 * sub; }
  else           { t.R = u;  t.J0 = 2 * (sub - r1 - 1); }
  t.first = t.J0 == 0;
  t.diag = t.J0 == 2 * t.R;
  return t;
}
__device__ __forceinline__ I8Item res_item(const I8Params &p, const I8Iter &c, const ResTile &t, int rank) {
  I8Item it;
  it.sliced = false;
  it.t0 = 0; it.t1 = p.n_time;
  it.nblk = 2; it.nblk_load = 1; it.jperm = 0; it.n_load = t.diag ? 0 : 1; it.a_slot = 0;
  it.chan = c.grp; it.I = 2 * t.R + rank; it.J0 = t.J0;
  it.dx = kPanelBytes; it.dz = 0; it.z0 = 0; it.za = 0;
  const int xc = c.grp * 2 * p.n_inputs;
  it.x0 = xc + (t.J0 + rank) * kPanelBytes;
  it.xa = xc + it.I * kPanelBytes;
  it.bk = 128; it.map = 1;
  return it;
}

template <bool kAtomic>
__device__ __forceinline__ void put_vis(int2 *dst, int re, int im) {
  if (kAtomic) {
    atomicAdd(&dst->x, re);
    if (im != 0) atomicAdd(&dst->y, im);
  } else {
    *dst = make_int2(re, im);
  }
}

}  // namespace corr

#include "xengine_i8_kernel.cuh"
