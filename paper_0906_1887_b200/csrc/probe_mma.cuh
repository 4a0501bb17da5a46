// probe_mma.cuh -- DIAGNOSTICS (built only with -DCORR_DIAG into libcorr_diag.so; include/corr_diag.h):
// tcgen05.mma.kind::i8 issue-rate probe (the int8 tensor peak is
// not in MEASURED_PEAKS.json, so it is measured here).  One CTA per SM; one thread issues `iters`
// back-to-back MMAs on zero-filled shared-memory operands (values do not matter for timing) into
// two alternating TMEM accumulators, then commits and waits.  No global traffic at all.
#pragma once
#include "ptx_sm100.cuh"

namespace corr {

struct ProbeParams {
  int iters;
  int m, n;        // MMA shape (M = 64 | 128, N multiple of 16 up to 256), K = 32
  int fill;        // 0: zero operands, 1: pseudo-random bytes (power draw differs, timing should not)
  int mn_major;    // 1: both operands MN-major (what the fused corner turn produces); 0: K-major
  unsigned long long *cycles;  // [2*gridDim.x]: elapsed SM cycles, elapsed globaltimer ns of the issue loop
};

__global__ void __launch_bounds__(128, 1) probe_mma_kernel(const ProbeParams p) {
  extern __shared__ __align__(1024) uint8_t psmem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(psmem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ __align__(8) uint64_t done_bar;
  __shared__ uint32_t tmem_base_smem;
  // operands: A at 0 (16 KB = 128 x 128 B), B at 16 KB (32 KB = 256 x 128 B)
  for (int i = threadIdx.x; i < 48 * 1024 / 16; i += blockDim.x) {
    const uint32_t v = (p.fill & 1) ? (i * 2654435761u + blockIdx.x * 40503u) : 0u;
    reinterpret_cast<uint4 *>(smem)[i] = make_uint4(v, v * 3u + 1u, v ^ 0x9E3779B9u, v * 7u);
  }
  if (threadIdx.x == 0) {
    mbar_init(&done_bar, 1);
    fence_mbar_init();
  }
  fence_proxy_async();
  if (threadIdx.x < 32) tmem_alloc(&tmem_base_smem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  if (threadIdx.x == 0) {
    const uint32_t a0 = smem_u32(smem), b0 = a0 + 16 * 1024;
    uint32_t idesc = idesc_i8_mn(p.m, p.n);
    if (!p.mn_major) idesc &= ~((1u << 15) | (1u << 16));
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    const long long t0 = clock64();
    for (int it = 0; it < p.iters; ++it) {
      const int k = it & 3;
      // MN-major: 32 k-rows of 128 B per MMA -> +4096 B; K-major: 32 B of each 128-B row -> +32 B
      uint32_t off = p.mn_major ? k * 4096 : k * 32;
      if (p.fill & 4) off = (it % 40) * 4096;  // walk over 160 KB of shared memory instead of 16 KB
      const uint32_t lbo = (p.fill & 32) ? 8 * 1024 : 16 * 1024;  // second 128-byte block of an N = 256 operand
      if (p.fill & 32) off = (it & 1) * 4096;
      const uint64_t a_desc = smem_desc_mn_sw128(a0 + off, lbo, 1024);
      const uint64_t b_desc = (p.fill & 2) ? a_desc : smem_desc_mn_sw128(b0 + off, lbo, 1024);
      uint32_t d = tmem_base + ((it >> 2) & 1) * 256;
      if (p.fill & 8) d = tmem_base + (it & 3) * 128;           // D rotates over four 128-column blocks
      if (p.fill & 16) d = tmem_base + (it & 1) * 256;          // D alternates between two 256-column chunks
      mma_i8_ss(d, a_desc, b_desc, idesc, it >= 8);
    }
    mma_commit(&done_bar);
    mbar_wait(&done_bar, 0);
    const long long t1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    p.cycles[2 * blockIdx.x] = static_cast<unsigned long long>(t1 - t0);
    p.cycles[2 * blockIdx.x + 1] = g1 - g0;
  }
  tc_fence_before();
  __syncthreads();
  if (threadIdx.x < 32) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

// FP32 FMA issue-rate probe (the "alu" roofline denominator of the float X-engine): every thread runs `iters`
// rounds of 16 independent register-resident FMAs -- scalar FFMA (packed = 0) or packed fma.rn.f32x2 (packed = 1,
// the instruction xengine_f32_n64_kernel uses).  No memory traffic inside the loop.
struct ProbeFfmaParams {
  int iters, packed;
  float b, c;                  // runtime multiplier / addend (keeps the chain from being folded)
  float *sink;                 // [gridDim.x * blockDim.x]
  unsigned long long *cycles;  // [2 * gridDim.x]: SM cycles, globaltimer ns of the loop (thread 0 of each CTA)
};
__global__ void __launch_bounds__(1024, 1) probe_ffma_kernel(const ProbeFfmaParams p) {
  extern __shared__ uint8_t ffma_pad[];  // 200 KB of dynamic shared memory: exactly one CTA per SM
  if (p.iters < 0) ffma_pad[threadIdx.x] = 0;
  float2 a[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) a[k] = make_float2(threadIdx.x * 1e-3f + k, blockIdx.x * 1e-3f - k);
  const float2 b2 = make_float2(p.b, p.b), c2 = make_float2(p.c, p.c);
  unsigned long long g0 = 0, g1 = 0;
  if (threadIdx.x == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
  const long long t0 = clock64();
  if (p.packed) {
    for (int it = 0; it < p.iters; ++it) {
#pragma unroll
      for (int k = 0; k < 8; ++k)
        asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(reinterpret_cast<unsigned long long &>(a[k]))
                     : "l"(reinterpret_cast<const unsigned long long &>(b2)), "l"(reinterpret_cast<const unsigned long long &>(c2)));
    }
  } else {
    for (int it = 0; it < p.iters; ++it) {
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[k].x) : "f"(p.b), "f"(p.c));
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[k].y) : "f"(p.b), "f"(p.c));
      }
    }
  }
  const long long t1 = clock64();
  if (threadIdx.x == 0) {
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    p.cycles[2 * blockIdx.x] = static_cast<unsigned long long>(t1 - t0);
    p.cycles[2 * blockIdx.x + 1] = g1 - g0;
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += a[k].x + a[k].y;
  p.sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace corr
