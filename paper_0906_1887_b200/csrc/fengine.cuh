// fengine.cuh -- the F-stage in front of the float X-engine: unpack + batched 128-point
// complex-to-complex transform (PAPER.md:77-78 steps 1 and 2; "converting to floating-point format
// and putting the samples into N_I arrays of length N_C"; "the FFT is N_C channels in input and
// output").
//
//   X[b][k][i] = sum_n x[b][n][i] exp(-2 pi i k n / 128)      (forward, unnormalised, natural channel order)
//
// raw voltages x: [batch][128 samples][N_I] complex int8 (input index fastest, the aggregator's order,
// PAPER.md:71); spectra X: [batch][128 channels][N_I] float2 -- exactly the X-engine's [time][chan][input].
// Both have the input index fastest, so the paper's unpack TRANSPOSE (and its non-coalesced reads,
// PAPER.md:103) disappears: the transform runs down the columns of a 128 x N_I matrix, one input per lane,
// every global access a contiguous run along the input axis.  HBM-bound (2 B in, 8 B out, ~35 flop per
// sample), so the design goal is one pass over HBM and little shared-memory traffic:
//   128 = 16 x 8 (n = 8 n1 + n2, k = k1 + 16 k2), two passes, each entirely in registers:
//   pass 1  warp n2 loads x[8 n1 + n2] (n1 = 0..15) straight from global memory, 16-point transform over n1,
//           twiddle W_128^(n2 k1), one shared-memory write                          [8 warps x 32 inputs]
//   pass 2  thread (k1, input) reads its 8 values, 8-point transform over n2, stores X[k1 + 16 k2] straight
//           to global memory (32 lanes x 8 B = 256 contiguous bytes per store)
// so each sample crosses shared memory once (8 B written, 8 B read).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace corr {

constexpr int kFftN = 128;
constexpr int kFftTile = 32;      // inputs per CTA (one per lane)
constexpr int kFftThreads = 256;  // 8 warps = the 8 residues n2

struct FftParams {
  const int8_t *raw;  // [n_batch][128][n_inputs][2] int8 pairs, or [n_batch][128][n_inputs] bytes (4+4-bit mode)
  float2 *spec;       // [n_batch][128][n_inputs]
  int n_batch, n_inputs, tiles_per_batch;
};

__constant__ float2 c_tw128[kFftN];  // exp(-2 pi i m / 128), filled by corr_fstage_create (float64 -> float32)

// Complex add / subtract as ONE packed instruction (add.f32x2 / sub.f32x2, sm_100): the transform is mostly
// complex additions and the FP32 pipes, not HBM, were the limit with scalar FADDs.
__device__ __forceinline__ float2 cadd(float2 a, float2 b) {
  float2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(reinterpret_cast<unsigned long long &>(r))
      : "l"(reinterpret_cast<const unsigned long long &>(a)), "l"(reinterpret_cast<const unsigned long long &>(b)));
  return r;
}
__device__ __forceinline__ float2 csub(float2 a, float2 b) {
  float2 r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(reinterpret_cast<unsigned long long &>(r))
      : "l"(reinterpret_cast<const unsigned long long &>(a)), "l"(reinterpret_cast<const unsigned long long &>(b)));
  return r;
}
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
  return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x);
}
__device__ __forceinline__ float2 mul_mi(float2 a) { return make_float2(a.y, -a.x); }  // a * (-i)

// 4-point forward transform, in place, natural order out
__device__ __forceinline__ void fft4(float2 &x0, float2 &x1, float2 &x2, float2 &x3) {
  const float2 t0 = cadd(x0, x2), t1 = csub(x0, x2), t2 = cadd(x1, x3), d = csub(x1, x3);
  x0 = cadd(t0, t2); x2 = csub(t0, t2);
  x1 = make_float2(t1.x + d.y, t1.y - d.x);  // t1 + (-i) d
  x3 = make_float2(t1.x - d.y, t1.y + d.x);  // t1 - (-i) d
}

// 8-point forward transform: v[n] -> v[k], natural order
__device__ __forceinline__ void fft8(float2 (&v)[8]) {
  constexpr float h = 0.70710678118654752440f;
  fft4(v[0], v[2], v[4], v[6]);  // even samples -> E[0..3] in v[0], v[2], v[4], v[6]
  fft4(v[1], v[3], v[5], v[7]);  // odd samples  -> O[0..3] in v[1], v[3], v[5], v[7]
  const float2 o0 = v[1];
  const float2 o1 = make_float2(h * (v[3].x + v[3].y), h * (v[3].y - v[3].x));   // O1 * (1 - i)/sqrt2
  const float2 o2 = mul_mi(v[5]);                                                // O2 * (-i)
  const float2 o3 = make_float2(h * (v[7].y - v[7].x), -h * (v[7].x + v[7].y));  // O3 * (-1 - i)/sqrt2
  const float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
  v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
  v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
  v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
  v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
}

// 16-point forward transform: v[n] -> v[k], natural order (16 = 4 x 4: n = 4 a + r, k = k1 + 4 k2)
__device__ __forceinline__ void fft16(float2 (&v)[16]) {
  constexpr float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;  // cos, sin(pi / 8)
  constexpr float h = 0.70710678118654752440f;
#pragma unroll
  for (int r = 0; r < 4; ++r) fft4(v[r], v[4 + r], v[8 + r], v[12 + r]);  // over a: y[r][k1] in v[4 k1 + r]
  // twiddles W_16^(r k1) = exp(-2 pi i r k1 / 16)
  v[4 * 1 + 1] = cmul(v[4 * 1 + 1], make_float2(c1, -s1));   // m = 1
  v[4 * 2 + 1] = cmul(v[4 * 2 + 1], make_float2(h, -h));     // m = 2
  v[4 * 3 + 1] = cmul(v[4 * 3 + 1], make_float2(s1, -c1));   // m = 3
  v[4 * 1 + 2] = cmul(v[4 * 1 + 2], make_float2(h, -h));     // m = 2
  v[4 * 2 + 2] = mul_mi(v[4 * 2 + 2]);                       // m = 4
  v[4 * 3 + 2] = cmul(v[4 * 3 + 2], make_float2(-h, -h));    // m = 6
  v[4 * 1 + 3] = cmul(v[4 * 1 + 3], make_float2(s1, -c1));   // m = 3
  v[4 * 2 + 3] = cmul(v[4 * 2 + 3], make_float2(-h, -h));    // m = 6
  v[4 * 3 + 3] = cmul(v[4 * 3 + 3], make_float2(-c1, s1));   // m = 9
#pragma unroll
  for (int k1 = 0; k1 < 4; ++k1) fft4(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);  // over r
  // now X[k1 + 4 k2] sits in v[4 k1 + k2]: transpose the 4 x 4 index to natural order
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = a + 1; b < 4; ++b) {
      const float2 t = v[4 * a + b];
      v[4 * a + b] = v[4 * b + a];
      v[4 * b + a] = t;
    }
}

// kPacked: the paper's "1-byte mode": one byte per complex sample, low nibble Re, high nibble Im,
// 4-bit two's complement (DESIGN reading R18) -- half the raw bytes over PCIe and HBM, same transform.
template <bool kPacked>
__device__ __forceinline__ void fengine_body(const FftParams &p) {
  __shared__ float2 z[kFftN * kFftTile];  // [n2][k1][lane], 32 KB
  const int lane = threadIdx.x & 31;
  const int w = threadIdx.x >> 5;  // pass 1: n2; pass 2: k1 (and k1 + 8)
  // CTA = (batch, input tile), tile fastest: the tiles of one batch run side by side, so that the 256-byte
  // row pieces they write meet in L2 / the same DRAM pages.  Element offsets fit 32 bits (corr_fstage_create).
  const uint32_t ni = static_cast<uint32_t>(p.n_inputs);
  const uint32_t b = blockIdx.x / static_cast<uint32_t>(p.tiles_per_batch);
  const uint32_t tile = blockIdx.x - b * static_cast<uint32_t>(p.tiles_per_batch);
  const uint32_t base = b * (kFftN * ni) + tile * kFftTile + lane;

  // ---- pass 1: unpack (int8 -> float) + 16-point transforms over n1 for residue n2 = w
  {
    float2 v[16];
    if (kPacked) {
      const uint8_t *src = reinterpret_cast<const uint8_t *>(p.raw) + (base + w * ni);
      uint8_t raw[16];
#pragma unroll
      for (int n1 = 0; n1 < 16; ++n1) raw[n1] = src[8u * n1 * ni];  // all 16 loads in flight
      // a nibble n is the value (n ^ 8) - 8; (n ^ 8) placed in the mantissa of 2^23 is the float 8388608 + (n ^ 8)
#pragma unroll
      for (int n1 = 0; n1 < 16; ++n1) {
        const uint32_t u = static_cast<uint32_t>(raw[n1]) ^ 0x88u;
        const float2 m = make_float2(__uint_as_float(0x4B000000u | (u & 15u)), __uint_as_float(0x4B000000u | (u >> 4)));
        v[n1] = csub(m, make_float2(8388616.0f, 8388616.0f));
      }
    } else {
      const char2 *src = reinterpret_cast<const char2 *>(p.raw) + (base + w * ni);
      char2 raw[16];
#pragma unroll
      for (int n1 = 0; n1 < 16; ++n1) raw[n1] = src[8u * n1 * ni];  // all 16 loads in flight
      // unpack ("converting to floating-point format") without the quarter-rate I2F: the byte u = x ^ 0x80
      // placed in the mantissa of 2^23 is the float 8388608 + u; subtracting 8388736 leaves x exactly
#pragma unroll
      for (int n1 = 0; n1 < 16; ++n1) {
        const uint32_t u = (static_cast<uint32_t>(static_cast<uint8_t>(raw[n1].x)) |
                            (static_cast<uint32_t>(static_cast<uint8_t>(raw[n1].y)) << 8)) ^ 0x8080u;
        const float2 m = make_float2(__uint_as_float(__byte_perm(u, 0x4B000000u, 0x7440)),
                                     __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7441)));
        v[n1] = csub(m, make_float2(8388736.0f, 8388736.0f));
      }
    }
    fft16(v);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
      const float2 y = k1 == 0 ? v[0] : cmul(v[k1], c_tw128[w * k1]);  // W_128^(n2 k1), warp-uniform index
      z[(w * 16 + k1) * kFftTile + lane] = y;
    }
  }
  __syncthreads();
  // ---- pass 2: 8-point transforms over n2 for k1 = w and w + 8; X[k1 + 16 k2] straight to global memory
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    const int k1 = w + 8 * half;
    float2 v[8];
#pragma unroll
    for (int n2 = 0; n2 < 8; ++n2) v[n2] = z[(n2 * 16 + k1) * kFftTile + lane];
    fft8(v);
    float2 *dst = p.spec + (base + k1 * ni);
#pragma unroll
    for (int k2 = 0; k2 < 8; ++k2) dst[16u * k2 * ni] = v[k2];
  }
}

__global__ void __launch_bounds__(kFftThreads, 4) fengine_kernel(const FftParams p) { fengine_body<false>(p); }
__global__ void __launch_bounds__(kFftThreads, 4) fengine_ci4_kernel(const FftParams p) { fengine_body<true>(p); }

}  // namespace corr
