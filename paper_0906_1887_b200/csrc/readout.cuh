// readout.cuh -- read-out side of the accumulators:
//   normalize_kernel : out[k] = sums[k] / count  (int32 / float / int64 / double sums -> float)
//                      "the accumulators are ... divided by the number of times they were updated";
//   fold_wide_kernel : acc[k] += vis[k] with acc twice as wide (int32 -> int64, float -> double): the
//                      persistent accumulators of a long accumulation (every batch is ADDED),
//                      promoted at batch boundaries so that no number of batches can overflow or lose bits.
// One pass each, 16-byte vectors, grid-stride.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace corr {

enum { kSumI32 = 0, kSumF32 = 1, kSumI64 = 2, kSumF64 = 3 };

struct NormParams {
  const void *vis;
  float *out;
  long long n;     // scalars (2 per visibility); a multiple of 4
  float inv_count;
  double inv_count_d;
  int kind;        // kSum*
};
__global__ void __launch_bounds__(256) normalize_kernel(const NormParams p) {
  const long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
  for (long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; k < p.n / 4; k += stride) {
    float4 o;
    if (p.kind == kSumI32) {
      const int4 v = reinterpret_cast<const int4 *>(p.vis)[k];
      o = make_float4(v.x * p.inv_count, v.y * p.inv_count, v.z * p.inv_count, v.w * p.inv_count);
    } else if (p.kind == kSumF32) {
      const float4 v = reinterpret_cast<const float4 *>(p.vis)[k];
      o = make_float4(v.x * p.inv_count, v.y * p.inv_count, v.z * p.inv_count, v.w * p.inv_count);
    } else if (p.kind == kSumI64) {
      // sums beyond 2^24 do not fit a float mantissa: divide in double, round once
      const longlong2 a = reinterpret_cast<const longlong2 *>(p.vis)[2 * k], b = reinterpret_cast<const longlong2 *>(p.vis)[2 * k + 1];
      o = make_float4(static_cast<float>(static_cast<double>(a.x) * p.inv_count_d), static_cast<float>(static_cast<double>(a.y) * p.inv_count_d),
                      static_cast<float>(static_cast<double>(b.x) * p.inv_count_d), static_cast<float>(static_cast<double>(b.y) * p.inv_count_d));
    } else {
      const double2 a = reinterpret_cast<const double2 *>(p.vis)[2 * k], b = reinterpret_cast<const double2 *>(p.vis)[2 * k + 1];
      o = make_float4(static_cast<float>(a.x * p.inv_count_d), static_cast<float>(a.y * p.inv_count_d),
                      static_cast<float>(b.x * p.inv_count_d), static_cast<float>(b.y * p.inv_count_d));
    }
    reinterpret_cast<float4 *>(p.out)[k] = o;
  }
}

struct FoldParams {
  const void *vis;  // int32 or float sums of one batch
  void *acc;        // int64 or double accumulators
  long long n;      // scalars; a multiple of 4
  int is_int;
};
__global__ void __launch_bounds__(256) fold_wide_kernel(const FoldParams p) {
  const long long stride = static_cast<long long>(gridDim.x) * blockDim.x;
  for (long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; k < p.n / 4; k += stride) {
    if (p.is_int) {
      const int4 v = reinterpret_cast<const int4 *>(p.vis)[k];
      longlong2 *a = reinterpret_cast<longlong2 *>(p.acc) + 2 * k;
      longlong2 a0 = a[0], a1 = a[1];
      a0.x += v.x; a0.y += v.y; a1.x += v.z; a1.y += v.w;
      a[0] = a0; a[1] = a1;
    } else {
      const float4 v = reinterpret_cast<const float4 *>(p.vis)[k];
      double2 *a = reinterpret_cast<double2 *>(p.acc) + 2 * k;
      double2 a0 = a[0], a1 = a[1];
      a0.x += v.x; a0.y += v.y; a1.x += v.z; a1.y += v.w;
      a[0] = a0; a[1] = a1;
    }
  }
}

}  // namespace corr
