// phs_devutil.cuh -- small device helpers shared by the CTA and cluster kernels.
#pragma once
#include <cuda_runtime.h>

namespace phs {

constexpr double kQuantum = 1.0 / 1048576.0;  // 2^-20 byte/s (reading R-FX)
constexpr double kInf = __builtin_huge_val();

// rate quanta -> byte/s: round-to-nearest conversion, exact power-of-two scale
__device__ __forceinline__ double rate_of(long long rq) { return __ll2double_rn(rq) * kQuantum; }

// a5: fair share of a link = floor(cap_rem / n), exact 64-bit integer division
__device__ __forceinline__ long long fair_share(long long cap_rem, int n) {
  return n == 1 ? cap_rem : cap_rem / (long long)n;
}

__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }

// non-negative doubles order like their bit patterns
__device__ __forceinline__ double warp_min(double v) {
  long long b = __double_as_longlong(v);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const long long x = __shfl_xor_sync(0xffffffffu, b, o);
    b = x < b ? x : b;
  }
  return __longlong_as_double(b);
}

}  // namespace phs
