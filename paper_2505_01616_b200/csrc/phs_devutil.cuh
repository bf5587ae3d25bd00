// phs_devutil.cuh -- small device helpers shared by the CTA and cluster kernels.
#pragma once
#include <cuda_runtime.h>

#include "phs_device.h"

namespace phs {

constexpr double kQuantum = 1.0 / 1048576.0;  // 2^-20 byte/s (reading R-FX)
constexpr double kInf = __builtin_huge_val();

// rate quanta -> byte/s: round-to-nearest conversion, exact power-of-two scale
__device__ __forceinline__ double rate_of(long long rq) { return __ll2double_rn(rq) * kQuantum; }

// a5: fair share of a link = floor(cap_rem / n), EXACT.  Two double-precision quotient estimates, each followed by
// an exact 64-bit remainder, then an integer correction: whatever the rounding of the estimates, the loop invariant
// q*n + r == cap_rem (64-bit integer arithmetic) makes the result the true floor.  The reciprocal comes from the
// fp32 reciprocal unit plus one Newton step (relative error ~2^-46), which keeps the first estimate within 2^16 of
// the quotient and the second within 1; that is much shorter than a double-precision division.  cap_rem >= 0, n >= 1.
__device__ __forceinline__ long long fair_share(long long cap_rem, int n) {
  if (n == 1) return cap_rem;
  const double dn = (double)n;
  double inv;
  if (n < (1 << 24)) {
    inv = (double)__frcp_rn((float)n);
    inv = inv * (2.0 - dn * inv);
  } else {
    inv = 1.0 / dn;
  }
  long long q = __double2ll_rz(__ll2double_rz(cap_rem) * inv);
  long long r = cap_rem - q * (long long)n;
  const long long q2 = __double2ll_rz(__ll2double_rn(r) * inv);
  q += q2;
  r -= q2 * (long long)n;
  while (r < 0) {
    --q;
    r += n;
  }
  while (r >= n) {
    ++q;
    r -= n;
  }
  return q;
}

__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }

// Throughput history (optional, off the hot path: not inlined): the flow at output position `flow` changes its rate
// to `rq` quanta at time `now`, in the unit's event `ev`.
static __device__ __noinline__ void append_history(HistRec *hist, unsigned long long *hist_n, long long hist_cap, double now,
                                            long long rq, uint32_t flow, uint32_t ev) {
  const unsigned long long i = atomicAdd(hist_n, 1ull);
  if (i < (unsigned long long)hist_cap) {
    HistRec h;
    h.t = now;
    h.rate = rate_of(rq);
    h.flow = flow;
    h.ev = ev;
    hist[i] = h;
  }
}

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
