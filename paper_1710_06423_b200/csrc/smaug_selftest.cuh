// smaug_selftest.cuh -- on-device exactness check of the branch-free division helpers of smaug_device.cuh
// (ddiv, drcp, ratio_div, kappa_ratio) against the compiler's own IEEE-754 `/` on seeded operands.  Every stage
// kernel's bit-identity with the oracle rests on these helpers returning the correctly rounded quotient on the
// operand ranges the kernels feed them; tests/test_gpu_division.py calls this through the C ABI
// (smaug_selftest_division) so that the claim in DESIGN.md section 4 is reproducible from committed files.
#pragma once
#include "smaug_device.cuh"

namespace smaug {

__device__ __forceinline__ unsigned long long xorshift64(unsigned long long& s) {
  s ^= s << 13; s ^= s >> 7; s ^= s << 17;
  return s;
}

// a double with a random 52-bit mantissa (the low `zero_bits` bits cleared) and binary exponent uniform in
// [exp_lo, exp_hi]; exponents below -1022 give denormals (built by scaling, exact)
__device__ __forceinline__ double draw(unsigned long long& s, int exp_lo, int exp_hi, int zero_bits) {
  const unsigned long long r = xorshift64(s);
  const unsigned long long mant = ((r >> 12) >> zero_bits) << zero_bits;
  const int e = exp_lo + (int)((xorshift64(s) >> 33) % (unsigned)(exp_hi - exp_lo + 1));
  if (e >= -1022) return __longlong_as_double((long long)(((unsigned long long)(e + 1023) << 52) | mant));
  const double m = __longlong_as_double((long long)((1023ULL << 52) | mant));      // [1, 2)
  return (m * 0x1p-500) * __longlong_as_double((long long)((unsigned long long)(e + 500 + 1023) << 52));
}

// counts[0..3]: mismatches of ddiv(a, b) vs a / b, drcp(b) vs 1.0 / b, ratio_div(m3, m1) vs m3 / m1 and
// kappa_ratio(m3, m1, cv) vs (m1 > 0 ? cv * (m3 / m1) : 0) on ratio-like operands m3 = m1 * 2^[-30, 2] (clamped to
// m3 <= 4 m1, mantissas with trailing zeros as differences of nearby numbers have; one draw in 16 has m1 = m3 = 0,
// one in 16 has m3 = 0 alone); counts[4]: draws per test.
__global__ void division_selftest_kernel(int exp_lo, int exp_hi, unsigned long long seed, int draws_per_thread,
                                         unsigned long long* counts) {
  unsigned long long s = seed * 0x9E3779B97F4A7C15ULL + (unsigned long long)(blockIdx.x * blockDim.x + threadIdx.x) * 2654435761ULL + 1ULL;
  for (int k = 0; k < 8; ++k) xorshift64(s);
  unsigned long long bad0 = 0, bad1 = 0, bad2 = 0, bad3 = 0;
  for (int k = 0; k < draws_per_thread; ++k) {
    const double a = draw(s, exp_lo, exp_hi, 0), b = draw(s, exp_lo, exp_hi, 0);
    bad0 += __double_as_longlong(ddiv(a, b)) != __double_as_longlong(a / b);
    bad1 += __double_as_longlong(drcp(b)) != __double_as_longlong(1.0 / b);
    const unsigned long long pick = xorshift64(s);
    double m1 = draw(s, exp_lo, exp_hi, (int)(pick & 31));
    const double f = draw(s, -30, 2, (int)((pick >> 5) & 31));
    double m3 = m1 * f;
    if (m3 > 4.0 * m1) m3 = 4.0 * m1;
    if (((pick >> 10) & 15) == 0) { m1 = 0.0; m3 = 0.0; }
    if (((pick >> 14) & 15) == 0) m3 = 0.0;
    const double cv = 0.4 * (1.0 + 0x1p-20 * (double)((pick >> 20) & 0xfffff));
    if (m1 > 0.0) bad2 += __double_as_longlong(ratio_div(m3, m1)) != __double_as_longlong(m3 / m1);
    const double ref = m1 > 0.0 ? cv * (m3 / m1) : 0.0;
    bad3 += __double_as_longlong(kappa_ratio(m3, m1, cv)) != __double_as_longlong(ref);
  }
  atomicAdd(&counts[0], bad0); atomicAdd(&counts[1], bad1); atomicAdd(&counts[2], bad2); atomicAdd(&counts[3], bad3);
  if (blockIdx.x == 0 && threadIdx.x == 0) counts[4] = (unsigned long long)gridDim.x * blockDim.x * (unsigned long long)draws_per_thread;
}

// fp64-pipe micro-benchmark behind the numbers DESIGN.md section 5 quotes ("one fp64 warp instruction per two cycles and
// sub-partition, dependent latency 9 cycles"): every warp runs `iters` trips of ILP independent dependent-DFMA chains;
// out[0] = clock64 cycles of warp 0 of CTA 0.  The grid is one CTA of 128 * warps_per_subpartition threads per SM.
template <int ILP>
__global__ void fp64_pipe_selftest_kernel(int iters, double seed, long long* out) {
  double x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) x[i] = seed + i + threadIdx.x;
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = fma(x[i], 1.0000001, 0.5);
  }
  const long long t1 = clock64();
  double sum = 0.0;
#pragma unroll
  for (int i = 0; i < ILP; ++i) sum += x[i];
  if (threadIdx.x == 0 && blockIdx.x == 0) out[0] = t1 - t0;
  if (sum == 12345.678) out[1] = 1;      // keeps the chains alive
}

}  // namespace smaug
