// smaug_stage_common.cuh -- what every fused stage kernel shares: the argument block of one RK stage, the combine /
// wave-speed modes, component indices, and the small exact helpers (max, |x|, the one-interface kappa, the central
// difference, cp.async).  The hot kernels (smaug_split_kernel.cuh, smaug_flux_kernel.cuh, smaug_line_kernel.cuh) include
// this and nothing of the second implementations (smaug_stage_kernel.cuh, smaug_march_kernel.cuh).
#pragma once
#include "smaug_aux_kernels.cuh"

namespace smaug {

// What the epilogue does with R (c-6).  dt is read from device memory (no host sync).
//   COMBINE_BASE : out = base + c dt R                      (stages 1..3 of RK4; Euler; midpoint)
//   COMBINE_ACC  : out = base + c dt R;  acc = (in - base) + 2 out          (stage 2 of RK4)
//   COMBINE_FINAL: out = in + (acc - 2 in)/3 + c dt R       (stage 4 of RK4, c = 1/6)
// which is w^{n+1} = (w1 + 2 w2 + w3 - w^n)/3 + dt/6 R(w3), algebraically the classical RK4 update,
// grouped so that R == 0 returns w^n bit for bit.
enum { COMBINE_BASE = 0, COMBINE_ACC = 1, COMBINE_FINAL = 2 };
// Wave-speed reduction of the written state: none, only {a^2, b^2} (v_t of the next stage), or all four.
enum { WS_NONE = 0, WS_VT = 1, WS_FULL = 2 };

struct StageArgs {
  Grid g;
  Params prm;
  CPlanes6 in;       // stage input (ghost-filled), read with its halo
  CPlanes6 base;     // w^n            (COMBINE_BASE / COMBINE_ACC)
  CPlanes6 acc_in;   // accumulator    (COMBINE_FINAL)
  Planes6 out;       // stage output (interior written)
  Planes6 acc_out;   // accumulator    (COMBINE_ACC)
  CPlanes4 bg;       // background (ghost-filled), only dereferenced when BG
  DeviceScalars* sc;
  int red_in;        // reduction set holding the maxima of `in`  (v_t)
  int red_out;       // reduction set receiving the maxima of `out`
  double c;          // RK coefficient multiplying dt R
  int combine;
  int ws_mode;
};

enum { K_RHO = 0, K_VX = 1, K_VY = 2, K_EPS = 3, K_B = 4 };                 // kappa families; Phi components
enum { C_RHO = 0, C_MX = 1, C_MY = 2, C_E = 3, C_B = 4 };

// max of two non-negative doubles: one DSETP + two selects (fmax() costs ~7 instructions on sm_100a
// because of its NaN-quieting semantics).  max is exact, so any evaluation order is bit-safe.
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
// |x| as one integer op on the high word (keeps the fp64 pipe free; bit-identical to fabs)
__device__ __forceinline__ double dabs(double x) {
  return __hiloint2double(__double2hiint(x) & 0x7fffffff, __double2loint(x));
}

// chunk geometry of a streaming kernel
struct MarchGeom {
  int rows_per_cta;   // output rows per CTA (chunk height)
};

// kappa at ONE interface from the six cells u[0..5] = cells -2 .. +3 around it (interface between u[2], u[3]).
__device__ __forceinline__ double kappa6(double u0, double u1, double u2, double u3, double u4, double u5,
                                         double cv, double& d1_mid) {
  const double a0 = u1 - u0, a1 = u2 - u1, a2 = u3 - u2, a3 = u4 - u3, a4 = u5 - u4;   // D1 at -2 .. +2
  const double t0 = dabs(fma(3.0, a1, -(u3 - u0)));     // D3 at interface -1
  const double t1 = dabs(fma(3.0, a2, -(u4 - u1)));     // D3 at interface  0
  const double t2 = dabs(fma(3.0, a3, -(u5 - u2)));     // D3 at interface +1
  const double m3 = dmax(dmax(t0, t1), t2);
  const double m1 = dmax(dmax(dmax(dabs(a0), dabs(a1)), dmax(dabs(a2), dabs(a3))), dabs(a4));
  d1_mid = a2;
  return kappa_ratio(m3, m1, cv);
}

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ double cd12v(double m2, double m1, double p1, double p2) {
  return fma(8.0, p1 - m1, -(p2 - m2));
}

}  // namespace smaug
