// smaug_flux_kernel.cuh -- streaming fused stage kernel for the case WITHOUT hyperdiffusion ("Without HD" column of
// the paper's Table 1): R = -(d^c_x F_x + d^c_y F_y) (+ the energy source and gravity in the BG / GRAV
// forms, see FluxSmem below), RK combine, wave-speed maxima.  About 90 fp64 operations against 144 bytes per cell and stage: this case
// sits on the memory side of the B200 ridge: what counts is that every byte crosses HBM once (SMAUG_FLUX_DEPTH below).
// Same arithmetic contract as every other stage kernel: bit-identical to the oracle.
//
// One CTA owns a strip of NT - 4 output columns (thread t <-> column x0 - 2 + t) and marches down a chunk of
// rows, newest ("head") row r, output ("tail") row j = r - 2:
//   head: derived quantities of row r; F_x(r) -> shared-memory ring (4 rows); F_y(r) -> five-row register history
//   -- one __syncthreads per row --
//   tail: central x-difference of F_x(j) from the ring (neighbour columns), central y-difference of F_y from
//         the history, R, RK combine, coalesced store, wave-speed maxima.
// Input rows arrive DEPTH - 1 rows ahead through cp.async into a thread-private ring (no registers held, 48 bytes
// per thread and row in flight); the RK operands of the tail row are plain loads issued at the top of the
// step.  The 4 halo columns of a strip, the 4 warm-up rows of a chunk and the pointwise re-read of the stage input at the
// tail row (stages 2 and 4) hit L1 / L2: DRAM traffic 1.01 - 1.03 x the algorithmic bytes per stage.
#pragma once
#include "smaug_split_kernel.cuh"

#ifndef SMAUG_FLUX_DEPTH
#define SMAUG_FLUX_DEPTH 2      // landing-ring rows.  Measured at 8000^2, HD off, ms per stage (NT = strip threads x CTAs per SM):
#endif                          // 128 x 4: depth 4 1.83, 3 1.74, 2 1.70;  256 x 2: depth 3 1.68, 2 1.66 (chosen);  512 x 1: 1.72.
                                // The shallow ring wins: what the kernel gains is shared memory handed back to L1 (the halo
                                // columns, the warm-up rows and the pointwise re-read of the tail row hit there), not bytes in
                                // flight.  Background form (stratified 4000^2): 128 x 3, depth 4 0.906 -> 256 x 2, depth 2 0.661.
#ifndef SMAUG_FLUX_L2HINT
#define SMAUG_FLUX_L2HINT 0     // 1: L2 eviction priorities -- in stages 2 and 4 the stage-input rows (read with their halo by the
#endif                          // cp.async ring and once more pointwise two rows later) are fetched with evict_last, RK operands and
                                // results go through with evict_first.  Measured at 8000^2 (profiles/r02_notes.md): DRAM bytes of
                                // stage 2 / 4 fall from 1.29x / 1.08x to 1.12x / 1.05x of the algorithmic bytes, but stages 1 / 3
                                // get slower and the step does not get faster (7.61 vs 7.53 ms): the kernel is bound by bytes in
                                // flight over ~20 concurrent plane streams (5.2 TB/s of real DRAM traffic in stage 2), not by
                                // the excess bytes.  Kept as a build option, off.

namespace smaug {

__device__ __forceinline__ unsigned long long l2_policy_evict_last() {
  unsigned long long p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
  unsigned long long p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ void cp_async8_hint(double* smem_dst, const double* gsrc, unsigned long long pol) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" ::"r"(sa), "l"(gsrc), "l"(pol) : "memory");
}
__device__ __forceinline__ double ld_hint(const double* p, unsigned long long pol) {
  double v;
  asm volatile("ld.global.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ void st_hint(double* p, double v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}

// BG = true: a background (with or without gravity): the four background planes ride in the landing ring, the
// fluxes take their background terms (c-2), vx / vy of the head row go into a second ring for the x-derivatives of
// the energy source S_e (their y-derivatives come from a five-row register history), gravity is three fmas (c-10).
template <int NT, bool BG = false>
struct FluxSmem {
  static constexpr int DEPTH = SMAUG_FLUX_DEPTH;           // input rows in the landing ring (DEPTH - 1 rows in flight)
  static constexpr int NIN = BG ? NF + NBG : NF;          // fields per landing row
  static constexpr int OFF_FXR = 0;                       // ring 4 rows x 5 planes: F_x
  static constexpr int OFF_VXR = OFF_FXR + 4 * 5 * NT;    // BG: ring 4 rows x 2 planes: vx, vy
  static constexpr int OFF_INR = OFF_VXR + (BG ? 4 * 2 * NT : 0);   // ring DEPTH rows x NIN fields: cp.async landing zone
  static constexpr int OFF_RED = OFF_INR + DEPTH * NIN * NT;
  static constexpr int TOTAL = OFF_RED + 4 * 32;
  static constexpr size_t BYTES = (size_t)TOTAL * sizeof(double);
  static constexpr int CTAS_PER_SM = NT <= 128 ? (BG ? 3 : 4) : 2;
};

template <int NT, bool BG = false, bool GRAV = false>      // GRAV: gravity on a zero background
__global__ void __launch_bounds__(NT, FluxSmem<NT, BG>::CTAS_PER_SM) flux_kernel(const StageArgs a, const MarchGeom mg) {
  using S = FluxSmem<NT, BG>;
  constexpr int DEPTH = S::DEPTH, NIN = S::NIN;
  extern __shared__ __align__(16) double smem[];
  double* const FXR = smem + S::OFF_FXR;
  [[maybe_unused]] double* const VXR = smem + S::OFF_VXR;
  double* const INR = smem + S::OFF_INR;
  double* const red_sh = smem + S::OFF_RED;
  const Grid& g = a.g;
  const int tid = threadIdx.x;
  constexpr int W = NT - 4;
  const int x0 = blockIdx.x * W;
  const int ci = x0 - 2 + tid;                            // interior column of this thread (>= -2: a ghost)
  // column used for loads: lanes right of the padded plane (a partial last strip) produce nothing; they read the columns one
  // strip width to their left -- distinct, coalesced addresses (hundreds of lanes clamped onto ONE address make cp.async
  // crawl: 2044^2 with 256-thread strips 0.168 -> 0.126 ms per stage)
  const int cl = ci <= g.nx + NG - 1 ? ci : max(ci - NT, -NG);
  const bool col_out = tid >= 2 && tid < NT - 2 && ci < g.nx;
  const int ystart = blockIdx.y * mg.rows_per_cta;
  const int yend = min(ystart + mg.rows_per_cta, g.ny);
  const double gm1 = a.prm.gamma - 1.0, gamma = a.prm.gamma;
  const double idx_ = a.prm.inv_dx, idy_ = a.prm.inv_dy;
  const double cdt = a.c * a.sc->dt;
  const int combine = a.combine, ws_mode = a.ws_mode;
  const unsigned upitch = (unsigned)g.pitch;
  // element offsets inside a plane (fewer than 2^31 elements: smaug_create checks)
  unsigned gin = (unsigned)(ystart - 2 + NG) * upitch + (unsigned)(cl + XOFF);     // (cl, next row to fetch)
  unsigned gj = (unsigned)(ystart + NG) * upitch + (unsigned)(cl + XOFF);           // (cl, tail row j)
  int fetched = ystart - 2;                               // next row to fetch
  const int last_row = g.ny + NG - 1;
  int slot_f = 0;                                         // landing slot of the next row to fetch
#if SMAUG_FLUX_L2HINT
  const unsigned long long pol_keep = l2_policy_evict_last(), pol_once = l2_policy_evict_first();
#endif
#if SMAUG_FLUX_L2HINT
#define LD_ONCE(p) ld_hint((p), pol_once)
#define ST_ONCE(p, v) st_hint((p), (v), pol_once)
#else
#define LD_ONCE(p) (*(p))
#define ST_ONCE(p, v) (*(p) = (v))
#endif
  auto fetch_row = [&]() {
    double* dst = INR + slot_f * NIN * NT + tid;
#if SMAUG_FLUX_L2HINT
    if (combine != COMBINE_BASE) {
#pragma unroll
      for (int f = 0; f < NF; ++f) cp_async8_hint(dst + f * NT, a.in.p[f] + gin, pol_keep);
    } else
#endif
    {
#pragma unroll
      for (int f = 0; f < NF; ++f) cp_async8(dst + f * NT, a.in.p[f] + gin);
    }
    if constexpr (BG) {
#pragma unroll
      for (int k = 0; k < NBG; ++k) cp_async8(dst + (NF + k) * NT, a.bg.p[k] + gin);
    }
    cp_async_commit();
    if (fetched < last_row) gin += upitch;                // rows below the padded plane are never dereferenced
    ++fetched;
    slot_f = slot_f == DEPTH - 1 ? 0 : slot_f + 1;
  };
#pragma unroll
  for (int k = 0; k < DEPTH - 1; ++k) fetch_row();
  int slot_r = 0;                                         // landing slot of row r
  int s4 = 0;                                             // FXR slot of row r (mod 4)

  double fy[5][5];                                        // F_y of rows r-4 .. r (index 4 = row r)
#pragma unroll
  for (int k = 0; k < 5; ++k)
#pragma unroll
    for (int f = 0; f < 5; ++f) fy[k][f] = 0.0;
  double wsmax[4] = {0.0, 0.0, 0.0, 0.0};
  [[maybe_unused]] double hvx[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, hvy[5] = {0.0, 0.0, 0.0, 0.0, 0.0};   // BG: rows r-4 .. r

#pragma unroll 1
  for (int r = ystart - 2; r < yend + 2; ++r) {
    const bool tail_on = r >= ystart + 2;                 // uniform over the CTA
    // operands of the RK combine for row j: issued here, consumed at the end of the step
    double jbase[NF], jacc[NF], jin[NF];
    if (tail_on) {
      if (combine == COMBINE_FINAL) {
#pragma unroll
        for (int f = 0; f < NF; ++f) { jin[f] = a.in.p[f][gj]; jacc[f] = LD_ONCE(a.acc_in.p[f] + gj); }
      } else {
#pragma unroll
        for (int f = 0; f < NF; ++f) jbase[f] = LD_ONCE(a.base.p[f] + gj);
        if (combine == COMBINE_ACC) {
#pragma unroll
          for (int f = 0; f < NF; ++f) jin[f] = a.in.p[f][gj];
        }
      }
    }
    cp_async_wait<DEPTH - 2>();                           // row r has landed (later rows may be in flight)
    const double* src = INR + slot_r * NIN * NT + tid;
    const double rhot = src[F_RHO * NT], mx = src[F_MX * NT], my = src[F_MY * NT];
    const double et = src[F_E * NT], bx = src[F_BX * NT], by = src[F_BY * NT];
    double rb = 0.0, eb = 0.0, Bbx = 0.0, Bby = 0.0;
    if constexpr (BG) {
      rb = src[(NF + BG_RHO) * NT]; eb = src[(NF + BG_E) * NT];
      Bbx = src[(NF + BG_BX) * NT]; Bby = src[(NF + BG_BY) * NT];
    }
    fetch_row();                                          // into the slot read one step ago
    slot_r = slot_r == DEPTH - 1 ? 0 : slot_r + 1;

    // ------------------------------------------------------------------ head: derived quantities, F_x, F_y of row r
    const double rho = BG ? rb + rhot : rhot;
    const double rr = drcp(rho);
    const double vx = mx * rr, vy = my * rr;
    const double b2h = 0.5 * fma(by, by, bx * bx);
    const double ke = 0.5 * fma(my, vy, mx * vx);
    const double btv = fma(by, vy, bx * vx);
    double* fxw = FXR + s4 * 5 * NT + tid;
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
      for (int f = 0; f < 5; ++f) fy[k][f] = fy[k + 1][f];
    if constexpr (BG) {
      const double cross = fma(Bby, by, Bbx * bx);
      const double eps = ((et - ke) - cross) - b2h;
      const double ptt = fma(gm1, eps, cross + b2h);
      const double Bx = Bbx + bx, By = Bby + by;
      const double Bbv = fma(Bby, vy, Bbx * vx);
      const double h = (et + eb) + ptt;
      fxw[C_RHO * NT] = rho * vx;
      fxw[C_MX * NT] = ((fma(mx, vx, -(bx * bx)) - bx * Bbx) - Bbx * bx) + ptt;
      fxw[C_MY * NT] = (fma(my, vx, -(by * bx)) - by * Bbx) - Bby * bx;
      fxw[C_E * NT] = (fma(vx, h, -(bx * btv)) - bx * Bbv) - Bbx * btv;
      fxw[C_B * NT] = fma(vx, By, -(Bx * vy));
      fy[4][C_RHO] = rho * vy;
      fy[4][C_MX] = (fma(mx, vy, -(bx * by)) - bx * Bby) - Bbx * by;
      fy[4][C_MY] = ((fma(my, vy, -(by * by)) - by * Bby) - Bby * by) + ptt;
      fy[4][C_E] = (fma(vy, h, -(by * btv)) - by * Bbv) - Bby * btv;
      fy[4][C_B] = fma(vy, Bx, -(By * vx));
      VXR[(s4 * 2 + 0) * NT + tid] = vx;
      VXR[(s4 * 2 + 1) * NT + tid] = vy;
#pragma unroll
      for (int k = 0; k < 4; ++k) { hvx[k] = hvx[k + 1]; hvy[k] = hvy[k + 1]; }
      hvx[4] = vx; hvy[4] = vy;
    } else {
      const double eps = (et - ke) - b2h;
      const double ptt = fma(gm1, eps, b2h);
      const double h = et + ptt;
      fxw[C_RHO * NT] = rho * vx;
      fxw[C_MX * NT] = fma(mx, vx, -(bx * bx)) + ptt;
      fxw[C_MY * NT] = fma(my, vx, -(by * bx));
      fxw[C_E * NT] = fma(vx, h, -(bx * btv));
      fxw[C_B * NT] = fma(vx, by, -(bx * vy));
      fy[4][C_RHO] = rho * vy;
      fy[4][C_MX] = fma(mx, vy, -(bx * by));
      fy[4][C_MY] = fma(my, vy, -(by * by)) + ptt;
      fy[4][C_E] = fma(vy, h, -(by * btv));
      fy[4][C_B] = fma(vy, bx, -(by * vx));
      if constexpr (GRAV) {
#pragma unroll
        for (int k = 0; k < 4; ++k) { hvx[k] = hvx[k + 1]; hvy[k] = hvy[k + 1]; }
        hvx[4] = vx; hvy[4] = vy;
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ tail: R(j), combine, write
    if (tail_on) {
      const int sj = (s4 + 2) & 3;                        // FXR slot of row j = r - 2
      const int tl = min(max(tid, 2), NT - 3);            // halo threads read in range; their result is unused
      const double* fxr = FXR + sj * 5 * NT + tl;
      double R[NF];
      double cdx[5], cdy[5];
#pragma unroll
      for (int f = 0; f < 5; ++f) {
        cdx[f] = cd12v(fxr[f * NT - 2], fxr[f * NT - 1], fxr[f * NT + 1], fxr[f * NT + 2]);
        cdy[f] = cd12v(fy[0][f], fy[1][f], fy[3][f], fy[4][f]);
      }
      R[F_RHO] = fma(cdx[C_RHO], idx_, cdy[C_RHO] * idy_) * (-1.0 / 12.0);
      R[F_MX] = fma(cdx[C_MX], idx_, cdy[C_MX] * idy_) * (-1.0 / 12.0);
      R[F_MY] = fma(cdx[C_MY], idx_, cdy[C_MY] * idy_) * (-1.0 / 12.0);
      R[F_E] = fma(cdx[C_E], idx_, cdy[C_E] * idy_) * (-1.0 / 12.0);
      R[F_BX] = (cdy[C_B] * idy_) * (-1.0 / 12.0);        // F_x(bx) == 0
      R[F_BY] = fma(cdx[C_B], idx_, 0.0) * (-1.0 / 12.0); // F_y(by) == 0
      if constexpr (!BG && GRAV) {     // gravity on a zero background (c-10: rho~ is the total density)
        const double rt = a.in.p[F_RHO][gj];
        R[F_MX] = fma(rt, a.prm.gx, R[F_MX]);
        R[F_MY] = fma(rt, a.prm.gy, R[F_MY]);
        R[F_E] = fma(rt, fma(a.prm.gy, hvy[2], a.prm.gx * hvx[2]), R[F_E]);
      }
      [[maybe_unused]] double jrb = 0.0, jeb = 0.0, jBbx = 0.0, jBby = 0.0;
      if constexpr (BG) {
        // energy source S_e (c-2) and gravity (c-10) at the tail cell (row j = r - 2: histories index 2)
        jrb = a.bg.p[BG_RHO][gj]; jeb = a.bg.p[BG_E][gj]; jBbx = a.bg.p[BG_BX][gj]; jBby = a.bg.p[BG_BY][gj];
        const double* vxr = VXR + (sj * 2 + 0) * NT + tl;
        const double* vyr = VXR + (sj * 2 + 1) * NT + tl;
        const double dxvx = (cd12v(vxr[-2], vxr[-1], vxr[1], vxr[2]) * idx_) * (1.0 / 12.0);
        const double dxvy = (cd12v(vyr[-2], vyr[-1], vyr[1], vyr[2]) * idx_) * (1.0 / 12.0);
        const double dyvx = (cd12v(hvx[0], hvx[1], hvx[3], hvx[4]) * idy_) * (1.0 / 12.0);
        const double dyvy = (cd12v(hvy[0], hvy[1], hvy[3], hvy[4]) * idy_) * (1.0 / 12.0);
        const double bb2h = 0.5 * fma(jBby, jBby, jBbx * jBbx);
        const double ptb = fma(gm1, jeb - bb2h, bb2h);
        const double S = fma(-ptb, dxvx + dyvy,
                             fma(jBby * jBby, dyvy, fma(jBbx * jBby, dxvy + dyvx, (jBbx * jBbx) * dxvx)));
        R[F_E] = R[F_E] + S;
        if (a.prm.grav_on) {
          const double rt = a.in.p[F_RHO][gj];             // rho~ of the tail cell
          R[F_MX] = fma(rt, a.prm.gx, R[F_MX]);
          R[F_MY] = fma(rt, a.prm.gy, R[F_MY]);
          R[F_E] = fma(rt, fma(a.prm.gy, hvy[2], a.prm.gx * hvx[2]), R[F_E]);
        }
      }
      double o[NF];
      if (combine == COMBINE_FINAL) {
#pragma unroll
        for (int f = 0; f < NF; ++f) o[f] = fma(cdt, R[f], fma(fma(-2.0, jin[f], jacc[f]), 1.0 / 3.0, jin[f]));
      } else {
#pragma unroll
        for (int f = 0; f < NF; ++f) o[f] = fma(cdt, R[f], jbase[f]);
      }
      if (col_out) {            // then cl == ci: gj is the address of the output cell as well
#pragma unroll
        for (int f = 0; f < NF; ++f) ST_ONCE(a.out.p[f] + gj, o[f]);
        if (combine == COMBINE_ACC) {
#pragma unroll
          for (int f = 0; f < NF; ++f) ST_ONCE(a.acc_out.p[f] + gj, fma(2.0, o[f], jin[f] - jbase[f]));
        }
        if (ws_mode != WS_NONE) {
          // split_wavespeeds (smaug_split_kernel.cuh): the same maxima, candidates entering with `c > m ? c : m`, and in
          // the last stage the two fast speeds only where they can still raise the thread's running maximum
          double ot[NF];
          if constexpr (BG) {
            ot[F_RHO] = jrb + o[F_RHO]; ot[F_MX] = o[F_MX]; ot[F_MY] = o[F_MY]; ot[F_E] = jeb + o[F_E];
            ot[F_BX] = jBbx + o[F_BX]; ot[F_BY] = jBby + o[F_BY];
          } else {
#pragma unroll
            for (int f = 0; f < NF; ++f) ot[f] = o[f];
          }
          if (ws_mode == WS_FULL) split_wavespeeds<WS_FULL>(ot, gamma, wsmax, wsmax[0], wsmax[1]);
          else split_wavespeeds<WS_VT>(ot, gamma, wsmax, 0.0, 0.0);
        }
      }
      gj += upitch;
    }
    s4 = (s4 + 1) & 3;
  }
  cp_async_wait<0>();
  if (ws_mode != WS_NONE) block_max4_atomic(wsmax, red_sh, a.sc->red[a.red_out], ws_mode == WS_FULL ? 0 : 2);
}

#undef LD_ONCE
#undef ST_ONCE

}  // namespace smaug
