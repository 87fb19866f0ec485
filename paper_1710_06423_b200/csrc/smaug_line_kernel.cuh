// smaug_line_kernel.cuh -- the small-grid path: WHOLE TIME STEPS of a one-dimensional problem (ny = 1: the paper's
// Brio-Wu shock tube, BASELINE config 1) in ONE persistent launch.
//
// An 800 x 1 grid is 38 KB of state: it lives in L2, and a step of nine ordinary launches (dt, 4 x {ghost fill, stage
// kernel}) is launch latency plus seven marched rows per stage of which six are copies of the only row (45 us per step
// even as a CUDA-graph replay).  Here one thread-block CLUSTER covers the line -- one CTA of LINE_NT threads per
// LINE_NT - 6 cells (thread <-> cell, three halo cells per side), at most 8 CTAs (the portable cluster size) -- and
// loops over steps and RK stages by itself.  The state never leaves the chip between stages: every CTA keeps its cells in
// its own shared memory (w^n and the accumulator of a cell in its thread's registers), the three halo cells per side are
// PULLED out of the owning neighbour's shared memory (distributed shared memory; the boundary rule of c-8 is the index
// map of that pull: periodic -> wrap, open -> clamp, fixed -> the frozen ghost cell, read once), the four wave-speed
// maxima are all-reduced the same way (one lane per CTA pulls, warp shuffles finish), dt is evaluated by every CTA from
// those four numbers, and ONE hardware cluster barrier (barrier.cluster) per stage orders it all.  Global memory is
// read at the start of the launch and written at its end; nothing returns to the host between steps.
//
// y-invariance.  With ny = 1 and a periodic or open y-boundary every ghost row is a copy of the row, so each y-difference
// the scheme takes is x - x = +0 exactly and every kappa_y is cv * (0 / 1) = +0 (c-5: M1 = 0 -> 0).  The arithmetic
// contract is kept to the bit, signs of zero included, by executing the y-terms of the other stage
// kernels with those literal zeros (fma(0, 1/dy, R) turns a -0 into +0 exactly as the oracle's does) and by leaving out
// only what cannot change a bit: C_y = F_y - G(.;y) is the same finite number on every row, so its central y-difference
// is +0 whatever it is, and it is never formed.  (A fixed y-boundary keeps its set_state ghosts, which are not copies:
// such a context takes the ordinary path.)  Same results as every other stage kernel: tests/test_gpu_parity.py.
#pragma once
#include <cooperative_groups.h>

#include "smaug_stage_common.cuh"

namespace smaug {

constexpr int LINE_NT = 128, LINE_HALO = 3, LINE_W = LINE_NT - 2 * LINE_HALO, LINE_MAX_CTAS = 8;
constexpr int LINE_MAX_NX = LINE_W * LINE_MAX_CTAS;

struct LineArgs {
  Grid g;
  Params prm;
  Planes6 buf[4];            // the context's four state buffers (buf[0]: the state between steps)
  DeviceScalars* sc;
  int state_set;             // reduction set holding the maxima of the state at entry (0 or 4)
  int n_steps;
  int rk_order;              // 4 or 2 (Euler swaps buffers between steps: not handled here)
  double cfl, fixed_dt, dx, dy;
};

struct LineSmem {
  static constexpr int PW = LINE_NT + 8;                  // padded plane width (index tid + 4)
  static constexpr int OFF_ST = 0;                        // 2 x 6 planes: the stage input / output (double-buffered by stage)
  static constexpr int OFF_U = OFF_ST + 2 * NF * PW;      // 5 planes: rho~, vx, vy, eps~, by~ of the row
  static constexpr int OFF_CX = OFF_U + 5 * PW;           // 5 planes: C_x = F_x - G(.;x)
  static constexpr int OFF_PX = OFF_CX + 5 * PW;          // 5 planes: Phi_x at interface (c | c+1)
  static constexpr int OFF_MAXO = OFF_PX + 5 * PW;        // 2 x 4: this CTA's maxima of the stage output (double-buffered)
  static constexpr int OFF_MAXS = OFF_MAXO + 8;           // 4: cluster-wide maxima of the current stage input
  static constexpr int OFF_RED = OFF_MAXS + 4;
  static constexpr int TOTAL = OFF_RED + 4 * 32;
  static constexpr size_t BYTES = (size_t)TOTAL * sizeof(double);
};

// c-8 along x as an index map: the padded column a stage reads for interior-relative column i
__device__ __forceinline__ int line_map_x(const Grid& g, int i) {
  if (i < 0) return g.bc[0] == BC_PERIODIC ? wrap_idx(i, g.nx) : (g.bc[0] == BC_OPEN ? 0 : max(i, -NG));
  if (i >= g.nx) return g.bc[1] == BC_PERIODIC ? wrap_idx(i, g.nx) : (g.bc[1] == BC_OPEN ? g.nx - 1 : min(i, g.nx + NG - 1));
  return i;
}

// One RK stage of the line (all LINE_NT threads of every CTA of the cluster).  The stage input of this thread's cell is
// `w` (pulled by the caller), the output goes to the CTA's own state plane `st_out` and into `o`; this CTA's maxima of
// the output go to maxo[4].
template <bool HD>
__device__ __forceinline__ void line_stage(const LineArgs& la, const bool col_out, double* const smem, const double (&w)[NF],
                                           double* const st_out, double* const maxo, const int combine, const double cdt,
                                           const int ws, const double (&jbase)[NF], double (&jacc)[NF], double (&o)[NF]) {
  using S = LineSmem;
  constexpr int PW = S::PW;
  double* const U = smem + S::OFF_U;
  double* const CX = smem + S::OFF_CX;
  double* const PX = smem + S::OFF_PX;
  double* const red_sh = smem + S::OFF_RED;
  const double* const MAXS = smem + S::OFF_MAXS;
  const int tid = threadIdx.x, tp = tid + 4;
  const double gm1 = la.prm.gamma - 1.0, gamma = la.prm.gamma;
  const double idx_ = la.prm.inv_dx, idy_ = la.prm.inv_dy;
  const double Z = 0.0;                                                 // every y-difference of a y-invariant state

  // ---- the cell: derived quantities, F_x (c-2)
  const double rho = w[F_RHO], mx = w[F_MX], my = w[F_MY], et = w[F_E], bx = w[F_BX], by = w[F_BY];
  const double rr = drcp(rho);
  const double vx = mx * rr, vy = my * rr;
  const double b2h = 0.5 * fma(by, by, bx * bx);
  const double ke = 0.5 * fma(my, vy, mx * vx);
  const double eps = (et - ke) - b2h;
  const double ptt = fma(gm1, eps, b2h);
  const double btv = fma(by, vy, bx * vx);
  const double h = et + ptt;
  double fx[5];
  fx[C_RHO] = rho * vx;
  fx[C_MX] = fma(mx, vx, -(bx * bx)) + ptt;
  fx[C_MY] = fma(my, vx, -(by * bx));
  fx[C_E] = fma(vx, h, -(bx * btv));
  fx[C_B] = fma(vx, by, -(bx * vy));
  if (HD) {
    // C_x = F_x - G(.;x): the mixed fluxes along x are built from kappa_y and central y-differences, all literal zeros
    // here (kv = (kappa_y + kappa_y)/2, d^c_y u = fma(8, u - u, -(u - u))); executed so that the signs of zero follow
    const double kv = 0.5 * (Z + Z), kb = 0.5 * (Z + Z);
    const double dcy = fma(8.0, Z, -Z);
    const double gm = ((0.5 * rho) * kv) * (dcy * (1.0 / 12.0));       // G(my ; x)
    const double gb = -(kb * (dcy * (1.0 / 12.0)));                     // G(by ; x)
    fx[C_MY] = fx[C_MY] - gm;
    fx[C_E] = fx[C_E] - fma(vy, gm, by * gb);
    fx[C_B] = fx[C_B] - gb;
  }
  U[0 * PW + tp] = rho; U[1 * PW + tp] = vx; U[2 * PW + tp] = vy; U[3 * PW + tp] = eps; U[4 * PW + tp] = by;
#pragma unroll
  for (int f = 0; f < 5; ++f) CX[f * PW + tp] = fx[f];
  __syncthreads();                                                      // (also publishes MAXS, written by thread 0)

  // ---- x-interface (c | c+1): kappa_x, Phi_x (c-5); threads LINE_NT-3.. have no right neighbours: their Phi is unused
  double px[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (HD) {
    const double vt = sqrt(MAXS[2]) + sqrt(MAXS[3]);
    const double cv_rho = la.prm.c_rho * vt, cv_mom = la.prm.c_mom * vt, cv_e = la.prm.c_e * vt, cv_b = la.prm.c_b * vt;
    const int t6 = min(max(tp, 6), PW - 4);                             // keeps the six-cell window inside the plane
    auto win = [&](int plane, double (&u)[6]) {
#pragma unroll
      for (int k = 0; k < 6; ++k) u[k] = U[plane * PW + t6 - 2 + k];
    };
    double u[6], d;
    win(0, u);
    const double k_rho = kappa6(u[0], u[1], u[2], u[3], u[4], u[5], cv_rho, d);
    const double rbar = 0.5 * (u[2] + u[3]);
    px[C_RHO] = k_rho * d;
    win(1, u);
    const double k_vx = kappa6(u[0], u[1], u[2], u[3], u[4], u[5], cv_mom, d);
    px[C_MX] = (rbar * k_vx) * d;
    const double vxbar = 0.5 * (u[2] + u[3]);
    win(2, u);
    const double k_vy = kappa6(u[0], u[1], u[2], u[3], u[4], u[5], cv_mom, d);
    px[C_MY] = ((0.5 * rbar) * k_vy) * d;
    const double vybar = 0.5 * (u[2] + u[3]);
    win(3, u);
    const double k_e = kappa6(u[0], u[1], u[2], u[3], u[4], u[5], cv_e, d);
    const double p_eps = k_e * d;
    win(4, u);
    const double k_b = kappa6(u[0], u[1], u[2], u[3], u[4], u[5], cv_b, d);
    px[C_B] = k_b * d;
    px[C_E] = fma(0.5 * (u[2] + u[3]), px[C_B], fma(vybar, px[C_MY], fma(vxbar, px[C_MX], p_eps)));
#pragma unroll
    for (int f = 0; f < 5; ++f) PX[f * PW + tp] = px[f];
    __syncthreads();
  }

  // ---- R, RK combine, wave-speed maxima (c-3, c-6, c-4): the Y role's assembly with y-terms of zero
  double wsmax[4] = {0.0, 0.0, 0.0, 0.0};
  if (col_out) {
    double cdx[5], R[NF];
#pragma unroll
    for (int f = 0; f < 5; ++f)
      cdx[f] = cd12v(CX[f * PW + tp - 2], CX[f * PW + tp - 1], CX[f * PW + tp + 1], CX[f * PW + tp + 2]);
    const double cdyi = fma(8.0, Z, -Z) * idy_;                          // d^c_y C_y of identical rows
    R[F_RHO] = fma(cdx[C_RHO], idx_, cdyi) * (-1.0 / 12.0);
    R[F_MX] = fma(cdx[C_MX], idx_, cdyi) * (-1.0 / 12.0);
    R[F_MY] = fma(cdx[C_MY], idx_, cdyi) * (-1.0 / 12.0);
    R[F_E] = fma(cdx[C_E], idx_, cdyi) * (-1.0 / 12.0);
    R[F_BX] = cdyi * (-1.0 / 12.0);
    R[F_BY] = fma(cdx[C_B], idx_, 0.0) * (-1.0 / 12.0);
    if (la.prm.grav_on) {                                               // c-10 on a zero background
      R[F_MX] = fma(rho, la.prm.gx, R[F_MX]);
      R[F_MY] = fma(rho, la.prm.gy, R[F_MY]);
      R[F_E] = fma(rho, fma(la.prm.gy, vy, la.prm.gx * vx), R[F_E]);
    }
    if (HD) {
      R[F_RHO] = fma(px[C_RHO] - PX[C_RHO * PW + tp - 1], idx_, R[F_RHO]);
      R[F_MX] = fma(px[C_MX] - PX[C_MX * PW + tp - 1], idx_, R[F_MX]);
      R[F_MY] = fma(px[C_MY] - PX[C_MY * PW + tp - 1], idx_, R[F_MY]);
      R[F_E] = fma(px[C_E] - PX[C_E * PW + tp - 1], idx_, R[F_E]);
      R[F_BY] = fma(px[C_B] - PX[C_B * PW + tp - 1], idx_, R[F_BY]);
      const double dpy = Z - Z;                                          // Phi_y(j | j+1) - Phi_y(j-1 | j), both +0
      R[F_RHO] = fma(dpy, idy_, R[F_RHO]);
      R[F_MX] = fma(dpy, idy_, R[F_MX]);
      R[F_MY] = fma(dpy, idy_, R[F_MY]);
      R[F_E] = fma(dpy, idy_, R[F_E]);
      R[F_BX] = fma(dpy, idy_, R[F_BX]);
    }
    if (combine == COMBINE_FINAL) {
#pragma unroll
      for (int f = 0; f < NF; ++f) o[f] = fma(cdt, R[f], fma(fma(-2.0, w[f], jacc[f]), 1.0 / 3.0, w[f]));
    } else {
#pragma unroll
      for (int f = 0; f < NF; ++f) o[f] = fma(cdt, R[f], jbase[f]);
    }
#pragma unroll
    for (int f = 0; f < NF; ++f) st_out[f * PW + tp] = o[f];
    if (combine == COMBINE_ACC) {
#pragma unroll
      for (int f = 0; f < NF; ++f) jacc[f] = fma(2.0, o[f], w[f] - jbase[f]);
    }
    if (ws != WS_NONE) cell_wavespeeds(o[F_RHO], o[F_MX], o[F_MY], o[F_E], o[F_BX], o[F_BY], gamma, ws == WS_FULL, wsmax);
  }
  // block maxima (warp shuffles, then one warp) -> maxo[4]; everything else of the reduction is the cluster's
#pragma unroll
  for (int k = 0; k < 4; ++k) wsmax[k] = warp_max(wsmax[k]);
  if ((tid & 31) == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) red_sh[k * 32 + (tid >> 5)] = wsmax[k];
  }
  __syncthreads();
  if (tid < 4) {
    double v = red_sh[tid * 32];
#pragma unroll
    for (int q = 1; q < LINE_NT / 32; ++q) v = fmax(v, red_sh[tid * 32 + q]);
    maxo[tid] = v;
  }
}

template <bool HD>
__global__ void __launch_bounds__(LINE_NT, 1) line_step_kernel(const LineArgs la) {
  namespace cg = cooperative_groups;
  using S = LineSmem;
  constexpr int PW = S::PW;
  extern __shared__ double smem[];
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank(), nct = (int)cluster.num_blocks();
  const Grid& g = la.g;
  const int tid = threadIdx.x, tp = tid + 4;
  const int i = rank * LINE_W - LINE_HALO + tid;                        // interior-relative column of this thread
  const bool col_out = tid >= LINE_HALO && tid < LINE_NT - LINE_HALO && i < g.nx;
  double* const ST = smem + S::OFF_ST;
  double* const MAXO = smem + S::OFF_MAXO;
  double* const MAXS = smem + S::OFF_MAXS;
  __shared__ double dt_sh;

  // Where this thread's stage input lives (c-8 as an index map, fixed for the whole launch): an output thread owns its
  // cell; a halo thread pulls cell s = map(i) out of the state plane of the CTA that owns it (distributed shared memory);
  // a ghost cell of a FIXED side is frozen: read once from global memory.
  const int s = line_map_x(g, min(i, g.nx + NG - 1));
  const bool frozen_src = s < 0 || s >= g.nx;
  const int owner = frozen_src ? rank : min(s / LINE_W, nct - 1);
  const int otp = frozen_src ? tp : s - owner * LINE_W + LINE_HALO + 4;
  const double* const pull = owner == rank ? ST : cluster.map_shared_rank(ST, owner);
  double frozen[NF] = {1.0, 0.0, 0.0, 1.0, 0.0, 0.0};
  if (frozen_src) {
#pragma unroll
    for (int f = 0; f < NF; ++f) frozen[f] = la.buf[0].p[f][cell_addr(g, s, 0)];
  }
  // the state into the CTA's plane 0; the state's maxima (set A: set_state's reduction or an earlier step) into MAXS
  if (col_out) {
#pragma unroll
    for (int f = 0; f < NF; ++f) ST[f * PW + tp] = la.buf[0].p[f][cell_addr(g, i, 0)];
  }
  if (tid < 4) MAXS[tid] = __longlong_as_double((long long)la.sc->red[la.state_set][tid]);
  double t_sim = 0.0, dt = 0.0;
  int bad = 0;
  if (rank == 0 && tid == 0) t_sim = la.sc->t;
  cluster.sync();

  const int vt_mode = HD ? WS_VT : WS_NONE;
  int cur = 0;                                                          // state plane holding the current stage input
  double jbase[NF] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, jacc[NF] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, o[NF] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  for (int step = 0; step < la.n_steps; ++step) {
    // c-7: dt from the maxima of w^n.  Every CTA evaluates the same formula on the same four numbers.
    if (tid == 0) {
      double d = la.fixed_dt;
      if (!(la.fixed_dt > 0.0)) {
        double m = __longlong_as_double(0x7ff0000000000000LL);   // +inf
        if (g.nx > 1) m = fmin(m, la.dx / MAXS[0]);
        if (g.ny > 1) m = fmin(m, la.dy / MAXS[1]);
        d = la.cfl * m;
      }
      dt_sh = d;
      if (!(d > 0.0) || isinf(d) || isnan(d)) bad = 1;
      t_sim += d;
    }
    __syncthreads();
    dt = dt_sh;
    const int nstages = la.rk_order == 4 ? 4 : 2;
    for (int k = 0; k < nstages; ++k) {
      int combine, ws;
      double coef;
      if (la.rk_order == 4) {        // c-6: w1 = wn + dt/2 R(wn), w2 = wn + dt/2 R(w1) (+ acc), w3 = wn + dt R(w2), final
        combine = k == 1 ? COMBINE_ACC : (k == 3 ? COMBINE_FINAL : COMBINE_BASE);
        coef = k < 2 ? 0.5 : (k == 2 ? 1.0 : 1.0 / 6.0);
        ws = k == 3 ? WS_FULL : vt_mode;
      } else {                       // midpoint rule
        combine = COMBINE_BASE; coef = k == 0 ? 0.5 : 1.0; ws = k == 0 ? vt_mode : WS_FULL;
      }
      double w[NF];
#pragma unroll
      for (int f = 0; f < NF; ++f) w[f] = frozen_src ? frozen[f] : pull[(cur * NF + f) * PW + otp];
      if (k == 0) {
#pragma unroll
        for (int f = 0; f < NF; ++f) jbase[f] = w[f];                    // w^n of this cell for the whole step
      }
      line_stage<HD>(la, col_out, smem, w, ST + (cur ^ 1) * NF * PW, MAXO + (cur ^ 1) * 4, combine, coef * dt, ws, jbase, jacc, o);
      cluster.sync();          // every CTA's stage output and maxima are in its shared memory, visible cluster-wide
      cur ^= 1;
      // the MAX all-reduce of the four maxima: one lane per CTA of the cluster pulls that CTA's, warp shuffles do the rest
      if (ws != WS_NONE && tid < 32) {
        double m4[4] = {0.0, 0.0, 0.0, 0.0};
        if (tid < nct) {
          const double* r = cluster.map_shared_rank(MAXO + cur * 4, tid);
#pragma unroll
          for (int q = 0; q < 4; ++q) m4[q] = r[q];
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) m4[q] = warp_max(m4[q]);
        if (tid == 0) {
          if (ws == WS_FULL) { MAXS[0] = m4[0]; MAXS[1] = m4[1]; }
          MAXS[2] = m4[2]; MAXS[3] = m4[3];
        }
      }
    }
  }
  // the state, its maxima, dt, t and the status back to global memory
  if (col_out) {
#pragma unroll
    for (int f = 0; f < NF; ++f) la.buf[0].p[f][cell_addr(g, i, 0)] = o[f];
  }
  __syncthreads();
  if (rank == 0 && tid == 0) {
    const int A = (la.n_steps & 1) ? (la.state_set == 0 ? 4 : 0) : la.state_set;
    for (int q = 0; q < 4; ++q) la.sc->red[A][q] = (unsigned long long)__double_as_longlong(MAXS[q]);
    la.sc->dt = dt;
    la.sc->t = t_sim;
    if (bad) la.sc->status = 1;
  }
  cluster.sync();              // no CTA exits while a neighbour may still pull from its shared memory
}

}  // namespace smaug
