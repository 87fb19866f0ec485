// smaug_stage_kernel.cuh -- the fused stage kernel: one launch = one Runge-Kutta stage over the grid.
//
// Per CTA: a TH x TW tile of interior cells plus a 3-cell halo is staged in shared memory as DERIVED
// planes; the flux divergence (c-2, c-3), the hyperdiffusion coefficients and fluxes (c-5), the energy
// source (c-2), the RK combine (c-6) and the wave-speed maxima of the state just written (c-4) are all
// computed in this one pass -- the state is read once and written once per stage.
//
// Phases (separated by __syncthreads):
//   P1  load w (+ background) for tile + halo 3, compute rho, 1/rho, v, eps~, p~_t, store the six HD
//       scalars (+ totals when a background exists) and the cell-centred fluxes F_x, F_y in smem
//   P2  hyperviscosity ratios kappa = c_u v_t M3/M1 at the x- and y-interfaces, computed in register runs
//       of R interfaces per thread (sliding |D1| / |D3| windows, no redundant differences)
//   P3  cell-centred mixed (cross) fluxes G and their energy companions, folded into F_x, F_y
//   P4  per cell: interface-flux differences, central differences of (F - G), source, RK combine, write,
//       wave-speed maxima -> warp shuffles -> one atomicMax pass per CTA
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

template <int TW_, int TH_>
struct Tile {
  static constexpr int TW = TW_, TH = TH_;
  static constexpr int W = TW + 2 * NG, H = TH + 2 * NG;   // staged extent
  static constexpr int P = (W % 2 == 0) ? W + 1 : W;       // odd row pitch -> conflict-free column access
  static constexpr int PLANE = P * H;
};

// plane indices inside the dynamic shared memory
enum {
  S_RHO = 0,  // total rho
  S_VX, S_VY, S_EPS, S_BX, S_BY,      // HD scalars v, eps~, b~   (rho~ = S_RHO when there is no background)
  S_KX0,                              // 5 planes: kappa at x-interfaces for rho~, vx, vy, eps~, by~
  S_KY0 = S_KX0 + 5,                  // 5 planes: kappa at y-interfaces for rho~, vx, vy, eps~, bx~
  S_CX0 = S_KY0 + 5,                  // 5 planes: F_x - G_x for rho, mx, my, e, by
  S_CY0 = S_CX0 + 5,                  // 5 planes: F_y - G_y for rho, mx, my, e, bx
  S_NOBG_END = S_CY0 + 5,
  S_RHOT = S_NOBG_END,                // background only: rho~ (perturbed), total Bx, total By
  S_BXT, S_BYT,
  S_BG_END
};
enum { K_RHO = 0, K_VX = 1, K_VY = 2, K_EPS = 3, K_B = 4 };
enum { C_RHO = 0, C_MX = 1, C_MY = 2, C_E = 3, C_B = 4 };

template <int TW, int TH, bool BG>
constexpr size_t stage_smem_bytes() {
  return (size_t)(BG ? S_BG_END : S_NOBG_END) * Tile<TW, TH>::PLANE * sizeof(double) + 4 * 32 * sizeof(double);
}

// kappa = coef * (M3 / M1) for R consecutive interfaces of one line (c-5).  u points at the cell left of
// the first interface; cells u[-2*s] .. u[(R+2)*s] are read.  Interface k (0..n-1) is written to out[k*os].
template <int R>
__device__ __forceinline__ void kappa_run(const double* __restrict__ u, int s, double cv, double* out,
                                          int os, int n) {
  double uu[R + 5];   // cells -2 .. R+2
#pragma unroll
  for (int k = 0; k < R + 5; ++k) uu[k] = u[(k - 2) * s];
  double d1[R + 4];   // signed D1 at interfaces -2 .. R+1:  D1_m = u_{m+1} - u_m
#pragma unroll
  for (int k = 0; k < R + 4; ++k) d1[k] = uu[k + 1] - uu[k];
  double d3[R + 2];   // |D3| at interfaces -1 .. R:  D3_m = 3 D1_m - (u_{m+2} - u_{m-1})
#pragma unroll
  for (int k = 0; k < R + 2; ++k) d3[k] = fabs(fma(3.0, d1[k + 1], -(uu[k + 3] - uu[k])));
#pragma unroll
  for (int k = 0; k < R; ++k) {
    const double m3 = fmax(fmax(d3[k], d3[k + 1]), d3[k + 2]);
    const double m1 = fmax(fmax(fmax(fabs(d1[k]), fabs(d1[k + 1])), fmax(fabs(d1[k + 2]), fabs(d1[k + 3]))),
                           fabs(d1[k + 4]));
    const double r = m1 > 0.0 ? cv * (m3 / m1) : 0.0;
    if (k < n) out[k * os] = r;
  }
}

template <int TW, int TH, int NT, bool BG, bool HD>
__global__ void __launch_bounds__(NT) stage_kernel(const StageArgs a) {
  using T = Tile<TW, TH>;
  extern __shared__ double smem[];
  double* const red_sh = smem + (size_t)(BG ? S_BG_END : S_NOBG_END) * T::PLANE;
  auto pl = [&](int k) { return smem + (size_t)k * T::PLANE; };
  const Grid& g = a.g;
  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;   // interior coordinates of the tile origin
  const double gamma = a.prm.gamma, gm1 = a.prm.gamma - 1.0;

  // ---------------------------------------------------------------- P1: stage derived planes + fluxes
  for (int idx = tid; idx < T::H * T::W; idx += NT) {
    const int r = idx / T::W, c = idx - r * T::W;
    const int i = min(x0 + c - NG, g.nx + NG - 1), j = min(y0 + r - NG, g.ny + NG - 1);
    const long long ga = cell_addr(g, i, j);
    const double rhot = a.in.p[F_RHO][ga], mx = a.in.p[F_MX][ga], my = a.in.p[F_MY][ga];
    const double et = a.in.p[F_E][ga], bx = a.in.p[F_BX][ga], by = a.in.p[F_BY][ga];
    double rho_b = 0.0, e_b = 0.0, Bbx = 0.0, Bby = 0.0;
    if (BG) {
      rho_b = a.bg.p[BG_RHO][ga]; e_b = a.bg.p[BG_E][ga];
      Bbx = a.bg.p[BG_BX][ga];    Bby = a.bg.p[BG_BY][ga];
    }
    const double rho = BG ? rho_b + rhot : rhot;
    const double rr = 1.0 / rho;
    const double vx = mx * rr, vy = my * rr;
    const double b2h = 0.5 * fma(by, by, bx * bx);
    const double cross = BG ? fma(Bby, by, Bbx * bx) : 0.0;
    const double ke = 0.5 * fma(my, vy, mx * vx);
    const double eps = BG ? ((et - ke) - cross) - b2h : (et - ke) - b2h;
    const double ptt = BG ? fma(gm1, eps, cross + b2h) : fma(gm1, eps, b2h);
    const double Bx = BG ? Bbx + bx : bx, By = BG ? Bby + by : by;
    const int s = r * T::P + c;
    pl(S_RHO)[s] = rho; pl(S_VX)[s] = vx; pl(S_VY)[s] = vy;
    pl(S_EPS)[s] = eps; pl(S_BX)[s] = bx; pl(S_BY)[s] = by;
    if (BG) { pl(S_RHOT)[s] = rhot; pl(S_BXT)[s] = Bx; pl(S_BYT)[s] = By; }
    const double btv = fma(by, vy, bx * vx);                      // b~ . v
    const double Bbv = BG ? fma(Bby, vy, Bbx * vx) : 0.0;         // B_b . v
    const double h = BG ? (et + e_b) + ptt : et + ptt;
    // F_x(rho, mx, my, e, by)      (c-2; F_x(bx) == 0); background terms are exact zeros without one
    pl(S_CX0 + C_RHO)[s] = rho * vx;
    pl(S_CY0 + C_RHO)[s] = rho * vy;
    if (BG) {
      pl(S_CX0 + C_MX)[s] = ((fma(mx, vx, -(bx * bx)) - bx * Bbx) - Bbx * bx) + ptt;
      pl(S_CX0 + C_MY)[s] = (fma(my, vx, -(by * bx)) - by * Bbx) - Bby * bx;
      pl(S_CX0 + C_E)[s] = (fma(vx, h, -(bx * btv)) - bx * Bbv) - Bbx * btv;
      pl(S_CY0 + C_MX)[s] = (fma(mx, vy, -(bx * by)) - bx * Bby) - Bbx * by;
      pl(S_CY0 + C_MY)[s] = ((fma(my, vy, -(by * by)) - by * Bby) - Bby * by) + ptt;
      pl(S_CY0 + C_E)[s] = (fma(vy, h, -(by * btv)) - by * Bbv) - Bby * btv;
    } else {
      pl(S_CX0 + C_MX)[s] = fma(mx, vx, -(bx * bx)) + ptt;
      pl(S_CX0 + C_MY)[s] = fma(my, vx, -(by * bx));
      pl(S_CX0 + C_E)[s] = fma(vx, h, -(bx * btv));
      pl(S_CY0 + C_MX)[s] = fma(mx, vy, -(bx * by));
      pl(S_CY0 + C_MY)[s] = fma(my, vy, -(by * by)) + ptt;
      pl(S_CY0 + C_E)[s] = fma(vy, h, -(by * btv));
    }
    pl(S_CX0 + C_B)[s] = fma(vx, By, -(Bx * vy));                 // F_x(by)
    pl(S_CY0 + C_B)[s] = fma(vy, Bx, -(By * vx));                 // F_y(bx)
  }
  __syncthreads();

  if (HD) {
    // v_t = sqrt(max a^2) + sqrt(max b^2) of the input state (c-5)
    const double vt = sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][2])) +
                      sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][3]));
    const double coef[5] = {a.prm.c_rho * vt, a.prm.c_mom * vt, a.prm.c_mom * vt, a.prm.c_e * vt,
                            a.prm.c_b * vt};
    // ------------------------------------------------------------ P2: kappa at interfaces, register runs
    // x-interfaces (c | c+1), c = 2 .. TW+2, on staged rows 1 .. TH+4; runs of RX interfaces.
    {
      constexpr int RX = 11, NRUN = (TW + 1 + RX - 1) / RX, ROWS = TH + 4;
      const int usrc[5] = {BG ? S_RHOT : S_RHO, S_VX, S_VY, S_EPS, S_BY};
      for (int it = tid; it < 5 * NRUN * ROWS; it += NT) {
        const int f = it / (NRUN * ROWS), rem = it - f * (NRUN * ROWS);
        const int run = rem / ROWS, r = 1 + (rem - run * ROWS);
        const int c0 = 2 + run * RX;
        kappa_run<RX>(pl(usrc[f]) + r * T::P + c0, 1, coef[f], pl(S_KX0 + f) + r * T::P + c0, 1,
                      min(RX, TW + 3 - c0));
      }
    }
    // y-interfaces (r | r+1), r = 2 .. TH+2, on staged columns 1 .. TW+4; runs of RY interfaces.
    {
      constexpr int RY = 9, NRUN = (TH + 1 + RY - 1) / RY, COLS = TW + 4;
      const int usrc[5] = {BG ? S_RHOT : S_RHO, S_VX, S_VY, S_EPS, S_BX};
      for (int it = tid; it < 5 * NRUN * COLS; it += NT) {
        const int f = it / (NRUN * COLS), rem = it - f * (NRUN * COLS);
        const int run = rem / COLS, c = 1 + (rem - run * COLS);
        const int r0 = 2 + run * RY;
        kappa_run<RY>(pl(usrc[f]) + r0 * T::P + c, T::P, coef[f], pl(S_KY0 + f) + r0 * T::P + c, T::P,
                      min(RY, TH + 3 - r0));
      }
    }
    __syncthreads();

    // ------------------------------------------------------------ P3: mixed fluxes folded into F (c-5)
    const int SBX = BG ? S_BXT : S_BX, SBY = BG ? S_BYT : S_BY;
    // G_x (needs y-derivatives): tile rows, staged columns 1 .. TW+4
    for (int idx = tid; idx < TH * (TW + 4); idx += NT) {
      const int r = NG + idx / (TW + 4), c = 1 + idx % (TW + 4);
      const int s = r * T::P + c;
      const double kv = 0.5 * (pl(S_KY0 + K_VX)[s - T::P] + pl(S_KY0 + K_VX)[s]);   // nubar_y(vx)/Delta_y
      const double kb = 0.5 * (pl(S_KY0 + K_B)[s - T::P] + pl(S_KY0 + K_B)[s]);     // nubar_y(bx~)/Delta_y
      const double gm = ((0.5 * pl(S_RHO)[s]) * kv) * (cd12(pl(S_VX) + s, T::P) * (1.0 / 12.0));  // G(my;x)
      const double gb = -(kb * (cd12(pl(S_BX) + s, T::P) * (1.0 / 12.0)));                        // G(by;x)
      pl(S_CX0 + C_MY)[s] -= gm;
      pl(S_CX0 + C_B)[s] -= gb;
      pl(S_CX0 + C_E)[s] -= fma(pl(S_VY)[s], gm, pl(SBY)[s] * gb);
    }
    // G_y (needs x-derivatives): staged rows 1 .. TH+4, tile columns
    for (int idx = tid; idx < (TH + 4) * TW; idx += NT) {
      const int r = 1 + idx / TW, c = NG + idx % TW;
      const int s = r * T::P + c;
      const double kv = 0.5 * (pl(S_KX0 + K_VY)[s - 1] + pl(S_KX0 + K_VY)[s]);      // nubar_x(vy)/Delta_x
      const double kb = 0.5 * (pl(S_KX0 + K_B)[s - 1] + pl(S_KX0 + K_B)[s]);        // nubar_x(by~)/Delta_x
      const double gm = ((0.5 * pl(S_RHO)[s]) * kv) * (cd12(pl(S_VY) + s, 1) * (1.0 / 12.0));     // G(mx;y)
      const double gb = -(kb * (cd12(pl(S_BY) + s, 1) * (1.0 / 12.0)));                           // G(bx;y)
      pl(S_CY0 + C_MX)[s] -= gm;
      pl(S_CY0 + C_B)[s] -= gb;
      pl(S_CY0 + C_E)[s] -= fma(pl(S_VX)[s], gm, pl(SBX)[s] * gb);
    }
    __syncthreads();
  }

  // ---------------------------------------------------------------- P4: per-cell RHS, combine, reduce
  const double dt = a.sc->dt;
  const double cdt = a.c * dt;
  const double idx_ = a.prm.inv_dx, idy_ = a.prm.inv_dy;
  double wsmax[4] = {0.0, 0.0, 0.0, 0.0};
  for (int idx = tid; idx < TH * TW; idx += NT) {
    const int ty = idx / TW, tx = idx - ty * TW;
    const int i = x0 + tx, j = y0 + ty;
    if (i >= g.nx || j >= g.ny) continue;
    const int s = (ty + NG) * T::P + (tx + NG);
    double R[NF];
    // central differences of the (mixed-flux-corrected) fluxes:  -(d^c_x C_x + d^c_y C_y)
    R[F_RHO] = fma(cd12(pl(S_CX0 + C_RHO) + s, 1), idx_, cd12(pl(S_CY0 + C_RHO) + s, T::P) * idy_) * (-1.0 / 12.0);
    R[F_MX] = fma(cd12(pl(S_CX0 + C_MX) + s, 1), idx_, cd12(pl(S_CY0 + C_MX) + s, T::P) * idy_) * (-1.0 / 12.0);
    R[F_MY] = fma(cd12(pl(S_CX0 + C_MY) + s, 1), idx_, cd12(pl(S_CY0 + C_MY) + s, T::P) * idy_) * (-1.0 / 12.0);
    R[F_E] = fma(cd12(pl(S_CX0 + C_E) + s, 1), idx_, cd12(pl(S_CY0 + C_E) + s, T::P) * idy_) * (-1.0 / 12.0);
    R[F_BX] = (cd12(pl(S_CY0 + C_B) + s, T::P) * idy_) * (-1.0 / 12.0);          // F_x(bx) == 0
    R[F_BY] = fma(cd12(pl(S_CX0 + C_B) + s, 1), idx_, 0.0) * (-1.0 / 12.0);       // F_y(by) == 0

    const long long ga = cell_addr(g, i, j);
    double rho_b = 0.0, e_b = 0.0, Bbx = 0.0, Bby = 0.0;
    if (BG) {
      rho_b = a.bg.p[BG_RHO][ga]; e_b = a.bg.p[BG_E][ga];
      Bbx = a.bg.p[BG_BX][ga];    Bby = a.bg.p[BG_BY][ga];
      // energy source S_e = -p_tb div v + B_b B_b : grad v      (c-2)
      const double bb2h = 0.5 * fma(Bby, Bby, Bbx * Bbx);
      const double ptb = fma(gm1, e_b - bb2h, bb2h);
      const double dxvx = (cd12(pl(S_VX) + s, 1) * idx_) * (1.0 / 12.0);
      const double dyvx = (cd12(pl(S_VX) + s, T::P) * idy_) * (1.0 / 12.0);
      const double dxvy = (cd12(pl(S_VY) + s, 1) * idx_) * (1.0 / 12.0);
      const double dyvy = (cd12(pl(S_VY) + s, T::P) * idy_) * (1.0 / 12.0);
      const double S = fma(-ptb, dxvx + dyvy,
                           fma(Bby * Bby, dyvy, fma(Bbx * Bby, dxvy + dyvx, (Bbx * Bbx) * dxvx)));
      R[F_E] = R[F_E] + S;
    }

    if (HD) {
      const int SRT = BG ? S_RHOT : S_RHO, SBX = BG ? S_BXT : S_BX, SBY = BG ? S_BYT : S_BY;
      // interface fluxes Phi = g kappa (q_b - q_a) at the two x- and the two y-interfaces of the cell
      double fx[2][5], fy[2][5];   // [side][rho, mx, my, e, b]
#pragma unroll
      for (int side = 0; side < 2; ++side) {
        {
          const int sa = s - 1 + side, sb = sa + 1;
          const double rbar = 0.5 * (pl(S_RHO)[sa] + pl(S_RHO)[sb]);
          const double p_rho = pl(S_KX0 + K_RHO)[sa] * (pl(SRT)[sb] - pl(SRT)[sa]);
          const double p_mx = (rbar * pl(S_KX0 + K_VX)[sa]) * (pl(S_VX)[sb] - pl(S_VX)[sa]);
          const double p_my = ((0.5 * rbar) * pl(S_KX0 + K_VY)[sa]) * (pl(S_VY)[sb] - pl(S_VY)[sa]);
          const double p_eps = pl(S_KX0 + K_EPS)[sa] * (pl(S_EPS)[sb] - pl(S_EPS)[sa]);
          const double p_b = pl(S_KX0 + K_B)[sa] * (pl(S_BY)[sb] - pl(S_BY)[sa]);
          fx[side][C_RHO] = p_rho; fx[side][C_MX] = p_mx; fx[side][C_MY] = p_my; fx[side][C_B] = p_b;
          fx[side][C_E] = fma(0.5 * (pl(SBY)[sa] + pl(SBY)[sb]), p_b,
                              fma(0.5 * (pl(S_VY)[sa] + pl(S_VY)[sb]), p_my,
                                  fma(0.5 * (pl(S_VX)[sa] + pl(S_VX)[sb]), p_mx, p_eps)));
        }
        {
          const int sa = s + (side - 1) * T::P, sb = sa + T::P;
          const double rbar = 0.5 * (pl(S_RHO)[sa] + pl(S_RHO)[sb]);
          const double p_rho = pl(S_KY0 + K_RHO)[sa] * (pl(SRT)[sb] - pl(SRT)[sa]);
          const double p_mx = ((0.5 * rbar) * pl(S_KY0 + K_VX)[sa]) * (pl(S_VX)[sb] - pl(S_VX)[sa]);
          const double p_my = (rbar * pl(S_KY0 + K_VY)[sa]) * (pl(S_VY)[sb] - pl(S_VY)[sa]);
          const double p_eps = pl(S_KY0 + K_EPS)[sa] * (pl(S_EPS)[sb] - pl(S_EPS)[sa]);
          const double p_b = pl(S_KY0 + K_B)[sa] * (pl(S_BX)[sb] - pl(S_BX)[sa]);
          fy[side][C_RHO] = p_rho; fy[side][C_MX] = p_mx; fy[side][C_MY] = p_my; fy[side][C_B] = p_b;
          fy[side][C_E] = fma(0.5 * (pl(SBX)[sa] + pl(SBX)[sb]), p_b,
                              fma(0.5 * (pl(S_VY)[sa] + pl(S_VY)[sb]), p_my,
                                  fma(0.5 * (pl(S_VX)[sa] + pl(S_VX)[sb]), p_mx, p_eps)));
        }
      }
      R[F_RHO] = fma(fx[1][C_RHO] - fx[0][C_RHO], idx_, R[F_RHO]);
      R[F_MX] = fma(fx[1][C_MX] - fx[0][C_MX], idx_, R[F_MX]);
      R[F_MY] = fma(fx[1][C_MY] - fx[0][C_MY], idx_, R[F_MY]);
      R[F_E] = fma(fx[1][C_E] - fx[0][C_E], idx_, R[F_E]);
      R[F_BY] = fma(fx[1][C_B] - fx[0][C_B], idx_, R[F_BY]);
      R[F_RHO] = fma(fy[1][C_RHO] - fy[0][C_RHO], idy_, R[F_RHO]);
      R[F_MX] = fma(fy[1][C_MX] - fy[0][C_MX], idy_, R[F_MX]);
      R[F_MY] = fma(fy[1][C_MY] - fy[0][C_MY], idy_, R[F_MY]);
      R[F_E] = fma(fy[1][C_E] - fy[0][C_E], idy_, R[F_E]);
      R[F_BX] = fma(fy[1][C_B] - fy[0][C_B], idy_, R[F_BX]);
    }

    // RK combine (c-6) and write
    double o[NF];
    if (a.combine == COMBINE_FINAL) {
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const double w3 = a.in.p[f][ga];
        o[f] = fma(cdt, R[f], fma(fma(-2.0, w3, a.acc_in.p[f][ga]), 1.0 / 3.0, w3));
      }
    } else {
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const double b = a.base.p[f][ga];
        o[f] = fma(cdt, R[f], b);
        if (a.combine == COMBINE_ACC) a.acc_out.p[f][ga] = fma(2.0, o[f], a.in.p[f][ga] - b);
      }
    }
#pragma unroll
    for (int f = 0; f < NF; ++f) a.out.p[f][ga] = o[f];

    if (a.ws_mode != WS_NONE) {
      double w4[4];
      if (BG)
        cell_wavespeeds(rho_b + o[F_RHO], o[F_MX], o[F_MY], e_b + o[F_E], Bbx + o[F_BX], Bby + o[F_BY], gamma,
                        a.ws_mode == WS_FULL, w4);
      else
        cell_wavespeeds(o[F_RHO], o[F_MX], o[F_MY], o[F_E], o[F_BX], o[F_BY], gamma, a.ws_mode == WS_FULL, w4);
#pragma unroll
      for (int k = 0; k < 4; ++k) wsmax[k] = fmax(wsmax[k], w4[k]);
    }
  }
  if (a.ws_mode != WS_NONE)
    block_max4_atomic(wsmax, red_sh, a.sc->red[a.red_out], a.ws_mode == WS_FULL ? 0 : 2);
}

}  // namespace smaug
