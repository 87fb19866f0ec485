// smaug_stage_kernel.cuh -- the fused stage kernel: one launch = one Runge-Kutta stage over the grid.
//
// Per CTA: a TH x TW tile of interior cells plus a 3-cell halo is staged in shared memory as DERIVED
// planes; the flux divergence (c-2, c-3), the hyperdiffusion coefficients and fluxes (c-5), the energy
// source (c-2), the RK combine (c-6) and the wave-speed maxima of the state just written (c-4) are all
// computed in this one pass -- the state is read once and written once per stage.
// Every value follows the arithmetic contract of DESIGN.md section 4 (explicit fma, -fmad=false), so the
// result is bit-identical to the oracle's.
//
// Phases (separated by __syncthreads):
//   P1  load w (+ background) for tile + halo 3, compute rho, 1/rho, v, eps~, p~_t; store the six HD
//       scalars (+ totals when a background exists) and the cell-centred fluxes F_x, F_y where needed
//   P2  hyperviscosity ratios kappa = c_u v_t M3/M1 at the x- and y-interfaces, computed in register runs
//       (one thread slides the |D1| / |D3| windows along R consecutive interfaces: no redundant differences)
//   P3  cell-centred mixed (cross) fluxes G and their energy companions, folded into F_x, F_y
//   P3b interface (diffusive) fluxes Phi, once per interface, written over the kappa planes
//   P4  per cell: central differences of (F - G), interface-flux differences, source, RK combine, write,
//       wave-speed maxima -> warp shuffles -> one atomicMax pass per CTA
#pragma once
#include "smaug_stage_common.cuh"

namespace smaug {

constexpr int odd_up(int v) { return (v % 2 == 0) ? v + 1 : v; }   // odd pitch: conflict-free columns

// Shared-memory layout of one tile.  Staged cell (r, c), r in [0, TH+6), c in [0, TW+6), is interior
// cell (x0 + c - 3, y0 + r - 3).
template <int TW_, int TH_, bool BG>
struct Tile {
  static constexpr int TW = TW_, TH = TH_;
  static constexpr int W = TW + 2 * NG, H = TH + 2 * NG;
  // U planes: H x W, all staged cells
  static constexpr int PU = odd_up(W), U_PLANE = PU * H, NU = BG ? 9 : 6;
  // KX planes (kappa, later Phi, at x-interfaces (c | c+1), c = 2 .. TW+2): rows r = 1 .. TH+4
  static constexpr int PKX = odd_up(TW + 1), KX_PLANE = PKX * (TH + 4);
  // KY planes (y-interfaces (r | r+1), r = 2 .. TH+2): columns c = 1 .. TW+4
  static constexpr int PKY = odd_up(TW + 4), KY_PLANE = PKY * (TH + 1);
  // CX planes (F_x - G_x): tile rows, columns c = 1 .. TW+4;   CY planes: rows r = 1 .. TH+4, tile columns
  static constexpr int PCX = odd_up(TW + 4), CX_PLANE = PCX * TH;
  static constexpr int PCY = odd_up(TW), CY_PLANE = PCY * (TH + 4);
  static constexpr int OFF_U = 0;
  static constexpr int OFF_KX = OFF_U + NU * U_PLANE;
  static constexpr int OFF_KY = OFF_KX + 5 * KX_PLANE;
  static constexpr int OFF_CX = OFF_KY + 5 * KY_PLANE;
  static constexpr int OFF_CY = OFF_CX + 5 * CX_PLANE;
  static constexpr int OFF_RED = OFF_CY + 5 * CY_PLANE;
  static constexpr int TOTAL = OFF_RED + 4 * 32;
  static constexpr size_t BYTES = (size_t)TOTAL * sizeof(double);
  __device__ static int u(int r, int c) { return r * PU + c; }
  __device__ static int kx(int r, int c) { return (r - 1) * PKX + (c - 2); }
  __device__ static int ky(int r, int c) { return (r - 2) * PKY + (c - 1); }
  __device__ static int cx(int r, int c) { return (r - NG) * PCX + (c - 1); }
  __device__ static int cy(int r, int c) { return (r - 1) * PCY + (c - NG); }
};

enum { U_RHO = 0, U_VX, U_VY, U_EPS, U_BX, U_BY, U_RHOT, U_BXT, U_BYT };   // last three: background only

// kappa = cv * (M3 / M1) for n <= R consecutive interfaces of one line (c-5).  u points at the cell left of
// the first interface (interface k lies between cells k and k+1); cells -2 .. R+2 are read with stride s.
// Sliding windows: D1_m = u_{m+1} - u_m;  D3_m = 3 D1_m - (u_{m+2} - u_{m-1});  M3 over m-1..m+1, M1 over m-2..m+2.
template <int R>
__device__ __forceinline__ void kappa_run(const double* __restrict__ u, int s, double cv, double* out,
                                          int os, int n) {
  double uu[R + 5];
#pragma unroll
  for (int k = 0; k < R + 5; ++k) uu[k] = u[(k - 2) * s];
  double d1[R + 4];
#pragma unroll
  for (int k = 0; k < R + 4; ++k) d1[k] = uu[k + 1] - uu[k];                       // interface k-2
  double d3[R + 2];
#pragma unroll
  for (int k = 0; k < R + 2; ++k) d3[k] = dabs(fma(3.0, d1[k + 1], -(uu[k + 3] - uu[k])));   // interface k-1
#pragma unroll
  for (int k = 0; k < R + 4; ++k) d1[k] = dabs(d1[k]);
#pragma unroll
  for (int k = 0; k < R; ++k) {
    const double m3 = dmax(dmax(d3[k], d3[k + 1]), d3[k + 2]);
    const double m1 = dmax(dmax(dmax(d1[k], d1[k + 1]), dmax(d1[k + 2], d1[k + 3])), d1[k + 4]);
    const double r = kappa_ratio(m3, m1, cv);
    if (k < n) out[k * os] = r;
  }
}

// One RK stage on the TH x TW tile whose first interior cell is (x0, y0); all NT threads of the CTA call it together.
// Reads a.in with its halo (ghosts filled), writes the tile's cells of a.out (and a.acc_out), reduces into a.sc->red.
template <int TW, int TH, int NT, bool BG, bool HD>
__device__ __forceinline__ void stage_tile(const StageArgs& a, const int x0, const int y0, double* const smem) {
  using T = Tile<TW, TH, BG>;
  double* const U = smem + T::OFF_U;
  double* const KX = smem + T::OFF_KX;
  double* const KY = smem + T::OFF_KY;
  double* const CX = smem + T::OFF_CX;
  double* const CY = smem + T::OFF_CY;
  double* const red_sh = smem + T::OFF_RED;
  const Grid& g = a.g;
  const int tid = threadIdx.x;
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
    const double rr = drcp(rho);
    const double vx = mx * rr, vy = my * rr;
    const double b2h = 0.5 * fma(by, by, bx * bx);
    const double cross = BG ? fma(Bby, by, Bbx * bx) : 0.0;
    const double ke = 0.5 * fma(my, vy, mx * vx);
    const double eps = BG ? ((et - ke) - cross) - b2h : (et - ke) - b2h;
    const double ptt = BG ? fma(gm1, eps, cross + b2h) : fma(gm1, eps, b2h);
    const double Bx = BG ? Bbx + bx : bx, By = BG ? Bby + by : by;
    const int s = T::u(r, c);
    U[U_RHO * T::U_PLANE + s] = rho; U[U_VX * T::U_PLANE + s] = vx; U[U_VY * T::U_PLANE + s] = vy;
    U[U_EPS * T::U_PLANE + s] = eps; U[U_BX * T::U_PLANE + s] = bx; U[U_BY * T::U_PLANE + s] = by;
    if (BG) {
      U[U_RHOT * T::U_PLANE + s] = rhot; U[U_BXT * T::U_PLANE + s] = Bx; U[U_BYT * T::U_PLANE + s] = By;
    }
    const bool in_rows = r >= NG && r < NG + TH, in_cols = c >= NG && c < NG + TW;
    const bool need_x = in_rows && c >= 1 && c <= TW + 4, need_y = in_cols && r >= 1 && r <= TH + 4;
    if (need_x || need_y) {
      const double btv = fma(by, vy, bx * vx);                      // b~ . v
      const double Bbv = BG ? fma(Bby, vy, Bbx * vx) : 0.0;         // B_b . v
      const double h = BG ? (et + e_b) + ptt : et + ptt;
      if (need_x) {   // F_x(rho, mx, my, e, by)   (c-2; F_x(bx) == 0)
        double* cxp = CX + T::cx(r, c);
        cxp[C_RHO * T::CX_PLANE] = rho * vx;
        if (BG) {
          cxp[C_MX * T::CX_PLANE] = ((fma(mx, vx, -(bx * bx)) - bx * Bbx) - Bbx * bx) + ptt;
          cxp[C_MY * T::CX_PLANE] = (fma(my, vx, -(by * bx)) - by * Bbx) - Bby * bx;
          cxp[C_E * T::CX_PLANE] = (fma(vx, h, -(bx * btv)) - bx * Bbv) - Bbx * btv;
        } else {
          cxp[C_MX * T::CX_PLANE] = fma(mx, vx, -(bx * bx)) + ptt;
          cxp[C_MY * T::CX_PLANE] = fma(my, vx, -(by * bx));
          cxp[C_E * T::CX_PLANE] = fma(vx, h, -(bx * btv));
        }
        cxp[C_B * T::CX_PLANE] = fma(vx, By, -(Bx * vy));
      }
      if (need_y) {   // F_y(rho, mx, my, e, bx)   (F_y(by) == 0)
        double* cyp = CY + T::cy(r, c);
        cyp[C_RHO * T::CY_PLANE] = rho * vy;
        if (BG) {
          cyp[C_MX * T::CY_PLANE] = (fma(mx, vy, -(bx * by)) - bx * Bby) - Bbx * by;
          cyp[C_MY * T::CY_PLANE] = ((fma(my, vy, -(by * by)) - by * Bby) - Bby * by) + ptt;
          cyp[C_E * T::CY_PLANE] = (fma(vy, h, -(by * btv)) - by * Bbv) - Bby * btv;
        } else {
          cyp[C_MX * T::CY_PLANE] = fma(mx, vy, -(bx * by));
          cyp[C_MY * T::CY_PLANE] = fma(my, vy, -(by * by)) + ptt;
          cyp[C_E * T::CY_PLANE] = fma(vy, h, -(by * btv));
        }
        cyp[C_B * T::CY_PLANE] = fma(vy, Bx, -(By * vx));
      }
    }
  }
  __syncthreads();

  constexpr int URT = BG ? U_RHOT : U_RHO, UBXT = BG ? U_BXT : U_BX, UBYT = BG ? U_BYT : U_BY;
  if (HD) {
    // v_t = sqrt(max a^2) + sqrt(max b^2) of the input state (c-5)
    const double vt = sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][2])) +
                      sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][3]));
    // ------------------------------------------------------------ P2: kappa at interfaces, register runs
    // x-interfaces (c | c+1), c = 2 .. TW+2.  Families rho~, vx, eps~ on tile rows; vy, by~ on rows 1 .. TH+4.
    {
      constexpr int RX = 11, NRUN = (TW + 1 + RX - 1) / RX;
      constexpr int N_TILE = 3 * TH * NRUN, N_WIDE = 2 * (TH + 4) * NRUN;
      for (int it = tid; it < N_TILE + N_WIDE; it += NT) {
        int f, run, r;
        if (it < N_TILE) {
          const int q = it / TH;
          r = NG + (it - q * TH);
          f = q / NRUN; run = q - f * NRUN;
          f = f == 0 ? K_RHO : (f == 1 ? K_VX : K_EPS);
        } else {
          const int it2 = it - N_TILE, q = it2 / (TH + 4);
          r = 1 + (it2 - q * (TH + 4));
          f = q / NRUN; run = q - f * NRUN;
          f = f == 0 ? K_VY : K_B;
        }
        const int up = f == K_RHO ? URT : (f == K_VX ? U_VX : (f == K_VY ? U_VY : (f == K_EPS ? U_EPS : U_BY)));
        const double cf = f == K_RHO ? a.prm.c_rho : (f == K_EPS ? a.prm.c_e : (f == K_B ? a.prm.c_b : a.prm.c_mom));
        const int c0 = 2 + run * RX;
        kappa_run<RX>(U + up * T::U_PLANE + T::u(r, c0), 1, cf * vt, KX + f * T::KX_PLANE + T::kx(r, c0), 1,
                      min(RX, TW + 3 - c0));
      }
    }
    // y-interfaces (r | r+1), r = 2 .. TH+2.  Families rho~, vy, eps~ on tile columns; vx, bx~ on columns 1 .. TW+4.
    {
      constexpr int RY = 9, NRUN = (TH + 1 + RY - 1) / RY;
      constexpr int N_TILE = 3 * TW * NRUN, N_WIDE = 2 * (TW + 4) * NRUN;
      for (int it = tid; it < N_TILE + N_WIDE; it += NT) {
        int f, run, c;
        if (it < N_TILE) {
          const int q = it / TW;
          c = NG + (it - q * TW);
          f = q / NRUN; run = q - f * NRUN;
          f = f == 0 ? K_RHO : (f == 1 ? K_VY : K_EPS);
        } else {
          const int it2 = it - N_TILE, q = it2 / (TW + 4);
          c = 1 + (it2 - q * (TW + 4));
          f = q / NRUN; run = q - f * NRUN;
          f = f == 0 ? K_VX : K_B;
        }
        const int up = f == K_RHO ? URT : (f == K_VX ? U_VX : (f == K_VY ? U_VY : (f == K_EPS ? U_EPS : U_BX)));
        const double cf = f == K_RHO ? a.prm.c_rho : (f == K_EPS ? a.prm.c_e : (f == K_B ? a.prm.c_b : a.prm.c_mom));
        const int r0 = 2 + run * RY;
        kappa_run<RY>(U + up * T::U_PLANE + T::u(r0, c), T::PU, cf * vt, KY + f * T::KY_PLANE + T::ky(r0, c),
                      T::PKY, min(RY, TH + 3 - r0));
      }
    }
    __syncthreads();

    // ------------------------------------------------------------ P3: mixed fluxes folded into F (c-5)
    // G(. ; x) needs y-derivatives: tile rows, staged columns 1 .. TW+4
    for (int idx = tid; idx < TH * (TW + 4); idx += NT) {
      const int q = idx / (TW + 4);
      const int r = NG + q, c = 1 + (idx - q * (TW + 4));
      const int s = T::u(r, c), k = T::ky(r, c);
      const double kv = 0.5 * (KY[K_VX * T::KY_PLANE + k - T::PKY] + KY[K_VX * T::KY_PLANE + k]);
      const double kb = 0.5 * (KY[K_B * T::KY_PLANE + k - T::PKY] + KY[K_B * T::KY_PLANE + k]);
      const double gm = ((0.5 * U[U_RHO * T::U_PLANE + s]) * kv) *
                        (cd12(U + U_VX * T::U_PLANE + s, T::PU) * (1.0 / 12.0));          // G(my ; x)
      const double gb = -(kb * (cd12(U + U_BX * T::U_PLANE + s, T::PU) * (1.0 / 12.0)));   // G(by ; x)
      double* cxp = CX + T::cx(r, c);
      cxp[C_MY * T::CX_PLANE] -= gm;
      cxp[C_B * T::CX_PLANE] -= gb;
      cxp[C_E * T::CX_PLANE] -= fma(U[U_VY * T::U_PLANE + s], gm, U[UBYT * T::U_PLANE + s] * gb);
    }
    // G(. ; y) needs x-derivatives: staged rows 1 .. TH+4, tile columns
    for (int idx = tid; idx < (TH + 4) * TW; idx += NT) {
      const int q = idx / TW;
      const int r = 1 + q, c = NG + (idx - q * TW);
      const int s = T::u(r, c), k = T::kx(r, c);
      const double kv = 0.5 * (KX[K_VY * T::KX_PLANE + k - 1] + KX[K_VY * T::KX_PLANE + k]);
      const double kb = 0.5 * (KX[K_B * T::KX_PLANE + k - 1] + KX[K_B * T::KX_PLANE + k]);
      const double gm = ((0.5 * U[U_RHO * T::U_PLANE + s]) * kv) *
                        (cd12(U + U_VY * T::U_PLANE + s, 1) * (1.0 / 12.0));               // G(mx ; y)
      const double gb = -(kb * (cd12(U + U_BY * T::U_PLANE + s, 1) * (1.0 / 12.0)));        // G(bx ; y)
      double* cyp = CY + T::cy(r, c);
      cyp[C_MX * T::CY_PLANE] -= gm;
      cyp[C_B * T::CY_PLANE] -= gb;
      cyp[C_E * T::CY_PLANE] -= fma(U[U_VX * T::U_PLANE + s], gm, U[UBXT * T::U_PLANE + s] * gb);
    }
    __syncthreads();

    // ------------------------------------------------------------ P3b: interface fluxes, once per interface
    // Phi = g kappa (q_b - q_a), written over kappa.  x-interfaces (c | c+1), c = 2 .. TW+2, tile rows.
    for (int idx = tid; idx < TH * (TW + 1); idx += NT) {
      const int q = idx / (TW + 1);
      const int r = NG + q, c = 2 + (idx - q * (TW + 1));
      const int sa = T::u(r, c), sb = sa + 1;
      double* kp = KX + T::kx(r, c);
      const double rbar = 0.5 * (U[U_RHO * T::U_PLANE + sa] + U[U_RHO * T::U_PLANE + sb]);
      const double vxa = U[U_VX * T::U_PLANE + sa], vxb = U[U_VX * T::U_PLANE + sb];
      const double vya = U[U_VY * T::U_PLANE + sa], vyb = U[U_VY * T::U_PLANE + sb];
      const double p_rho = kp[K_RHO * T::KX_PLANE] * (U[URT * T::U_PLANE + sb] - U[URT * T::U_PLANE + sa]);
      const double p_mx = (rbar * kp[K_VX * T::KX_PLANE]) * (vxb - vxa);
      const double p_my = ((0.5 * rbar) * kp[K_VY * T::KX_PLANE]) * (vyb - vya);
      const double p_eps = kp[K_EPS * T::KX_PLANE] * (U[U_EPS * T::U_PLANE + sb] - U[U_EPS * T::U_PLANE + sa]);
      const double p_b = kp[K_B * T::KX_PLANE] * (U[U_BY * T::U_PLANE + sb] - U[U_BY * T::U_PLANE + sa]);
      const double Bbar = 0.5 * (U[UBYT * T::U_PLANE + sa] + U[UBYT * T::U_PLANE + sb]);
      kp[C_RHO * T::KX_PLANE] = p_rho; kp[C_MX * T::KX_PLANE] = p_mx; kp[C_MY * T::KX_PLANE] = p_my;
      kp[C_B * T::KX_PLANE] = p_b;
      kp[C_E * T::KX_PLANE] = fma(Bbar, p_b, fma(0.5 * (vya + vyb), p_my, fma(0.5 * (vxa + vxb), p_mx, p_eps)));
    }
    // y-interfaces (r | r+1), r = 2 .. TH+2, tile columns.
    for (int idx = tid; idx < (TH + 1) * TW; idx += NT) {
      const int q = idx / TW;
      const int r = 2 + q, c = NG + (idx - q * TW);
      const int sa = T::u(r, c), sb = sa + T::PU;
      double* kp = KY + T::ky(r, c);
      const double rbar = 0.5 * (U[U_RHO * T::U_PLANE + sa] + U[U_RHO * T::U_PLANE + sb]);
      const double vxa = U[U_VX * T::U_PLANE + sa], vxb = U[U_VX * T::U_PLANE + sb];
      const double vya = U[U_VY * T::U_PLANE + sa], vyb = U[U_VY * T::U_PLANE + sb];
      const double p_rho = kp[K_RHO * T::KY_PLANE] * (U[URT * T::U_PLANE + sb] - U[URT * T::U_PLANE + sa]);
      const double p_mx = ((0.5 * rbar) * kp[K_VX * T::KY_PLANE]) * (vxb - vxa);
      const double p_my = (rbar * kp[K_VY * T::KY_PLANE]) * (vyb - vya);
      const double p_eps = kp[K_EPS * T::KY_PLANE] * (U[U_EPS * T::U_PLANE + sb] - U[U_EPS * T::U_PLANE + sa]);
      const double p_b = kp[K_B * T::KY_PLANE] * (U[U_BX * T::U_PLANE + sb] - U[U_BX * T::U_PLANE + sa]);
      const double Bbar = 0.5 * (U[UBXT * T::U_PLANE + sa] + U[UBXT * T::U_PLANE + sb]);
      kp[C_RHO * T::KY_PLANE] = p_rho; kp[C_MX * T::KY_PLANE] = p_mx; kp[C_MY * T::KY_PLANE] = p_my;
      kp[C_B * T::KY_PLANE] = p_b;
      kp[C_E * T::KY_PLANE] = fma(Bbar, p_b, fma(0.5 * (vya + vyb), p_my, fma(0.5 * (vxa + vxb), p_mx, p_eps)));
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
    const int r = ty + NG, c = tx + NG;
    const double* cxp = CX + T::cx(r, c);
    const double* cyp = CY + T::cy(r, c);
    double R[NF];
    // central differences of the (mixed-flux-corrected) fluxes:  -(d^c_x C_x + d^c_y C_y)
    R[F_RHO] = fma(cd12(cxp + C_RHO * T::CX_PLANE, 1), idx_, cd12(cyp + C_RHO * T::CY_PLANE, T::PCY) * idy_) * (-1.0 / 12.0);
    R[F_MX] = fma(cd12(cxp + C_MX * T::CX_PLANE, 1), idx_, cd12(cyp + C_MX * T::CY_PLANE, T::PCY) * idy_) * (-1.0 / 12.0);
    R[F_MY] = fma(cd12(cxp + C_MY * T::CX_PLANE, 1), idx_, cd12(cyp + C_MY * T::CY_PLANE, T::PCY) * idy_) * (-1.0 / 12.0);
    R[F_E] = fma(cd12(cxp + C_E * T::CX_PLANE, 1), idx_, cd12(cyp + C_E * T::CY_PLANE, T::PCY) * idy_) * (-1.0 / 12.0);
    R[F_BX] = (cd12(cyp + C_B * T::CY_PLANE, T::PCY) * idy_) * (-1.0 / 12.0);         // F_x(bx) == 0
    R[F_BY] = fma(cd12(cxp + C_B * T::CX_PLANE, 1), idx_, 0.0) * (-1.0 / 12.0);        // F_y(by) == 0

    const long long ga = cell_addr(g, i, j);
    double rho_b = 0.0, e_b = 0.0, Bbx = 0.0, Bby = 0.0;
    if (BG) {
      rho_b = a.bg.p[BG_RHO][ga]; e_b = a.bg.p[BG_E][ga];
      Bbx = a.bg.p[BG_BX][ga];    Bby = a.bg.p[BG_BY][ga];
      // energy source S_e = -p_tb div v + B_b B_b : grad v      (c-2)
      const int s = T::u(r, c);
      const double bb2h = 0.5 * fma(Bby, Bby, Bbx * Bbx);
      const double ptb = fma(gm1, e_b - bb2h, bb2h);
      const double dxvx = (cd12(U + U_VX * T::U_PLANE + s, 1) * idx_) * (1.0 / 12.0);
      const double dyvx = (cd12(U + U_VX * T::U_PLANE + s, T::PU) * idy_) * (1.0 / 12.0);
      const double dxvy = (cd12(U + U_VY * T::U_PLANE + s, 1) * idx_) * (1.0 / 12.0);
      const double dyvy = (cd12(U + U_VY * T::U_PLANE + s, T::PU) * idy_) * (1.0 / 12.0);
      const double S = fma(-ptb, dxvx + dyvy,
                           fma(Bby * Bby, dyvy, fma(Bbx * Bby, dxvy + dyvx, (Bbx * Bbx) * dxvx)));
      R[F_E] = R[F_E] + S;
    }
    if (a.prm.grav_on) {
      // gravity in the split form (c-10): S(m) = rho~ g, S(e) = rho~ (g.v), on the PERTURBED density
      const int s = T::u(r, c);
      const double rt = U[URT * T::U_PLANE + s];
      const double gv = fma(a.prm.gy, U[U_VY * T::U_PLANE + s], a.prm.gx * U[U_VX * T::U_PLANE + s]);
      R[F_MX] = fma(rt, a.prm.gx, R[F_MX]);
      R[F_MY] = fma(rt, a.prm.gy, R[F_MY]);
      R[F_E] = fma(rt, gv, R[F_E]);
    }

    if (HD) {
      const double* px = KX + T::kx(r, c);      // interface (c | c+1); (c-1 | c) is at px[-1]
      const double* py = KY + T::ky(r, c);      // interface (r | r+1); (r-1 | r) is at py[-PKY]
      R[F_RHO] = fma(px[C_RHO * T::KX_PLANE] - px[C_RHO * T::KX_PLANE - 1], idx_, R[F_RHO]);
      R[F_MX] = fma(px[C_MX * T::KX_PLANE] - px[C_MX * T::KX_PLANE - 1], idx_, R[F_MX]);
      R[F_MY] = fma(px[C_MY * T::KX_PLANE] - px[C_MY * T::KX_PLANE - 1], idx_, R[F_MY]);
      R[F_E] = fma(px[C_E * T::KX_PLANE] - px[C_E * T::KX_PLANE - 1], idx_, R[F_E]);
      R[F_BY] = fma(px[C_B * T::KX_PLANE] - px[C_B * T::KX_PLANE - 1], idx_, R[F_BY]);
      R[F_RHO] = fma(py[C_RHO * T::KY_PLANE] - py[C_RHO * T::KY_PLANE - T::PKY], idy_, R[F_RHO]);
      R[F_MX] = fma(py[C_MX * T::KY_PLANE] - py[C_MX * T::KY_PLANE - T::PKY], idy_, R[F_MX]);
      R[F_MY] = fma(py[C_MY * T::KY_PLANE] - py[C_MY * T::KY_PLANE - T::PKY], idy_, R[F_MY]);
      R[F_E] = fma(py[C_E * T::KY_PLANE] - py[C_E * T::KY_PLANE - T::PKY], idy_, R[F_E]);
      R[F_BX] = fma(py[C_B * T::KY_PLANE] - py[C_B * T::KY_PLANE - T::PKY], idy_, R[F_BX]);
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
      for (int k = 0; k < 4; ++k) wsmax[k] = dmax(wsmax[k], w4[k]);
    }
  }
  if (a.ws_mode != WS_NONE)
    block_max4_atomic(wsmax, red_sh, a.sc->red[a.red_out], a.ws_mode == WS_FULL ? 0 : 2);
}

template <int TW, int TH, int NT, bool BG, bool HD>
__global__ void __launch_bounds__(NT) stage_kernel(const StageArgs a) {
  extern __shared__ double smem[];
  stage_tile<TW, TH, NT, BG, HD>(a, blockIdx.x * TW, blockIdx.y * TH, smem);
}

}  // namespace smaug
