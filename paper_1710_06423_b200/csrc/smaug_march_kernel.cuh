// smaug_march_kernel.cuh -- the streaming ("marching") form of the fused stage kernel, used when there is
// no background and hyperdiffusion is on (the benchmark configurations).
//
// One CTA owns a strip of W = NT - 6 output columns (thread t <-> column x0 - 3 + t) and marches down a
// chunk of rows.  Everything that differences along y lives in the marching thread: six-row register
// histories of the five y-families, thread-private shared-memory rings for the y-fluxes; everything that
// differences along x goes through three small row buffers in shared memory (two __syncthreads per row).
// No cell is staged twice, there is no y-halo recompute, the x-halo costs 6/NT, and global memory is read
// as perfectly coalesced rows.  Arithmetic: the contract of DESIGN.md section 4, bit-identical to the oracle.
//
// Pipeline at step r (newest row r, output row j = r - 3):
//   head  : derived(r); publish the x-families of row r; F_y(r)
//   tail A: kappa_y and Phi_y at interface (j | j+1) from the histories; G(. ; x)(j); C_x(j) = F_x(j) - G; publish
//   -- sync --
//   head  : kappa_x and Phi_x at (i | i+1) of row r from the neighbours; publish them
//   tail B: central x-difference of C_x(j)
//   -- sync --
//   head  : Phi_x difference of row r -> ring; G(. ; y)(r); C_y(r) = F_y(r) - G -> ring
//   tail C: central y-difference of C_y(j) from the ring; R(j); RK combine; write row j; wave-speed maxima
#pragma once
#include "smaug_stage_common.cuh"

namespace smaug {

template <int NT>
struct MarchSmem {
  static constexpr int PW = NT + 8;          // padded row-buffer width (index tid + 4)
  static constexpr int OFF_UP = 0;           // 5 planes: rho, vx, vy, eps, by of the head row
  static constexpr int OFF_CXP = OFF_UP + 5 * PW;     // 5 planes: C_x of the tail row
  static constexpr int OFF_PK = OFF_CXP + 5 * PW;     // 7 planes: Phi_x[5], kappa_x(vy), kappa_x(by)
  static constexpr int OFF_DXR = OFF_PK + 7 * PW;     // ring 4 rows x 5: Phi_x differences (thread-private)
  static constexpr int OFF_CYR = OFF_DXR + 4 * 5 * NT;  // ring 6 rows x 5: C_y (thread-private)
  static constexpr int OFF_INR = OFF_CYR + 6 * 5 * NT;  // ring 4 rows x 6: cp.async landing zone of the input rows
  static constexpr int OFF_TLR = OFF_INR + 4 * 6 * NT;  // ring 4 rows x 3: raw mx, my, e of the rows r-3 .. r
  static constexpr int OFF_RED = OFF_TLR + 4 * 3 * NT;
  static constexpr int TOTAL = OFF_RED + 4 * 32;
  static constexpr size_t BYTES = (size_t)TOTAL * sizeof(double);
};

template <int NT>
__global__ void __launch_bounds__(NT, 1) march_kernel(const StageArgs a, const MarchGeom mg) {
  using S = MarchSmem<NT>;
  extern __shared__ double smem[];
  double* const UP = smem + S::OFF_UP;
  double* const CXP = smem + S::OFF_CXP;
  double* const PK = smem + S::OFF_PK;
  double* const DXR = smem + S::OFF_DXR;
  double* const CYR = smem + S::OFF_CYR;
  double* const INR = smem + S::OFF_INR;
  double* const TLR = smem + S::OFF_TLR;
  double* const red_sh = smem + S::OFF_RED;
  constexpr int PW = S::PW;
  const Grid& g = a.g;
  const int tid = threadIdx.x, tp = tid + 4;
  const int W = NT - 2 * NG;
  const int x0 = blockIdx.x * W;
  const int ci = x0 - NG + tid;                          // interior column of this thread
  const int cl = min(ci, g.nx + NG - 1);                 // clamped for loads
  const int ystart = blockIdx.y * mg.rows_per_cta;
  const int yend = min(ystart + mg.rows_per_cta, g.ny);
  const bool col_out = tid >= NG && tid < NT - NG && ci < g.nx;
  const double gm1 = a.prm.gamma - 1.0, gamma = a.prm.gamma;
  const double idx_ = a.prm.inv_dx, idy_ = a.prm.inv_dy;
  const double vt = sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][2])) +
                    sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][3]));
  const double cv_rho = a.prm.c_rho * vt, cv_mom = a.prm.c_mom * vt, cv_e = a.prm.c_e * vt, cv_b = a.prm.c_b * vt;
  const double dt = a.sc->dt;
  const double cdt = a.c * dt;
  const int combine = a.combine, ws_mode = a.ws_mode;

  // six-row histories (index 0 = row r-5 ... 5 = row r) of the y-families, four rows of by
  double hr[6], hvx[6], hvy[6], he[6], hbx[6], hby[4];
#pragma unroll
  for (int k = 0; k < 6; ++k) { hr[k] = 1.0; hvx[k] = 0.0; hvy[k] = 0.0; he[k] = 0.0; hbx[k] = 0.0; }
#pragma unroll
  for (int k = 0; k < 4; ++k) hby[k] = 0.0;
  double py_prev[5] = {0.0, 0.0, 0.0, 0.0, 0.0};        // Phi_y at interface (j-1 | j)
  double kyv_prev = 0.0, kyb_prev = 0.0;                 // kappa_y(vx), kappa_y(bx) at (j-1 | j)
  double wsmax[4] = {0.0, 0.0, 0.0, 0.0};

  const long long colbase = (long long)NG * g.pitch + (cl + XOFF);   // address of (cl, row 0)
  // the input rows arrive two steps ahead through cp.async into a thread-private ring (no registers held)
  auto fetch_row = [&](int row) {
    const long long ga = colbase + (long long)min(row, g.ny + NG - 1) * g.pitch;
    const int slot = (row + 4096) & 3;
#pragma unroll
    for (int f = 0; f < NF; ++f) cp_async8(INR + (slot * NF + f) * NT + tid, a.in.p[f] + ga);
    cp_async_commit();
  };
  fetch_row(ystart - NG);
  fetch_row(ystart - NG + 1);
  int s6 = 0;                                             // ring slot (mod 6) of row r in CYR

#pragma unroll 1
  for (int r = ystart - NG; r < yend + NG; ++r) {
    const int j = r - NG;                                 // tail (output) row
    const bool tail_on = j >= ystart;                     // uniform over the CTA
    const bool ky_on = r >= ystart + NG - 1;              // six rows of history are valid
    cp_async_wait<1>();                                   // row r has landed (row r+1 may be in flight)
    const int slot4 = (r + 4096) & 3;
    const double rho = INR[(slot4 * NF + F_RHO) * NT + tid], mx = INR[(slot4 * NF + F_MX) * NT + tid];
    const double my = INR[(slot4 * NF + F_MY) * NT + tid], et = INR[(slot4 * NF + F_E) * NT + tid];
    const double bx = INR[(slot4 * NF + F_BX) * NT + tid], by = INR[(slot4 * NF + F_BY) * NT + tid];
    fetch_row(r + 2);
    TLR[(slot4 * 3 + 0) * NT + tid] = mx; TLR[(slot4 * 3 + 1) * NT + tid] = my; TLR[(slot4 * 3 + 2) * NT + tid] = et;
    const long long gj = colbase + (long long)max(j, -NG) * g.pitch;

    // ------------------------------------------------------------------ head: derived quantities of row r
    const double rr = drcp(rho);
    const double vx = mx * rr, vy = my * rr;
    const double b2h = 0.5 * fma(by, by, bx * bx);
    const double ke = 0.5 * fma(my, vy, mx * vx);
    const double eps = (et - ke) - b2h;
    const double ptt = fma(gm1, eps, b2h);
    const double btv = fma(by, vy, bx * vx);
    const double h = et + ptt;
#pragma unroll
    for (int k = 0; k < 5; ++k) { hr[k] = hr[k + 1]; hvx[k] = hvx[k + 1]; hvy[k] = hvy[k + 1]; he[k] = he[k + 1]; hbx[k] = hbx[k + 1]; }
    hr[5] = rho; hvx[5] = vx; hvy[5] = vy; he[5] = eps; hbx[5] = bx;
#pragma unroll
    for (int k = 0; k < 3; ++k) hby[k] = hby[k + 1];
    hby[3] = by;
    UP[0 * PW + tp] = rho; UP[1 * PW + tp] = vx; UP[2 * PW + tp] = vy; UP[3 * PW + tp] = eps; UP[4 * PW + tp] = by;
    // F_y(rho, mx, my, e, bx) of row r
    double cyn[5];
    cyn[C_RHO] = rho * vy;
    cyn[C_MX] = fma(mx, vy, -(bx * by));
    cyn[C_MY] = fma(my, vy, -(by * by)) + ptt;
    cyn[C_E] = fma(vy, h, -(by * btv));
    cyn[C_B] = fma(vy, bx, -(by * vx));

    // ------------------------------------------------------------------ tail A: y-interface (j | j+1), C_x(j)
    double py[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    double kyv = 0.0, kyb = 0.0;
    if (ky_on) {
      double d_rho, d_vx, d_vy, d_e, d_bx;
      const double k_rho = kappa6(hr[0], hr[1], hr[2], hr[3], hr[4], hr[5], cv_rho, d_rho);
      kyv = kappa6(hvx[0], hvx[1], hvx[2], hvx[3], hvx[4], hvx[5], cv_mom, d_vx);
      const double k_vy = kappa6(hvy[0], hvy[1], hvy[2], hvy[3], hvy[4], hvy[5], cv_mom, d_vy);
      const double k_e = kappa6(he[0], he[1], he[2], he[3], he[4], he[5], cv_e, d_e);
      kyb = kappa6(hbx[0], hbx[1], hbx[2], hbx[3], hbx[4], hbx[5], cv_b, d_bx);
      const double rbar = 0.5 * (hr[2] + hr[3]);
      const double p_rho = k_rho * d_rho;
      const double p_mx = ((0.5 * rbar) * kyv) * d_vx;
      const double p_my = (rbar * k_vy) * d_vy;
      const double p_eps = k_e * d_e;
      const double p_b = kyb * d_bx;
      py[C_RHO] = p_rho; py[C_MX] = p_mx; py[C_MY] = p_my; py[C_B] = p_b;
      py[C_E] = fma(0.5 * (hbx[2] + hbx[3]), p_b,
                    fma(0.5 * (hvy[2] + hvy[3]), p_my, fma(0.5 * (hvx[2] + hvx[3]), p_mx, p_eps)));
    }
    if (tail_on) {
      // G(my ; x), G(by ; x) and their energy companion at (ci, j); histories index 2 = row j
      const double kv = 0.5 * (kyv_prev + kyv);
      const double kb = 0.5 * (kyb_prev + kyb);
      const double gm = ((0.5 * hr[2]) * kv) * (cd12v(hvx[0], hvx[1], hvx[3], hvx[4]) * (1.0 / 12.0));
      const double gb = -(kb * (cd12v(hbx[0], hbx[1], hbx[3], hbx[4]) * (1.0 / 12.0)));
      // F_x(rho, mx, my, e, by) of row j
      const int js = (j + 4096) & 3;
      const double jmx = TLR[(js * 3 + 0) * NT + tid], jmy = TLR[(js * 3 + 1) * NT + tid], jet = TLR[(js * 3 + 2) * NT + tid];
      const double jrho = hr[2], jvx = hvx[2], jvy = hvy[2], jeps = he[2], jbx = hbx[2], jby = hby[0];
      const double jb2h = 0.5 * fma(jby, jby, jbx * jbx);
      const double jptt = fma(gm1, jeps, jb2h);
      const double jbtv = fma(jby, jvy, jbx * jvx);
      const double jh = jet + jptt;
      CXP[C_RHO * PW + tp] = jrho * jvx;
      CXP[C_MX * PW + tp] = fma(jmx, jvx, -(jbx * jbx)) + jptt;
      CXP[C_MY * PW + tp] = fma(jmy, jvx, -(jby * jbx)) - gm;
      CXP[C_E * PW + tp] = fma(jvx, jh, -(jbx * jbtv)) - fma(jvy, gm, jby * gb);
      CXP[C_B * PW + tp] = fma(jvx, jby, -(jbx * jvy)) - gb;
    }
    __syncthreads();

    // operands of the RK combine for row j: issued here, consumed at the end of the step
    double jbase[NF], jacc[NF], jin[NF];
    if (tail_on) {
      if (combine == COMBINE_FINAL) {
#pragma unroll
        for (int f = 0; f < NF; ++f) { jin[f] = a.in.p[f][gj]; jacc[f] = a.acc_in.p[f][gj]; }
      } else {
#pragma unroll
        for (int f = 0; f < NF; ++f) jbase[f] = a.base.p[f][gj];
        if (combine == COMBINE_ACC) {
#pragma unroll
          for (int f = 0; f < NF; ++f) jin[f] = a.in.p[f][gj];
        }
      }
    }

    // ------------------------------------------------------------------ head: x-interface (ci | ci+1) of row r
    double px[5], kxv, kxb, dcx_vy, dcx_by;
    {
      double um2, um1, up1, up2, up3, d;
      um2 = UP[0 * PW + tp - 2]; um1 = UP[0 * PW + tp - 1]; up1 = UP[0 * PW + tp + 1]; up2 = UP[0 * PW + tp + 2]; up3 = UP[0 * PW + tp + 3];
      const double k_rho = kappa6(um2, um1, rho, up1, up2, up3, cv_rho, d);
      const double rbar = 0.5 * (rho + up1);
      px[C_RHO] = k_rho * d;
      um2 = UP[1 * PW + tp - 2]; um1 = UP[1 * PW + tp - 1]; up1 = UP[1 * PW + tp + 1]; up2 = UP[1 * PW + tp + 2]; up3 = UP[1 * PW + tp + 3];
      const double k_vx = kappa6(um2, um1, vx, up1, up2, up3, cv_mom, d);
      px[C_MX] = (rbar * k_vx) * d;
      const double vxbar = 0.5 * (vx + up1);
      um2 = UP[2 * PW + tp - 2]; um1 = UP[2 * PW + tp - 1]; up1 = UP[2 * PW + tp + 1]; up2 = UP[2 * PW + tp + 2]; up3 = UP[2 * PW + tp + 3];
      kxv = kappa6(um2, um1, vy, up1, up2, up3, cv_mom, d);
      px[C_MY] = ((0.5 * rbar) * kxv) * d;
      const double vybar = 0.5 * (vy + up1);
      dcx_vy = cd12v(um2, um1, up1, up2);
      um2 = UP[3 * PW + tp - 2]; um1 = UP[3 * PW + tp - 1]; up1 = UP[3 * PW + tp + 1]; up2 = UP[3 * PW + tp + 2]; up3 = UP[3 * PW + tp + 3];
      const double k_e = kappa6(um2, um1, eps, up1, up2, up3, cv_e, d);
      const double p_eps = k_e * d;
      um2 = UP[4 * PW + tp - 2]; um1 = UP[4 * PW + tp - 1]; up1 = UP[4 * PW + tp + 1]; up2 = UP[4 * PW + tp + 2]; up3 = UP[4 * PW + tp + 3];
      kxb = kappa6(um2, um1, by, up1, up2, up3, cv_b, d);
      px[C_B] = kxb * d;
      dcx_by = cd12v(um2, um1, up1, up2);
      px[C_E] = fma(0.5 * (by + up1), px[C_B], fma(vybar, px[C_MY], fma(vxbar, px[C_MX], p_eps)));
    }
#pragma unroll
    for (int f = 0; f < 5; ++f) PK[f * PW + tp] = px[f];
    PK[5 * PW + tp] = kxv;
    PK[6 * PW + tp] = kxb;
    // ------------------------------------------------------------------ tail B: central x-difference of C_x(j)
    double R[NF];
    if (tail_on) {
      double cdx[5];
#pragma unroll
      for (int f = 0; f < 5; ++f)
        cdx[f] = cd12v(CXP[f * PW + tp - 2], CXP[f * PW + tp - 1], CXP[f * PW + tp + 1], CXP[f * PW + tp + 2]);
      R[F_RHO] = cdx[C_RHO]; R[F_MX] = cdx[C_MX]; R[F_MY] = cdx[C_MY]; R[F_E] = cdx[C_E]; R[F_BY] = cdx[C_B];
      R[F_BX] = 0.0;
    }
    __syncthreads();

    // ------------------------------------------------------------------ head: Phi_x difference, G(. ; y), C_y(r)
    {
      const double kvl = PK[5 * PW + tp - 1], kbl = PK[6 * PW + tp - 1];
#pragma unroll
      for (int f = 0; f < 5; ++f) DXR[(slot4 * 5 + f) * NT + tid] = px[f] - PK[f * PW + tp - 1];
      const double kv = 0.5 * (kvl + kxv);
      const double kb = 0.5 * (kbl + kxb);
      const double gm = ((0.5 * rho) * kv) * (dcx_vy * (1.0 / 12.0));      // G(mx ; y)
      const double gb = -(kb * (dcx_by * (1.0 / 12.0)));                   // G(bx ; y)
      CYR[(s6 * 5 + C_RHO) * NT + tid] = cyn[C_RHO];
      CYR[(s6 * 5 + C_MX) * NT + tid] = cyn[C_MX] - gm;
      CYR[(s6 * 5 + C_MY) * NT + tid] = cyn[C_MY];
      CYR[(s6 * 5 + C_E) * NT + tid] = cyn[C_E] - fma(vx, gm, bx * gb);
      CYR[(s6 * 5 + C_B) * NT + tid] = cyn[C_B] - gb;
    }
    // ------------------------------------------------------------------ tail C: assemble R(j), combine, write
    if (tail_on) {
      // rows j-2, j-1, j+1, j+2 = r-5, r-4, r-2, r-1 in the mod-6 ring
      const int jm2 = s6 + 1 >= 6 ? s6 - 5 : s6 + 1, jm1 = s6 + 2 >= 6 ? s6 - 4 : s6 + 2;
      const int jp1 = s6 + 4 >= 6 ? s6 - 2 : s6 + 4, jp2 = s6 + 5 >= 6 ? s6 - 1 : s6 + 5;
      double cdy[5];
#pragma unroll
      for (int f = 0; f < 5; ++f)
        cdy[f] = cd12v(CYR[(jm2 * 5 + f) * NT + tid], CYR[(jm1 * 5 + f) * NT + tid], CYR[(jp1 * 5 + f) * NT + tid],
                       CYR[(jp2 * 5 + f) * NT + tid]);
      R[F_RHO] = fma(R[F_RHO], idx_, cdy[C_RHO] * idy_) * (-1.0 / 12.0);
      R[F_MX] = fma(R[F_MX], idx_, cdy[C_MX] * idy_) * (-1.0 / 12.0);
      R[F_MY] = fma(R[F_MY], idx_, cdy[C_MY] * idy_) * (-1.0 / 12.0);
      R[F_E] = fma(R[F_E], idx_, cdy[C_E] * idy_) * (-1.0 / 12.0);
      R[F_BX] = (cdy[C_B] * idy_) * (-1.0 / 12.0);
      R[F_BY] = fma(R[F_BY], idx_, 0.0) * (-1.0 / 12.0);
      const int js4 = (j + 4096) & 3;
      R[F_RHO] = fma(DXR[(js4 * 5 + C_RHO) * NT + tid], idx_, R[F_RHO]);
      R[F_MX] = fma(DXR[(js4 * 5 + C_MX) * NT + tid], idx_, R[F_MX]);
      R[F_MY] = fma(DXR[(js4 * 5 + C_MY) * NT + tid], idx_, R[F_MY]);
      R[F_E] = fma(DXR[(js4 * 5 + C_E) * NT + tid], idx_, R[F_E]);
      R[F_BY] = fma(DXR[(js4 * 5 + C_B) * NT + tid], idx_, R[F_BY]);
      R[F_RHO] = fma(py[C_RHO] - py_prev[C_RHO], idy_, R[F_RHO]);
      R[F_MX] = fma(py[C_MX] - py_prev[C_MX], idy_, R[F_MX]);
      R[F_MY] = fma(py[C_MY] - py_prev[C_MY], idy_, R[F_MY]);
      R[F_E] = fma(py[C_E] - py_prev[C_E], idy_, R[F_E]);
      R[F_BX] = fma(py[C_B] - py_prev[C_B], idy_, R[F_BX]);

      double o[NF];
      if (combine == COMBINE_FINAL) {
#pragma unroll
        for (int f = 0; f < NF; ++f) o[f] = fma(cdt, R[f], fma(fma(-2.0, jin[f], jacc[f]), 1.0 / 3.0, jin[f]));
      } else {
#pragma unroll
        for (int f = 0; f < NF; ++f) o[f] = fma(cdt, R[f], jbase[f]);
      }
      if (col_out && j < yend) {
        const long long go = (long long)(j + NG) * g.pitch + (ci + XOFF);
#pragma unroll
        for (int f = 0; f < NF; ++f) a.out.p[f][go] = o[f];
        if (combine == COMBINE_ACC) {
#pragma unroll
          for (int f = 0; f < NF; ++f) a.acc_out.p[f][go] = fma(2.0, o[f], jin[f] - jbase[f]);
        }
        if (ws_mode != WS_NONE) {
          double w4[4];
          cell_wavespeeds(o[F_RHO], o[F_MX], o[F_MY], o[F_E], o[F_BX], o[F_BY], gamma, ws_mode == WS_FULL, w4);
#pragma unroll
          for (int k = 0; k < 4; ++k) wsmax[k] = dmax(wsmax[k], w4[k]);
        }
      }
    }
#pragma unroll
    for (int f = 0; f < 5; ++f) py_prev[f] = py[f];
    kyv_prev = kyv; kyb_prev = kyb;
    s6 = s6 == 5 ? 0 : s6 + 1;
  }
  cp_async_wait<0>();
  if (ws_mode != WS_NONE)
    block_max4_atomic(wsmax, red_sh, a.sc->red[a.red_out], ws_mode == WS_FULL ? 0 : 2);
}

}  // namespace smaug
