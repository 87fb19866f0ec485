// smaug_aux_kernels.cuh -- the small kernels of the step: ghost fill (c-8), standalone wave-speed
// reduction (c-4), device-resident dt (c-7).  sm_100a, fp64.  The non-template kernels are `static`: smaug.cu and
// smaug_static.cu both include this header.
#pragma once
#include "smaug_device.cuh"

namespace smaug {

// ------------------------------------------------------------------------------------------------
// Per-cell wave-speed quantities (c-4), from TOTAL fields:
//   a^2 = gamma p_k / rho, p_k = (gamma-1)(e - rho v^2/2 - B^2/2);   b^2 = B^2/rho
//   c_f,d^2 = ( a^2+b^2 + sqrt(max(0,(a^2+b^2)^2 - 4 a^2 B_d^2/rho)) ) / 2;   out: |v_d| + c_f,d, a^2, b^2
// full = false skips the two fast speeds (only a^2, b^2 are needed for v_t of an intermediate stage).
// Results are clamped to >= 0 with fmax, which also drops NaNs (the oracle skips NaNs the same way).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cell_wavespeeds(double rho, double mx, double my, double e, double Bx,
                                                double By, double gamma, bool full, double out[4]) {
  const double rr = drcp(rho);
  const double vx = mx * rr, vy = my * rr;
  const double B2 = fma(By, By, Bx * Bx);
  const double pk = (gamma - 1.0) * ((e - 0.5 * fma(my, vy, mx * vx)) - 0.5 * B2);
  const double a2 = (gamma * pk) * rr;
  const double b2 = B2 * rr;
  out[2] = fmax(a2, 0.0);
  out[3] = fmax(b2, 0.0);
  if (full) {
    const double s = a2 + b2;
    const double fa = (4.0 * a2) * rr;
    const double cfx2 = 0.5 * (s + sqrt(fmax(0.0, fma(s, s, -(fa * (Bx * Bx))))));
    const double cfy2 = 0.5 * (s + sqrt(fmax(0.0, fma(s, s, -(fa * (By * By))))));
    out[0] = fmax(fabs(vx) + sqrt(cfx2), 0.0);
    out[1] = fmax(fabs(vy) + sqrt(cfy2), 0.0);
  } else {
    out[0] = 0.0;
    out[1] = 0.0;
  }
}

// Block-level max of 4 values per thread, then one atomicMax per value per block (warp shuffles + one
// atomic pass, north_star).  `sh` is 4 * 32 doubles of shared memory.  All threads of the block must call.
__device__ __forceinline__ void block_max4_atomic(double m[4], double* sh, unsigned long long* slots,
                                                  int nvals_from) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int k = 0; k < 4; ++k) m[k] = warp_max(m[k]);
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) sh[k * 32 + wid] = m[k];
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double v = lane < nw ? sh[k * 32 + lane] : 0.0;
      v = warp_max(v);
      if (lane == 0 && k >= nvals_from) atomic_max_nonneg(&slots[k], v);
    }
  }
}

// Standalone reduction over the interior of one state (used by smaug_set_state / smaug_get_wavespeeds).
template <bool BG>
__global__ void __launch_bounds__(256) wavespeed_kernel(Grid g, CPlanes6 w, CPlanes4 bg, double gamma,
                                                        unsigned long long* slots) {
  __shared__ double sh[4 * 32];
  double m[4] = {0.0, 0.0, 0.0, 0.0};
  const long long n = (long long)g.nx * g.ny;
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n;
       q += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(q / g.nx), i = (int)(q - (long long)j * g.nx);
    const long long a = cell_addr(g, i, j);
    double rho = w.p[F_RHO][a], e = w.p[F_E][a], Bx = w.p[F_BX][a], By = w.p[F_BY][a];
    if (BG) {
      rho = bg.p[BG_RHO][a] + rho;
      e = bg.p[BG_E][a] + e;
      Bx = bg.p[BG_BX][a] + Bx;
      By = bg.p[BG_BY][a] + By;
    }
    double o[4];
    cell_wavespeeds(rho, w.p[F_MX][a], w.p[F_MY][a], e, Bx, By, gamma, true, o);
#pragma unroll
    for (int k = 0; k < 4; ++k) m[k] = fmax(m[k], o[k]);
  }
  block_max4_atomic(m, sh, slots, 0);
}

// ------------------------------------------------------------------------------------------------
// Ghost fill (c-8), one launch for all ghost cells of up to 6 planes (blockIdx.y = plane).
// The oracle fills x over interior rows, then y over the padded width; composing the two maps gives,
// for a ghost cell (i, j), the source cell (mapx(i), mapy(j)) with map = wrap (periodic) or clamp (open);
// a FIXED side is never rewritten (its ghosts were frozen at set_state), and a corner next to a fixed
// x side copies that frozen ghost along y.  freeze = 1 (set_state, background): fixed acts like open.
// Reads only interior cells or frozen ghosts, writes only ghosts => no race within the launch.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int wrap_idx(int i, int n) {
  int r = i % n;
  return r < 0 ? r + n : r;
}

// the ghost cells of one plane, shared out over `nthreads` threads of which this is number `t`
__device__ __forceinline__ void ghost_fill_plane(const Grid& g, double* p, int freeze, long long t, long long nthreads) {
  const int wpad = g.nx + 2 * NG;
  const long long n_y = 2LL * NG * wpad;                 // cells in the 6 ghost rows
  const long long total = n_y + 2LL * NG * g.ny;         // + 6 ghost columns of every interior row
  for (long long q = t; q < total; q += nthreads) {
    int i, j;
    if (q < n_y) {
      const int row = (int)(q / wpad);
      i = (int)(q - (long long)row * wpad) - NG;
      j = row < NG ? row - NG : g.ny + (row - NG);
    } else {
      const long long r = q - n_y;
      j = (int)(r / (2 * NG));
      const int s = (int)(r - (long long)j * (2 * NG));
      i = s < NG ? s - NG : g.nx + (s - NG);
    }
    const int kx = i < 0 ? g.bc[0] : (i >= g.nx ? g.bc[1] : -1);   // -1: interior along x
    const int ky = j < 0 ? g.bc[2] : (j >= g.ny ? g.bc[3] : -1);
    int si = i, sj = j;
    if (ky >= 0) {
      if (ky == BC_FIXED && !freeze) continue;
      sj = ky == BC_PERIODIC ? wrap_idx(j, g.ny) : (j < 0 ? 0 : g.ny - 1);
      if (kx >= 0 && !(kx == BC_FIXED && !freeze))
        si = kx == BC_PERIODIC ? wrap_idx(i, g.nx) : (i < 0 ? 0 : g.nx - 1);
    } else {
      if (kx == BC_FIXED && !freeze) continue;
      si = kx == BC_PERIODIC ? wrap_idx(i, g.nx) : (i < 0 ? 0 : g.nx - 1);
    }
    p[cell_addr(g, i, j)] = p[cell_addr(g, si, sj)];
  }
}

static __global__ void __launch_bounds__(256) ghost_fill_kernel(Grid g, Planes6 pl, int freeze) {
  ghost_fill_plane(g, pl.p[blockIdx.y], freeze, (long long)blockIdx.x * blockDim.x + threadIdx.x,
                   (long long)gridDim.x * blockDim.x);
}

// ------------------------------------------------------------------------------------------------
// dt (c-7), one thread:  dt = cfl * min_d(Delta_d / cmax_d), an axis with n = 1 excluded; or fixed_dt.
// Also advances t, raises the sticky status on a non-finite / non-positive dt, and clears the reduction
// sets the coming step will accumulate into (bit mask `clear_sets`).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dt_body(DeviceScalars* s, int state_set, unsigned clear_sets, double cfl, double fixed_dt,
                                        double dx, double dy, int nx, int ny) {
  {
    double dt = fixed_dt;
    if (!(fixed_dt > 0.0)) {
      const double cx = __longlong_as_double((long long)s->red[state_set][0]);
      const double cy = __longlong_as_double((long long)s->red[state_set][1]);
      double m = __longlong_as_double(0x7ff0000000000000LL);   // +inf
      if (nx > 1) m = fmin(m, dx / cx);
      if (ny > 1) m = fmin(m, dy / cy);
      dt = cfl * m;
    }
    if (!(dt > 0.0) || isinf(dt) || isnan(dt)) s->status = 1;
    s->dt = dt;
    s->t += dt;
    for (int k = 0; k < NRED; ++k)
      if (clear_sets & (1u << k)) {
        s->red[k][0] = 0ULL; s->red[k][1] = 0ULL; s->red[k][2] = 0ULL; s->red[k][3] = 0ULL;
      }
  }
}

static __global__ void dt_kernel(DeviceScalars* s, int state_set, unsigned clear_sets, double cfl, double fixed_dt,
                          double dx, double dy, int nx, int ny) {
  if (threadIdx.x == 0 && blockIdx.x == 0) dt_body(s, state_set, clear_sets, cfl, fixed_dt, dx, dy, nx, ny);
}

static __global__ void clear_red_kernel(DeviceScalars* s, unsigned clear_sets) {
  if (threadIdx.x == 0 && blockIdx.x == 0)
    for (int k = 0; k < NRED; ++k)
      if (clear_sets & (1u << k)) {
        s->red[k][0] = 0ULL; s->red[k][1] = 0ULL; s->red[k][2] = 0ULL; s->red[k][3] = 0ULL;
      }
}

}  // namespace smaug
