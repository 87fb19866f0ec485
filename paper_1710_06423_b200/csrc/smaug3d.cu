// smaug3d.cu -- the three-dimensional form of the SMAUG+ hot path on B200 (C ABI in
// include/smaug3d.h).  fp64, sm_100a, -fmad=false: the arithmetic contract of DESIGN.md section 4 holds (every
// formula is the explicit IEEE operation sequence the 3-D oracle documents; results are bit-identical to it).
// Product code: shares nothing with oracle/.
//
// First 3-D form: an RK stage is three kernels over padded volumes in HBM,
//   ghost3_kernel     ghost cells of the stage input and of its derived quantities, six sides, edges and corners by composing
//                     the three maps (c-8); only the ghost shell gets threads
//   kappa3_kernel     per interface along each axis d: the seven hyperviscosity ratios (c-5) and the interface fluxes
//                     Phi_d of all fields; keeps kappa_d(v_k), kappa_d(b_k), k != d, for the mixed terms
//   stage3_kernel     per 32 x 4 x 4 tile: C_k = F_k - G_k (c-2 fluxes minus the mixed fluxes of c-5 / c-11) through shared
//                     memory, one direction at a time; R = -sum_k d^c_k C_k + gravity + sum_d (Phi_d+ - Phi_d-)/Delta_d; the RK
//                     combine in the epilogue, the store, the derived quantities v, eps of the written state (c-2) and its
//                     wave-speed maxima (warp shuffles, one atomicMax pass per CTA)
// (SMAUG3_PARAM_KERNEL = 0: cflux3_kernel + assemble3_kernel, the same with the C_k volumes in HBM; derive3_kernel: v, eps on
// every padded cell, at set_state).  dt, t and the maxima stay on the device; one host synchronisation per smaug3_step call.
// DESIGN.md section 5 has the byte counts and what taking kappa / Phi out of HBM as well would need.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/smaug3d.h"
#include "smaug_device.cuh"

namespace smaug3 {

using smaug::ddiv;
using smaug::drcp;
using smaug::kappa_ratio;
using smaug::NG;
using smaug::XOFF;

constexpr int NF = 8;
enum { F_RHO = 0, F_MX = 1, F_MY = 2, F_MZ = 3, F_E = 4, F_BX = 5, F_BY = 6, F_BZ = 7 };
enum { BC_PERIODIC = 0, BC_OPEN = 1, BC_FIXED = 2 };
enum { COMBINE_BASE = 0, COMBINE_ACC = 1, COMBINE_FINAL = 2 };
enum { WS_VT = 1, WS_FULL = 2 };
constexpr int NRED = 5;       // reduction sets
constexpr int NDER = 4;       // vx, vy, vz, eps
constexpr int NPHI = 7;       // Phi_d / C_d components: rho, mx, my, mz, e, b_l1, b_l2 (l1 < l2, both != d)
constexpr int NKM = 4;
#ifndef SMAUG3_BX
#define SMAUG3_BX 32      // thread-block shape of the stencil kernels (kappa3, cflux3, assemble3): BX x BY x BZ = 128 threads;
#define SMAUG3_BY 4       // a block that is several cells thick across x finds part of its y- and z-neighbours in L1
#define SMAUG3_BZ 1
#endif
constexpr int BX = SMAUG3_BX, BY = SMAUG3_BY, BZ = SMAUG3_BZ;
static_assert(BX * BY * BZ == 128 && BX % 32 == 0, "stencil kernels run 128 threads, whole warps along x");        // kappa_d(v_k1), kappa_d(v_k2), kappa_d(b_k1), kappa_d(b_k2), k1 < k2, both != d

// Padded volume: (nz + 6) planes of (ny + 6) rows of `pitch` doubles; interior cell (i, j, k) at
// ((k + 3)(ny + 6) + (j + 3)) pitch + i + 16 (interior column 0 is 128-byte aligned).
struct Grid3 {
  int n[3];
  int pitch, rows;          // rows = ny + 6
  long long plane, vol;     // doubles per plane / per volume
  int bc[6];
};
__host__ __device__ inline long long addr3(const Grid3& g, int i, int j, int k) {
  return ((long long)(k + NG) * g.rows + (j + NG)) * g.pitch + (i + XOFF);
}
__host__ __device__ inline long long stride3(const Grid3& g, int d) { return d == 0 ? 1 : (d == 1 ? g.pitch : g.plane); }

struct V8 { double* p[NF]; };
struct CV8 { const double* p[NF]; };
struct V7 { double* p[NPHI]; };
struct CV7 { const double* p[NPHI]; };
struct V4 { double* p[4]; };
struct V12 { double* p[NF + 4]; };     // the state and its derived quantities (ghost fill)
struct CV4 { const double* p[4]; };

struct Scalars3 {
  unsigned long long red[NRED][5];      // {cmax_x, cmax_y, cmax_z, max a^2, max b^2} as fp64 bit patterns (>= 0)
  double dt, t;
  int status, pad;
};

struct Params3 {
  double gamma;
  double inv_d[3];
  double c_rho, c_mom, c_e, c_b;
  double g[3];
  int grav_on;
};

__device__ __forceinline__ double dabs(double x) { return __hiloint2double(__double2hiint(x) & 0x7fffffff, __double2loint(x)); }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double cd12v(double m2, double m1, double p1, double p2) { return fma(8.0, p1 - m1, -(p2 - m2)); }
__device__ __forceinline__ double cd12p(const double* f, long long s) { return fma(8.0, f[s] - f[-s], -(f[2 * s] - f[-2 * s])); }

// kappa at the interface between p[0] and p[s] from the six cells p[-2s .. 3s] (c-5); d_mid = p[s] - p[0]
__device__ __forceinline__ double kappa_at(const double* p, long long s, double cv, double& d_mid, double& lo, double& hi) {
  const double u0 = p[-2 * s], u1 = p[-s], u2 = p[0], u3 = p[s], u4 = p[2 * s], u5 = p[3 * s];
  const double a0 = u1 - u0, a1 = u2 - u1, a2 = u3 - u2, a3 = u4 - u3, a4 = u5 - u4;
  const double t0 = dabs(fma(3.0, a1, -(u3 - u0)));
  const double t1 = dabs(fma(3.0, a2, -(u4 - u1)));
  const double t2 = dabs(fma(3.0, a3, -(u5 - u2)));
  const double m3 = dmax(dmax(t0, t1), t2);
  const double m1 = dmax(dmax(dmax(dabs(a0), dabs(a1)), dmax(dabs(a2), dabs(a3))), dabs(a4));
  d_mid = a2;
  lo = u2;
  hi = u3;
  return kappa_ratio(m3, m1, cv);
}

__device__ __forceinline__ int wrap_idx(int i, int n) {
  int r = i % n;
  return r < 0 ? r + n : r;
}

// ------------------------------------------------------------------------------------------------ ghost fill (c-8)
// The oracle fills x over interior (j, k), then y over the padded x-extent, then z over the padded x- and y-extents.
// Composed: a ghost cell takes the cell reached by mapping z, then y, then x (periodic: wrap, open: clamp); a FIXED
// side is never rewritten -- if the outermost out-of-range axis (z before y before x) is fixed the cell is skipped,
// and a fixed axis met later stops the mapping (the source is then a frozen ghost).  freeze: fixed acts like open
// (set_state).  Reads interior cells or frozen ghosts, writes other ghosts: no race within the launch.  The derived
// quantities (v, eps) ride along: a ghost cell's derived values are those of its source cell, bit for bit.
__device__ __forceinline__ void ghost_cell(const Grid3& g, const V12& w, int freeze, int i, int j, int k) {
  int c[3] = {i, j, k};
  bool first = true;
#pragma unroll
  for (int a = 2; a >= 0; --a) {
    if (c[a] >= 0 && c[a] < g.n[a]) continue;
    const int kind = g.bc[2 * a + (c[a] < 0 ? 0 : 1)];
    if (kind == BC_FIXED && !freeze) {
      if (first) return;
      break;
    }
    c[a] = kind == BC_PERIODIC ? wrap_idx(c[a], g.n[a]) : (c[a] < 0 ? 0 : g.n[a] - 1);
    first = false;
  }
  const long long dst = addr3(g, i, j, k), src = addr3(g, c[0], c[1], c[2]);
#pragma unroll
  for (int f = 0; f < NF + 4; ++f) w.p[f][dst] = w.p[f][src];
}
// ghost index 0..5 -> -3, -2, -1, n, n+1, n+2
__device__ __forceinline__ int ghost_coord(int s, int n) { return s < NG ? s - NG : n + (s - NG); }

// The ghost shell in three launches (only ghost cells get a thread): SLAB 2: the six ghost planes (all i, j);
// SLAB 1: the six ghost rows of every interior plane (all i); SLAB 0: the six ghost columns of every interior row.
template <int SLAB>
__global__ void __launch_bounds__(128) ghost3_kernel(Grid3 g, V12 w, int freeze) {
  int i, j, k;
  if (SLAB == 2) {
    i = (int)(blockIdx.x * blockDim.x + threadIdx.x) - NG;
    j = (int)blockIdx.y - NG;
    k = ghost_coord((int)blockIdx.z, g.n[2]);
    if (i >= g.n[0] + NG) return;
  } else if (SLAB == 1) {
    i = (int)(blockIdx.x * blockDim.x + threadIdx.x) - NG;
    j = ghost_coord((int)blockIdx.y, g.n[1]);
    k = (int)blockIdx.z;
    if (i >= g.n[0] + NG) return;
  } else {
    const int t = (int)(blockIdx.x * blockDim.x + threadIdx.x);      // 6 ghost columns x ny interior rows of plane k
    if (t >= 2 * NG * g.n[1]) return;
    j = t / (2 * NG);
    i = ghost_coord(t - j * 2 * NG, g.n[0]);
    k = (int)blockIdx.y;
  }
  ghost_cell(g, w, freeze, i, j, k);
}

// ------------------------------------------------------------------------------------------------ derived (c-2)
__global__ void __launch_bounds__(128) derive3_kernel(Grid3 g, CV8 w, V4 der) {
  const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x) - NG;
  if (i >= g.n[0] + NG) return;
  const long long q = addr3(g, i, (int)blockIdx.y - NG, (int)blockIdx.z - NG);
  const double rr = drcp(w.p[F_RHO][q]);
  const double mx = w.p[F_MX][q], my = w.p[F_MY][q], mz = w.p[F_MZ][q];
  const double vx = mx * rr, vy = my * rr, vz = mz * rr;
  const double bx = w.p[F_BX][q], by = w.p[F_BY][q], bz = w.p[F_BZ][q];
  const double b2h = 0.5 * fma(bz, bz, fma(by, by, bx * bx));
  const double ke = 0.5 * fma(mz, vz, fma(my, vy, mx * vx));
  der.p[0][q] = vx; der.p[1][q] = vy; der.p[2][q] = vz;
  der.p[3][q] = (w.p[F_E][q] - ke) - b2h;
}

// ------------------------------------------------------------------------------------------------ kappa, Phi (c-5)
// One thread per interface (cell q | cell q + stride(D)); interfaces -1 .. n-1 along D, cells [-2, n+2) across it
// (the mixed terms read kappa there).  Phi = g kappa (q_b - q_a); energy: Phi(eps) + sum_l vbar_l Phi(m_l)
// + sum_{l != D} Bbar_l Phi(b_l), l ascending, v before B (c-11).
struct KappaCv { double rho, mom, e, b; };
template <int D>
__device__ __forceinline__ void kappa_dir(const Grid3& g, const KappaCv& cv, const CV8& w, const CV4& der, long long q,
                                          const V7& phi, const V4& km) {
  constexpr int A1 = D == 0 ? 1 : 0, A2 = D == 2 ? 1 : 2;          // the two axes across D, ascending
  const long long s = stride3(g, D);
  double d, lo, hi;
  const double k_rho = kappa_at(w.p[F_RHO] + q, s, cv.rho, d, lo, hi);
  const double rbar = 0.5 * (lo + hi);
  phi.p[0][q] = k_rho * d;
  const double k_e = kappa_at(der.p[3] + q, s, cv.e, d, lo, hi);
  double e = k_e * d;
  double kv[3];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    kv[l] = kappa_at(der.p[l] + q, s, cv.mom, d, lo, hi);
    const double gl = l == D ? rbar : 0.5 * rbar;
    const double pm = (gl * kv[l]) * d;
    phi.p[1 + l][q] = pm;
    e = fma(0.5 * (lo + hi), pm, e);
  }
  km.p[0][q] = kv[A1];
  km.p[1][q] = kv[A2];
  {
    const double kb = kappa_at(w.p[F_BX + A1] + q, s, cv.b, d, lo, hi);
    const double pb = kb * d;
    phi.p[5][q] = pb;
    km.p[2][q] = kb;
    e = fma(0.5 * (lo + hi), pb, e);
  }
  {
    const double kb = kappa_at(w.p[F_BX + A2] + q, s, cv.b, d, lo, hi);
    const double pb = kb * d;
    phi.p[6][q] = pb;
    km.p[3][q] = kb;
    e = fma(0.5 * (lo + hi), pb, e);
  }
  phi.p[4][q] = e;
}

// One launch for the three axes: a thread owns cell c in [-2, n+2)^3 and evaluates the interface (c | c + e_d) for every
// axis d with -1 <= c_d <= n_d - 1 (the windows of the three axes share their centre cells; the y- and z-windows of
// neighbouring cells are L1 / L2 hits, so the eight input volumes are read from DRAM once instead of three times).
struct KappaOut { V7 phi[3]; V4 km[3]; };
// (12 CTAs per SM = 40 registers: 1.93 -> 1.64 ms per stage at 256^3; 16 CTAs = 32 registers spill: 2.22)
__global__ void __launch_bounds__(128, 12) kappa3_kernel(Grid3 g, Params3 prm, CV8 w, CV4 der, const Scalars3* sc, int red_in,
                                                     KappaOut o) {
  const int c0 = (int)(blockIdx.x * BX + threadIdx.x) - 2;
  const int c1 = (int)(blockIdx.y * BY + threadIdx.y) - 2, c2 = (int)(blockIdx.z * BZ + threadIdx.z) - 2;
  if (c0 >= g.n[0] + 2 || c1 >= g.n[1] + 2 || c2 >= g.n[2] + 2) return;
  const long long q = addr3(g, c0, c1, c2);
  const double vt = sqrt(__longlong_as_double((long long)sc->red[red_in][3])) +
                    sqrt(__longlong_as_double((long long)sc->red[red_in][4]));
  const KappaCv cv = {prm.c_rho * vt, prm.c_mom * vt, prm.c_e * vt, prm.c_b * vt};
  if (c0 >= -1 && c0 <= g.n[0] - 1) kappa_dir<0>(g, cv, w, der, q, o.phi[0], o.km[0]);
  if (c1 >= -1 && c1 <= g.n[1] - 1) kappa_dir<1>(g, cv, w, der, q, o.phi[1], o.km[1]);
  if (c2 >= -1 && c2 <= g.n[2] - 1) kappa_dir<2>(g, cv, w, der, q, o.phi[2], o.km[2]);
}

// ------------------------------------------------------------------------------------------------ C_k = F_k - G_k
// One thread per cell, [-2, n+2) along K, interior across it.  F: c-2.  G (hyperdiffusion on): for each
// l != K ascending, G(m_l; K) = (rho/2) kbar_l(v_K) d^c_l v_K, G(b_l; K) = - kbar_l(b_K) d^c_l b_K,
// G(e; K) = sum_l v_l G(m_l; K) + b_l G(b_l; K) (c-11).  kmA / kmB: the kappa arrays of directions l1 < l2.
struct CellVals { double rho, e, eps, ptt, bv, m[3], b[3], v[3]; };
template <int K, bool HD>
__device__ __forceinline__ void cflux_dir(const Grid3& g, const CellVals& u, const CV8& w, const CV4& der, const CV4& kmA,
                                          const CV4& kmB, long long q, double (&F)[NPHI]) {
  constexpr int L1 = K == 0 ? 1 : 0, L2 = K == 2 ? 1 : 2;
  const double* m = u.m; const double* b = u.b; const double* v = u.v;
  const double h = u.e + u.ptt;
  F[0] = u.rho * v[K];
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const double f = fma(m[l], v[K], -(b[l] * b[K]));
    F[1 + l] = l == K ? f + u.ptt : f;
  }
  F[4] = fma(v[K], h, -(b[K] * u.bv));
  F[5] = fma(v[K], b[L1], -(b[K] * v[L1]));
  F[6] = fma(v[K], b[L2], -(b[K] * v[L2]));
  if (HD) {
    // position of component K among the stored kappa components of direction l: K - (K > l)
    constexpr int P1 = K - (K > L1 ? 1 : 0), P2 = K - (K > L2 ? 1 : 0);
    const long long s1 = stride3(g, L1), s2 = stride3(g, L2);
    const double kbv1 = 0.5 * (kmA.p[P1][q - s1] + kmA.p[P1][q]);
    const double kbb1 = 0.5 * (kmA.p[2 + P1][q - s1] + kmA.p[2 + P1][q]);
    const double dv1 = cd12p(der.p[K] + q, s1) * (1.0 / 12.0);
    const double db1 = cd12p(w.p[F_BX + K] + q, s1) * (1.0 / 12.0);
    const double gm1 = ((0.5 * u.rho) * kbv1) * dv1;
    const double gb1 = -(kbb1 * db1);
    const double kbv2 = 0.5 * (kmB.p[P2][q - s2] + kmB.p[P2][q]);
    const double kbb2 = 0.5 * (kmB.p[2 + P2][q - s2] + kmB.p[2 + P2][q]);
    const double dv2 = cd12p(der.p[K] + q, s2) * (1.0 / 12.0);
    const double db2 = cd12p(w.p[F_BX + K] + q, s2) * (1.0 / 12.0);
    const double gm2 = ((0.5 * u.rho) * kbv2) * dv2;
    const double gb2 = -(kbb2 * db2);
    double ge = fma(v[L1], gm1, b[L1] * gb1);
    ge = fma(b[L2], gb2, fma(v[L2], gm2, ge));
    F[1 + L1] = F[1 + L1] - gm1;
    F[1 + L2] = F[1 + L2] - gm2;
    F[4] = F[4] - ge;
    F[5] = F[5] - gb1;
    F[6] = F[6] - gb2;
  }
}

// the point values of cell q that the three flux directions share (12 loads, p_t, b.v)
__device__ __forceinline__ void load_cell(const Params3& prm, const CV8& w, const CV4& der, long long q, CellVals& u) {
  u.rho = w.p[F_RHO][q];
  u.e = w.p[F_E][q];
#pragma unroll
  for (int l = 0; l < 3; ++l) { u.m[l] = w.p[F_MX + l][q]; u.b[l] = w.p[F_BX + l][q]; u.v[l] = der.p[l][q]; }
  u.eps = der.p[3][q];
  const double b2h = 0.5 * fma(u.b[2], u.b[2], fma(u.b[1], u.b[1], u.b[0] * u.b[0]));
  u.ptt = fma(prm.gamma - 1.0, u.eps, b2h);
  u.bv = fma(u.b[2], u.v[2], fma(u.b[1], u.v[1], u.b[0] * u.v[0]));
}

// One launch for the three flux directions: a thread owns cell c in [-2, n+2)^3; C_k is needed on [-2, n_k + 2) along k and
// on interior cells across it, so an interior cell evaluates all three and a halo cell the one direction it extends.
// The point values (12 loads, p_t, b.v) are shared by the three directions.
struct CfluxIO { CV4 km[3]; V7 cf[3]; };
template <bool HD>
__global__ void __launch_bounds__(128) cflux3_kernel(Grid3 g, Params3 prm, CV8 w, CV4 der, CfluxIO io) {
  const int c0 = (int)(blockIdx.x * BX + threadIdx.x) - 2;
  const int c1 = (int)(blockIdx.y * BY + threadIdx.y) - 2, c2 = (int)(blockIdx.z * BZ + threadIdx.z) - 2;
  if (c0 >= g.n[0] + 2 || c1 >= g.n[1] + 2 || c2 >= g.n[2] + 2) return;
  const bool in0 = c0 >= 0 && c0 < g.n[0], in1 = c1 >= 0 && c1 < g.n[1], in2 = c2 >= 0 && c2 < g.n[2];
  if ((int)in0 + (int)in1 + (int)in2 < 2) return;            // an edge or corner of the extended box: no direction needs it
  const long long q = addr3(g, c0, c1, c2);
  CellVals u;
  load_cell(prm, w, der, q, u);
  double F[NPHI];
  if (in1 && in2) {
    cflux_dir<0, HD>(g, u, w, der, io.km[1], io.km[2], q, F);
#pragma unroll
    for (int f = 0; f < NPHI; ++f) io.cf[0].p[f][q] = F[f];
  }
  if (in0 && in2) {
    cflux_dir<1, HD>(g, u, w, der, io.km[0], io.km[2], q, F);
#pragma unroll
    for (int f = 0; f < NPHI; ++f) io.cf[1].p[f][q] = F[f];
  }
  if (in0 && in1) {
    cflux_dir<2, HD>(g, u, w, der, io.km[0], io.km[1], q, F);
#pragma unroll
    for (int f = 0; f < NPHI; ++f) io.cf[2].p[f][q] = F[f];
  }
}

// ------------------------------------------------------------------------------------------------ assembly
struct AsmArgs {
  Grid3 g;
  Params3 prm;
  CV7 cf[3], phi[3];
  CV4 der;            // derived quantities of the stage input
  V4 der_out;         // ... of the stage output, written by the epilogue (another set of volumes: neighbouring CTAs of the
                      // fused kernel may still be reading `der` when this one writes)
  CV8 in, base, acc_in;
  V8 out, acc_out;
  Scalars3* sc;
  int red_out;
  double c;
};

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double t = __shfl_xor_sync(0xffffffffu, v, o);
    v = t > v ? t : v;
  }
  return v;
}

// slot of field component `l` of b (or the marker -1 for l == d) inside the 7-component C_d / Phi_d arrays
__host__ __device__ constexpr int bslot(int l, int d) { return l == d ? -1 : 5 + l - (l > d ? 1 : 0); }

// Everything after the central flux divergence of one interior cell: gravity (c-10), the interface-flux differences along
// x, y, z (c-5), the RK combine (c-6), the stores, the derived quantities of the written cell (the next stage's input:
// derive3_kernel's operations) and its wave speeds (c-4), which share every sub-expression with them.
template <int COMBINE, int WS, bool HD>
__device__ __forceinline__ void finish_cell(const AsmArgs& a, long long q, double (&R)[NF], double (&wsm)[5]) {
  const long long st[3] = {1, a.g.pitch, a.g.plane};
  if (a.prm.grav_on) {
    const double rt = a.in.p[F_RHO][q];
    const double gv = fma(a.prm.g[2], a.der.p[2][q], fma(a.prm.g[1], a.der.p[1][q], a.prm.g[0] * a.der.p[0][q]));
#pragma unroll
    for (int l = 0; l < 3; ++l) R[F_MX + l] = fma(rt, a.prm.g[l], R[F_MX + l]);
    R[F_E] = fma(rt, gv, R[F_E]);
  }
  if (HD) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const int slot = f < F_BX ? f : bslot(f - F_BX, d);
        const double diff = slot < 0 ? 0.0 : a.phi[d].p[slot][q] - a.phi[d].p[slot][q - st[d]];
        R[f] = fma(diff, a.prm.inv_d[d], R[f]);
      }
    }
  }
  const double cdt = a.c * a.sc->dt;
  double o[NF];
  if (COMBINE == COMBINE_FINAL) {
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const double w3 = a.in.p[f][q];
      o[f] = fma(cdt, R[f], fma(fma(-2.0, w3, a.acc_in.p[f][q]), 1.0 / 3.0, w3));
    }
  } else {
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const double wb = a.base.p[f][q];
      o[f] = fma(cdt, R[f], wb);
      if (COMBINE == COMBINE_ACC) a.acc_out.p[f][q] = fma(2.0, o[f], a.in.p[f][q] - wb);
    }
  }
#pragma unroll
  for (int f = 0; f < NF; ++f) a.out.p[f][q] = o[f];
  const double rr = drcp(o[F_RHO]);
  const double vx = o[F_MX] * rr, vy = o[F_MY] * rr, vz = o[F_MZ] * rr;
  const double B2 = fma(o[F_BZ], o[F_BZ], fma(o[F_BY], o[F_BY], o[F_BX] * o[F_BX]));
  const double eps = (o[F_E] - 0.5 * fma(o[F_MZ], vz, fma(o[F_MY], vy, o[F_MX] * vx))) - 0.5 * B2;
  a.der_out.p[0][q] = vx; a.der_out.p[1][q] = vy; a.der_out.p[2][q] = vz; a.der_out.p[3][q] = eps;
  const double pk = (a.prm.gamma - 1.0) * eps;
  const double a2 = (a.prm.gamma * pk) * rr;
  const double b2 = B2 * rr;
  wsm[3] = a2 > 0.0 ? a2 : 0.0;
  wsm[4] = b2 > 0.0 ? b2 : 0.0;
  if (WS == WS_FULL) {
    const double s = a2 + b2;
    const double fa = (4.0 * a2) * rr;
    const double vv[3] = {vx, vy, vz};
    const double bb[3] = {o[F_BX], o[F_BY], o[F_BZ]};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double disc = fma(s, s, -(fa * (bb[d] * bb[d])));
      const double cf2 = 0.5 * (s + sqrt(disc > 0.0 ? disc : 0.0));
      const double cc = fabs(vv[d]) + sqrt(cf2);
      wsm[d] = cc > 0.0 ? cc : 0.0;
    }
  }
}

// block maximum of the five candidates (warp shuffles), one atomicMax per value and CTA; NaNs never enter (x > 0 ? x : 0).
// sh: 5 * NW doubles of shared memory; every thread of the CTA calls.
template <int WS, int NW>
__device__ __forceinline__ void block_max5_atomic(const double (&wsm)[5], double* sh, int tid, unsigned long long* slots) {
  const int lane = tid & 31, wid = tid >> 5;
  constexpr int FROM = WS == WS_FULL ? 0 : 3;
#pragma unroll
  for (int v = FROM; v < 5; ++v) {
    const double m = warp_max(wsm[v]);
    if (lane == 0) sh[v * NW + wid] = m;
  }
  __syncthreads();
  if (tid < 5 && tid >= FROM) {
    double m = sh[tid * NW];
    for (int w2 = 1; w2 < NW; ++w2) m = sh[tid * NW + w2] > m ? sh[tid * NW + w2] : m;
    atomicMax(&slots[tid], (unsigned long long)__double_as_longlong(m));
  }
}

// multi-pass form: C_d from the volumes cflux3_kernel wrote
template <int COMBINE, int WS, bool HD>
__global__ void __launch_bounds__(128) assemble3_kernel(const AsmArgs a) {
  __shared__ double sh[5 * 4];
  const Grid3& g = a.g;
  const int i = (int)(blockIdx.x * BX + threadIdx.x);
  const int j = (int)(blockIdx.y * BY + threadIdx.y), k = (int)(blockIdx.z * BZ + threadIdx.z);
  const int tid = (int)((threadIdx.z * BY + threadIdx.y) * BX + threadIdx.x);
  double wsm[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (i < g.n[0] && j < g.n[1] && k < g.n[2]) {
    const long long q = addr3(g, i, j, k);
    const long long st[3] = {1, g.pitch, g.plane};
    double R[NF];
    // -(1/12) sum_d cd12(C_d) / Delta_d, nested x outermost: fma(cd_x, 1/dx, fma(cd_y, 1/dy, cd_z (1/dz)))
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      double cd[3];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const int slot = f < F_BX ? f : bslot(f - F_BX, d);
        cd[d] = slot < 0 ? 0.0 : cd12p(a.cf[d].p[slot] + q, st[d]);
      }
      R[f] = fma(cd[0], a.prm.inv_d[0], fma(cd[1], a.prm.inv_d[1], cd[2] * a.prm.inv_d[2])) * (-1.0 / 12.0);
    }
    finish_cell<COMBINE, WS, HD>(a, q, R, wsm);
  }
  block_max5_atomic<WS, 4>(wsm, sh, tid, a.sc->red[a.red_out]);
}

// Fused form of the two kernels above (SMAUG3_PARAM_KERNEL = 1, the default): a CTA owns a tile of TX x TY x TZ cells and,
// one direction at a time (z, y, x: the nesting order of the sum), evaluates C_d = F_d - G_d on the tile extended by two
// cells along d into shared memory, takes the central difference from there and folds it into R -- the 21 C_d volumes
// never exist in HBM.  The halo cells repeat (TX+4)/TX, (TY+4)/TY, (TZ+4)/TZ of the flux evaluations (1.7x for
// 32 x 4 x 4), which are cheap; their loads are L1 / L2 hits.
#ifndef SMAUG3_TY
#define SMAUG3_TY 4
#define SMAUG3_TZ 4
#endif
#ifndef SMAUG3_ZFAST
#define SMAUG3_ZFAST 0      // 1: blockIdx.x runs over the z-tiles (then y, then x), so that CTAs resident at the same time are
#endif                      //    neighbours along z and y (measured: 3.21 vs 3.11 ms per stage at 256^3 -- no gain; off)
constexpr int TX = 32, TY = SMAUG3_TY, TZ = SMAUG3_TZ, TT = TX * TY * TZ;
constexpr int cmax3(int a, int b, int c) { return a > b ? (a > c ? a : c) : (b > c ? b : c); }
constexpr int TEXT = cmax3((TX + 4) * TY * TZ, TX * (TY + 4) * TZ, TX * TY * (TZ + 4));      // cells of the largest extended tile
constexpr size_t STAGE3_SMEM = (size_t)(NPHI * TEXT + 5 * (TT / 32)) * sizeof(double);

template <int D, bool HD>
__device__ __forceinline__ void tile_cflux(const AsmArgs& a, const CV4 (&km)[3], int x0, int y0, int z0, int tid, double* sC) {
  constexpr int L1 = D == 0 ? 1 : 0, L2 = D == 2 ? 1 : 2;
  constexpr int NE = D == 0 ? (TX + 4) * TY * TZ : (D == 1 ? TX * (TY + 4) * TZ : TX * TY * (TZ + 4));
  const Grid3& g = a.g;
  for (int e = tid; e < NE; e += TT) {
    int i, j, k;
    if (D == 0) { i = e % (TX + 4) - 2; j = (e / (TX + 4)) % TY; k = e / ((TX + 4) * TY); }
    else if (D == 1) { i = e % TX; j = (e / TX) % (TY + 4) - 2; k = e / (TX * (TY + 4)); }
    else { i = e % TX; j = (e / TX) % TY; k = e / (TX * TY) - 2; }
    const int c[3] = {x0 + i, y0 + j, z0 + k};
    bool ok = true;
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) ok = ok && (ax == D ? (c[ax] >= -2 && c[ax] < g.n[ax] + 2) : (c[ax] >= 0 && c[ax] < g.n[ax]));
    if (!ok) continue;
    const long long q = addr3(g, c[0], c[1], c[2]);
    CellVals u;
    load_cell(a.prm, a.in, a.der, q, u);
    double F[NPHI];
    cflux_dir<D, HD>(g, u, a.in, a.der, km[L1], km[L2], q, F);
#pragma unroll
    for (int f = 0; f < NPHI; ++f) sC[f * TEXT + e] = F[f];
  }
}

struct KmIn { CV4 km[3]; };

template <int COMBINE, int WS, bool HD>
__global__ void __launch_bounds__(TT, 1024 / TT) stage3_kernel(const AsmArgs a, const KmIn kin) {
  extern __shared__ __align__(16) double sm3[];
  double* const sC = sm3;
  double* const sh = sm3 + NPHI * TEXT;
  const Grid3& g = a.g;
  const int tx = threadIdx.x, ty = threadIdx.y, tz = threadIdx.z;
  const int tid = (tz * TY + ty) * TX + tx;
  const int x0 = (SMAUG3_ZFAST ? blockIdx.z : blockIdx.x) * TX, y0 = blockIdx.y * TY, z0 = (SMAUG3_ZFAST ? blockIdx.x : blockIdx.z) * TZ;
  const int i = x0 + tx, j = y0 + ty, k = z0 + tz;
  const bool cell = i < g.n[0] && j < g.n[1] && k < g.n[2];
  double R[NF];
  // z: T = cd_z (1/dz)
  tile_cflux<2, HD>(a, kin.km, x0, y0, z0, tid, sC);
  __syncthreads();
  {
    const double* p = sC + ((tz + 2) * TY + ty) * TX + tx;
    constexpr int S = TX * TY;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const int slot = f < F_BX ? f : bslot(f - F_BX, 2);
      const double cd = slot < 0 ? 0.0 : cd12v(p[slot * TEXT - 2 * S], p[slot * TEXT - S], p[slot * TEXT + S], p[slot * TEXT + 2 * S]);
      R[f] = cd * a.prm.inv_d[2];
    }
  }
  __syncthreads();
  // y: T = fma(cd_y, 1/dy, T)
  tile_cflux<1, HD>(a, kin.km, x0, y0, z0, tid, sC);
  __syncthreads();
  {
    const double* p = sC + (tz * (TY + 4) + ty + 2) * TX + tx;
    constexpr int S = TX;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const int slot = f < F_BX ? f : bslot(f - F_BX, 1);
      const double cd = slot < 0 ? 0.0 : cd12v(p[slot * TEXT - 2 * S], p[slot * TEXT - S], p[slot * TEXT + S], p[slot * TEXT + 2 * S]);
      R[f] = fma(cd, a.prm.inv_d[1], R[f]);
    }
  }
  __syncthreads();
  // x: R = fma(cd_x, 1/dx, T) (-1/12)
  tile_cflux<0, HD>(a, kin.km, x0, y0, z0, tid, sC);
  __syncthreads();
  double wsm[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (cell) {
    const double* p = sC + (tz * TY + ty) * (TX + 4) + tx + 2;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const int slot = f < F_BX ? f : bslot(f - F_BX, 0);
      const double cd = slot < 0 ? 0.0 : cd12v(p[slot * TEXT - 2], p[slot * TEXT - 1], p[slot * TEXT + 1], p[slot * TEXT + 2]);
      R[f] = fma(cd, a.prm.inv_d[0], R[f]) * (-1.0 / 12.0);
    }
    finish_cell<COMBINE, WS, HD>(a, addr3(g, i, j, k), R, wsm);
  }
  block_max5_atomic<WS, TT / 32>(wsm, sh, tid, a.sc->red[a.red_out]);
}

// standalone reduction of all five maxima over the interior (set_state)
__global__ void __launch_bounds__(128) wavespeed3_kernel(Grid3 g, CV8 w, double gamma, Scalars3* sc, int set) {
  __shared__ double sh[5 * 4];
  const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x);
  double wsm[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (i < g.n[0]) {
    const long long q = addr3(g, i, (int)blockIdx.y, (int)blockIdx.z);
    const double rr = drcp(w.p[F_RHO][q]);
    const double mx = w.p[F_MX][q], my = w.p[F_MY][q], mz = w.p[F_MZ][q];
    const double vv[3] = {mx * rr, my * rr, mz * rr};
    const double bb[3] = {w.p[F_BX][q], w.p[F_BY][q], w.p[F_BZ][q]};
    const double B2 = fma(bb[2], bb[2], fma(bb[1], bb[1], bb[0] * bb[0]));
    const double pk = (gamma - 1.0) * ((w.p[F_E][q] - 0.5 * fma(mz, vv[2], fma(my, vv[1], mx * vv[0]))) - 0.5 * B2);
    const double a2 = (gamma * pk) * rr;
    const double b2 = B2 * rr;
    wsm[3] = a2 > 0.0 ? a2 : 0.0;
    wsm[4] = b2 > 0.0 ? b2 : 0.0;
    const double s = a2 + b2;
    const double fa = (4.0 * a2) * rr;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double disc = fma(s, s, -(fa * (bb[d] * bb[d])));
      const double cf2 = 0.5 * (s + sqrt(disc > 0.0 ? disc : 0.0));
      const double cc = fabs(vv[d]) + sqrt(cf2);
      wsm[d] = cc > 0.0 ? cc : 0.0;
    }
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const double m = warp_max(wsm[k]);
    if (lane == 0) sh[k * 4 + wid] = m;
  }
  __syncthreads();
  if (threadIdx.x < 5) {
    const int k = threadIdx.x;
    double m = sh[k * 4];
    for (int w2 = 1; w2 < 4; ++w2) m = sh[k * 4 + w2] > m ? sh[k * 4 + w2] : m;
    atomicMax(&sc->red[set][k], (unsigned long long)__double_as_longlong(m));
  }
}

// dt = cfl min_d (Delta_d / cmax_d) over the axes with n > 1 (c-7), t += dt, status, and the reduction sets of the coming
// step cleared; one thread
__global__ void dt3_kernel(Scalars3* s, int state_set, unsigned clear_sets, double cfl, double fixed_dt, double dx, double dy,
                           double dz, int nx, int ny, int nz) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double dt = fixed_dt;
  if (!(fixed_dt > 0.0)) {
    double m = __longlong_as_double(0x7ff0000000000000LL);
    if (nx > 1) m = fmin(m, dx / __longlong_as_double((long long)s->red[state_set][0]));
    if (ny > 1) m = fmin(m, dy / __longlong_as_double((long long)s->red[state_set][1]));
    if (nz > 1) m = fmin(m, dz / __longlong_as_double((long long)s->red[state_set][2]));
    dt = cfl * m;
  }
  if (!(dt > 0.0) || isinf(dt) || isnan(dt)) s->status = 1;
  s->dt = dt;
  s->t += dt;
  for (int k = 0; k < NRED; ++k)
    if (clear_sets & (1u << k))
      for (int v = 0; v < 5; ++v) s->red[k][v] = 0ULL;
}

// flat [8][nz][ny][nx] <-> padded interior
__global__ void __launch_bounds__(128) pack3_kernel(Grid3 g, const double* flat, V8 w, int to_flat, double* flat_out) {
  const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x);
  if (i >= g.n[0]) return;
  const int j = blockIdx.y, k = blockIdx.z;
  const long long q = addr3(g, i, j, k);
  const long long nvol = (long long)g.n[0] * g.n[1] * g.n[2];
  const long long o = ((long long)k * g.n[1] + j) * g.n[0] + i;
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    if (to_flat) flat_out[f * nvol + o] = w.p[f][q];
    else w.p[f][q] = flat[f * nvol + o];
  }
}

// ================================================================================================ host side
thread_local std::string g_err;
int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}
#define CUDA_TRY(x)                                                                                  \
  do {                                                                                               \
    cudaError_t e_ = (x);                                                                            \
    if (e_ != cudaSuccess) return fail(SMAUG3_ECUDA, std::string(#x) + ": " + cudaGetErrorString(e_)); \
  } while (0)

struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != dev) cudaSetDevice(dev);
    else prev = -1;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

struct Ctx {
  Grid3 g;
  int device = 0;
  cudaStream_t stream = nullptr;
  double gamma = 0;
  double L[3] = {1.0, 1.0, 1.0};
  int hd_on = 1, rk_order = 4;
  double c_rho = 0.02, c_mom = 0.4, c_e = 0.02, c_b = 0.02, fixed_dt = 0.0;
  double grav[3] = {0.0, 0.0, 0.0};
  double* mem = nullptr;        // one allocation: all volumes
  V8 buf[4];                    // w^n / state, w1 -> w3, w2, accumulator
  V4 der[2];                    // derived quantities: of the current stage input (dcur) and of its output
  int dcur = 0;
  int fused = 1;                // SMAUG3_PARAM_KERNEL: 1 fused cflux + assembly (stage3_kernel), 0 multi-pass
  V7 phi[3], cf[3];
  V4 km[3];
  Scalars3* sc = nullptr;
  int cur = 0;                  // reduction set holding the maxima of the state (0 or 4)
  long long launches = 0;
  bool timing = false;
  bool timing_broken = false;   // an event could not be created / recorded: timing was switched off, the totals are void
  std::vector<cudaEvent_t> ev;
  std::vector<int> ev_kind;
  size_t ev_used = 0;
  double ms[5] = {0, 0, 0, 0, 0};
  long long nk[5] = {0, 0, 0, 0, 0};
};

constexpr int NVOL = 4 * NF + 2 * NDER + 3 * (NPHI + NPHI + NKM);      // 32 + 8 + 54 = 94 padded volumes

int make_grid(int nx, int ny, int nz, const int bc[6], Grid3& g) {
  g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
  g.pitch = (XOFF + nx + NG + 15) / 16 * 16;
  g.rows = ny + 2 * NG;
  g.plane = (long long)g.pitch * g.rows;
  g.vol = g.plane * (nz + 2 * NG);
  for (int s = 0; s < 6; ++s) g.bc[s] = bc ? bc[s] : 0;
  return 0;
}

template <class T>
CV8 cv8(const T& v) { CV8 c; for (int f = 0; f < NF; ++f) c.p[f] = v.p[f]; return c; }
CV7 cv7(const V7& v) { CV7 c; for (int f = 0; f < NPHI; ++f) c.p[f] = v.p[f]; return c; }
CV4 cv4(const V4& v) { CV4 c; for (int f = 0; f < 4; ++f) c.p[f] = v.p[f]; return c; }

Params3 params(const Ctx& c) {
  Params3 p;
  p.gamma = c.gamma;
  for (int d = 0; d < 3; ++d) { p.inv_d[d] = c.g.n[d] / c.L[d]; p.g[d] = c.grav[d]; }
  p.c_rho = c.c_rho; p.c_mom = c.c_mom; p.c_e = c.c_e; p.c_b = c.c_b;
  p.grav_on = c.grav[0] != 0.0 || c.grav[1] != 0.0 || c.grav[2] != 0.0;
  return p;
}

// event bracket around one launch when timing is on
struct Timed {
  Ctx& c;
  int kind;
  Timed(Ctx& c_, int kind_) : c(c_), kind(kind_) {
    ++c.launches;
    if (c.timing) mark();
  }
  ~Timed() {
    if (c.timing) mark();
  }
  // Never throws and never fails the step: if the event pool cannot grow or an event cannot be recorded, timing is
  // abandoned (smaug3_get_kernel_timing then reports it) and the launches go on untimed.
  void give_up() {
    cudaGetLastError();
    c.timing = false;
    c.timing_broken = true;
  }
  void mark() {
    if (c.ev_used == c.ev.size()) {
      cudaEvent_t e = nullptr;
      if (cudaEventCreate(&e) != cudaSuccess) return give_up();
      try {
        c.ev_kind.push_back(kind);
        c.ev.push_back(e);
      } catch (...) {
        cudaEventDestroy(e);
        return give_up();
      }
    }
    c.ev_kind[c.ev_used] = kind;
    if (cudaEventRecord(c.ev[c.ev_used], c.stream) != cudaSuccess) return give_up();
    ++c.ev_used;
  }
};

dim3 grid_for(int nxr, int nyr, int nzr) { return dim3((unsigned)((nxr + 127) / 128), (unsigned)nyr, (unsigned)nzr); }
// grid / block of the stencil kernels (BX x BY x BZ threads)
dim3 sgrid_for(int nxr, int nyr, int nzr) { return dim3((unsigned)((nxr + BX - 1) / BX), (unsigned)((nyr + BY - 1) / BY), (unsigned)((nzr + BZ - 1) / BZ)); }
const dim3 SBLOCK(BX, BY, BZ);

void launch_ghost(Ctx& c, const V8& w8, int freeze) {
  Timed t(c, 0);
  const Grid3& g = c.g;
  V12 w;
  for (int f = 0; f < NF; ++f) w.p[f] = w8.p[f];
  for (int f = 0; f < 4; ++f) w.p[NF + f] = c.der[c.dcur].p[f];
  ghost3_kernel<2><<<grid_for(g.n[0] + 6, g.n[1] + 6, 6), 128, 0, c.stream>>>(g, w, freeze);
  ghost3_kernel<1><<<grid_for(g.n[0] + 6, 6, g.n[2]), 128, 0, c.stream>>>(g, w, freeze);
  ghost3_kernel<0><<<dim3((unsigned)((6 * g.n[1] + 127) / 128), (unsigned)g.n[2], 1), 128, 0, c.stream>>>(g, w, freeze);
  c.launches += 2;
}

void launch_kappa(Ctx& c, const Params3& p, const V8& in, int red_in) {
  Timed t(c, 2);
  const Grid3& g = c.g;
  KappaOut o;
  for (int d = 0; d < 3; ++d) { o.phi[d] = c.phi[d]; o.km[d] = c.km[d]; }
  kappa3_kernel<<<sgrid_for(g.n[0] + 4, g.n[1] + 4, g.n[2] + 4), SBLOCK, 0, c.stream>>>(g, p, cv8(in), cv4(c.der[c.dcur]), c.sc, red_in, o);
}

void launch_cflux(Ctx& c, const Params3& p, const V8& in) {
  Timed t(c, 3);
  const Grid3& g = c.g;
  CfluxIO io;
  for (int d = 0; d < 3; ++d) { io.km[d] = cv4(c.km[d]); io.cf[d] = c.cf[d]; }
  const dim3 gr = sgrid_for(g.n[0] + 4, g.n[1] + 4, g.n[2] + 4);
  if (c.hd_on) cflux3_kernel<true><<<gr, SBLOCK, 0, c.stream>>>(g, p, cv8(in), cv4(c.der[c.dcur]), io);
  else cflux3_kernel<false><<<gr, SBLOCK, 0, c.stream>>>(g, p, cv8(in), cv4(c.der[c.dcur]), io);
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute of a kernel: raised once per (instantiation,
// device).  A failure leaves the bit clear; the launch that follows then fails and the step reports it.
template <typename K>
void raise_smem_once(K kern, int device, unsigned long long& mask) {
  if (device >= 0 && device < 64 && (mask >> device & 1ULL)) return;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)STAGE3_SMEM) == cudaSuccess) {
    if (device >= 0 && device < 64) mask |= 1ULL << device;
  } else {
    cudaGetLastError();
  }
}

template <int COMBINE, int WS>
void launch_assemble(Ctx& c, const AsmArgs& a) {
  Timed t(c, 4);
  const Grid3& g = c.g;
  if (c.fused) {
    KmIn kin;
    for (int d = 0; d < 3; ++d) kin.km[d] = cv4(c.km[d]);
    const unsigned gx = (unsigned)((g.n[0] + TX - 1) / TX), gz = (unsigned)((g.n[2] + TZ - 1) / TZ);
    const dim3 gr(SMAUG3_ZFAST ? gz : gx, (unsigned)((g.n[1] + TY - 1) / TY), SMAUG3_ZFAST ? gx : gz);
    const dim3 bl(TX, TY, TZ);
    static unsigned long long raised_hd = 0, raised_plain = 0;      // per instantiation: devices already configured
    if (c.hd_on) {
      raise_smem_once(stage3_kernel<COMBINE, WS, true>, c.device, raised_hd);
      stage3_kernel<COMBINE, WS, true><<<gr, bl, STAGE3_SMEM, c.stream>>>(a, kin);
    } else {
      raise_smem_once(stage3_kernel<COMBINE, WS, false>, c.device, raised_plain);
      stage3_kernel<COMBINE, WS, false><<<gr, bl, STAGE3_SMEM, c.stream>>>(a, kin);
    }
    return;
  }
  const dim3 gr = sgrid_for(g.n[0], g.n[1], g.n[2]);
  if (c.hd_on) assemble3_kernel<COMBINE, WS, true><<<gr, SBLOCK, 0, c.stream>>>(a);
  else assemble3_kernel<COMBINE, WS, false><<<gr, SBLOCK, 0, c.stream>>>(a);
}

// one RK stage: out = combine(in, R(in)); the maxima of `in` are in set red_in, those of `out` go to red_out
void stage(Ctx& c, int in, int base, int out, int combine, int ws, double coef, int red_in, int red_out) {
  const Params3 p = params(c);
  launch_ghost(c, c.buf[in], 0);        // (the derived quantities of `in` were written by the stage that produced it)
  if (c.hd_on) launch_kappa(c, p, c.buf[in], red_in);
  if (!c.fused) launch_cflux(c, p, c.buf[in]);
  AsmArgs a;
  a.g = c.g;
  a.prm = p;
  for (int d = 0; d < 3; ++d) { a.cf[d] = cv7(c.cf[d]); a.phi[d] = cv7(c.phi[d]); }
  a.der = cv4(c.der[c.dcur]);
  a.der_out = c.der[c.dcur ^ 1];
  a.in = cv8(c.buf[in]);
  a.base = cv8(c.buf[base]);
  a.acc_in = cv8(c.buf[3]);
  a.out = c.buf[out];
  a.acc_out = c.buf[3];
  a.sc = c.sc;
  a.red_out = red_out;
  a.c = coef;
  if (combine == COMBINE_BASE && ws == WS_VT) launch_assemble<COMBINE_BASE, WS_VT>(c, a);
  else if (combine == COMBINE_BASE) launch_assemble<COMBINE_BASE, WS_FULL>(c, a);
  else if (combine == COMBINE_ACC) launch_assemble<COMBINE_ACC, WS_VT>(c, a);
  else launch_assemble<COMBINE_FINAL, WS_FULL>(c, a);
  c.dcur ^= 1;        // the derived quantities of `out` are now the current ones
}

void enqueue_step(Ctx& c, double cfl) {
  const int cur = c.cur, nxt = cur == 0 ? 4 : 0;
  {
    Timed t(c, 0);
    dt3_kernel<<<1, 32, 0, c.stream>>>(c.sc, cur, (1u << 1) | (1u << 2) | (1u << 3) | (1u << nxt), cfl, c.fixed_dt,
                                       c.L[0] / c.g.n[0], c.L[1] / c.g.n[1], c.L[2] / c.g.n[2], c.g.n[0], c.g.n[1], c.g.n[2]);
  }
  if (c.rk_order == 1) {
    // Euler: w^{n+1} = w^n + dt R(w^n) written into buffer 1, then the buffers swap roles
    stage(c, 0, 0, 1, COMBINE_BASE, WS_FULL, 1.0, cur, nxt);
    std::swap(c.buf[0], c.buf[1]);
  } else if (c.rk_order == 2) {
    stage(c, 0, 0, 1, COMBINE_BASE, WS_VT, 0.5, cur, 1);
    stage(c, 1, 0, 2, COMBINE_BASE, WS_FULL, 1.0, 1, nxt);
    std::swap(c.buf[0], c.buf[2]);
  } else {
    stage(c, 0, 0, 1, COMBINE_BASE, WS_VT, 0.5, cur, 1);
    stage(c, 1, 0, 2, COMBINE_ACC, WS_VT, 0.5, 1, 2);
    stage(c, 2, 0, 1, COMBINE_BASE, WS_VT, 1.0, 2, 3);
    stage(c, 1, 0, 0, COMBINE_FINAL, WS_FULL, 1.0 / 6.0, 3, nxt);
  }
  c.cur = nxt;
}

}  // namespace smaug3

using namespace smaug3;
#define CTX(p) (reinterpret_cast<smaug3::Ctx*>(p))

extern "C" {

const char* smaug3_last_error(void) { return g_err.c_str(); }

size_t smaug3_workspace_bytes(int nx, int ny, int nz) {
  if (nx < 1 || ny < 1 || nz < 1) return 0;
  Grid3 g;
  make_grid(nx, ny, nz, nullptr, g);
  return (size_t)g.vol * NVOL * sizeof(double) + 4096;
}

int smaug3_create(int nx, int ny, int nz, double gamma, const int bc[6], void* stream, smaug3_ctx** out) {
  if (!out || !bc) return fail(SMAUG3_EINVAL, "NULL argument");
  *out = nullptr;
  if (nx < 1 || ny < 1 || nz < 1) return fail(SMAUG3_EINVAL, "nx, ny, nz must be >= 1");
  if (!(gamma > 1.0)) return fail(SMAUG3_EINVAL, "gamma must be > 1");
  for (int s = 0; s < 6; ++s)
    if (bc[s] < 0 || bc[s] > 2) return fail(SMAUG3_EINVAL, "unknown boundary kind");
  for (int a = 0; a < 3; ++a)
    if ((bc[2 * a] == BC_PERIODIC) != (bc[2 * a + 1] == BC_PERIODIC))
      return fail(SMAUG3_EINVAL, "periodic must be set on both sides of an axis");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(SMAUG3_ECUDA, "no CUDA device: libsmaug has no CPU fallback");
  }
  Ctx* c = new (std::nothrow) Ctx();
  if (!c) return fail(SMAUG3_ENOMEM, "host allocation failed");
  make_grid(nx, ny, nz, bc, c->g);
  if (c->g.vol >= (1LL << 31)) { delete c; return fail(SMAUG3_EINVAL, "a padded volume must have fewer than 2^31 elements"); }
  if (nz + 6 > 65535 || ny + 6 > 65535) { delete c; return fail(SMAUG3_EINVAL, "ny, nz must be below 65529"); }
  c->gamma = gamma;
  c->stream = (cudaStream_t)stream;
  if (cudaGetDevice(&c->device) != cudaSuccess) { delete c; return fail(SMAUG3_ECUDA, "cudaGetDevice failed"); }
  const size_t bytes = (size_t)c->g.vol * NVOL * sizeof(double) + 4096;
  if (cudaMalloc(&c->mem, bytes) != cudaSuccess) {
    cudaGetLastError();
    delete c;
    return fail(SMAUG3_ENOMEM, "device allocation of " + std::to_string(bytes) + " bytes failed");
  }
  if (cudaMemsetAsync(c->mem, 0, bytes, c->stream) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(c->mem);
    delete c;
    return fail(SMAUG3_ECUDA, "clearing the device memory failed");
  }
  double* p = c->mem;
  auto take = [&]() { double* r = p; p += c->g.vol; return r; };
  for (int b = 0; b < 4; ++b)
    for (int f = 0; f < NF; ++f) c->buf[b].p[f] = take();
  for (int b = 0; b < 2; ++b)
    for (int f = 0; f < NDER; ++f) c->der[b].p[f] = take();
  for (int d = 0; d < 3; ++d) {
    for (int f = 0; f < NPHI; ++f) c->phi[d].p[f] = take();
    for (int f = 0; f < NPHI; ++f) c->cf[d].p[f] = take();
    for (int f = 0; f < NKM; ++f) c->km[d].p[f] = take();
  }
  c->sc = reinterpret_cast<Scalars3*>(p);
  *out = reinterpret_cast<smaug3_ctx*>(c);
  return SMAUG3_OK;
}

void smaug3_destroy(smaug3_ctx* ctx) {
  if (!ctx) return;
  Ctx* c = CTX(ctx);
  DeviceGuard guard_(c->device);
  cudaStreamSynchronize(c->stream);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  cudaFree(c->mem);
  delete c;
}

int smaug3_set_param(smaug3_ctx* ctx, int key, double v) {
  if (!ctx) return fail(SMAUG3_EINVAL, "NULL ctx");
  Ctx& c = *CTX(ctx);
  switch (key) {
    case SMAUG3_PARAM_LX: if (!(v > 0)) break; c.L[0] = v; return SMAUG3_OK;
    case SMAUG3_PARAM_LY: if (!(v > 0)) break; c.L[1] = v; return SMAUG3_OK;
    case SMAUG3_PARAM_LZ: if (!(v > 0)) break; c.L[2] = v; return SMAUG3_OK;
    case SMAUG3_PARAM_HD_ON: c.hd_on = v != 0.0; return SMAUG3_OK;
    case SMAUG3_PARAM_C_RHO: if (!(v >= 0)) break; c.c_rho = v; return SMAUG3_OK;
    case SMAUG3_PARAM_C_MOM: if (!(v >= 0)) break; c.c_mom = v; return SMAUG3_OK;
    case SMAUG3_PARAM_C_E: if (!(v >= 0)) break; c.c_e = v; return SMAUG3_OK;
    case SMAUG3_PARAM_C_B: if (!(v >= 0)) break; c.c_b = v; return SMAUG3_OK;
    case SMAUG3_PARAM_RK_ORDER: if (v != 1 && v != 2 && v != 4) break; c.rk_order = (int)v; return SMAUG3_OK;
    case SMAUG3_PARAM_FIXED_DT: if (!(v >= 0)) break; c.fixed_dt = v; return SMAUG3_OK;
    case SMAUG3_PARAM_GX: if (!std::isfinite(v)) break; c.grav[0] = v; return SMAUG3_OK;
    case SMAUG3_PARAM_GY: if (!std::isfinite(v)) break; c.grav[1] = v; return SMAUG3_OK;
    case SMAUG3_PARAM_GZ: if (!std::isfinite(v)) break; c.grav[2] = v; return SMAUG3_OK;
    case SMAUG3_PARAM_KERNEL: if (v != 0 && v != 1) break; c.fused = (int)v; return SMAUG3_OK;
    default: return fail(SMAUG3_EINVAL, "unknown parameter key");
  }
  return fail(SMAUG3_EINVAL, "parameter value out of range");
}

int smaug3_set_state(smaug3_ctx* ctx, const void* w) {
  if (!ctx || !w) return fail(SMAUG3_EINVAL, "NULL argument");
  Ctx& c = *CTX(ctx);
  DeviceGuard guard_(c.device);
  const Grid3& g = c.g;
  const size_t nflat = (size_t)NF * g.n[0] * g.n[1] * g.n[2];
  double* staging = c.cf[0].p[0];        // the C_d volumes (21 of them, contiguous with Phi / kappa) are free between steps
  // the staging area must hold 8 flat volumes: cf[0] .. are contiguous allocations of padded volumes >= flat ones
  CUDA_TRY(cudaMemcpyAsync(staging, w, nflat * sizeof(double), cudaMemcpyDefault, c.stream));
  const dim3 gi = grid_for(g.n[0], g.n[1], g.n[2]);
  pack3_kernel<<<gi, 128, 0, c.stream>>>(g, staging, c.buf[0], 0, nullptr);
  ++c.launches;
  launch_ghost(c, c.buf[0], 1);
  {
    Timed t(c, 1);     // derived quantities on every padded cell, once (afterwards the stage epilogues keep them current)
    // (both sets: the frozen ghosts of fixed sides are never written again)
    derive3_kernel<<<grid_for(g.n[0] + 6, g.n[1] + 6, g.n[2] + 6), 128, 0, c.stream>>>(g, cv8(c.buf[0]), c.der[0]);
    derive3_kernel<<<grid_for(g.n[0] + 6, g.n[1] + 6, g.n[2] + 6), 128, 0, c.stream>>>(g, cv8(c.buf[0]), c.der[1]);
    ++c.launches;
  }
  // the other two buffers that are read with a halo get the same frozen ghosts (fixed sides are never rewritten)
  for (int b = 1; b <= 2; ++b)
    for (int f = 0; f < NF; ++f)
      CUDA_TRY(cudaMemcpyAsync(c.buf[b].p[f], c.buf[0].p[f], (size_t)g.vol * sizeof(double), cudaMemcpyDeviceToDevice, c.stream));
  CUDA_TRY(cudaMemsetAsync(c.sc, 0, sizeof(Scalars3), c.stream));
  c.cur = 0;
  wavespeed3_kernel<<<gi, 128, 0, c.stream>>>(g, cv8(c.buf[0]), c.gamma, c.sc, 0);
  ++c.launches;
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaStreamSynchronize(c.stream));
  return SMAUG3_OK;
}

int smaug3_step(smaug3_ctx* ctx, int n_steps, double cfl) {
  if (!ctx || n_steps < 0) return fail(SMAUG3_EINVAL, "bad argument");
  Ctx& c = *CTX(ctx);
  if (c.fixed_dt <= 0.0 && !(cfl > 0.0)) return fail(SMAUG3_EINVAL, "cfl must be > 0");
  DeviceGuard guard_(c.device);
  for (int s = 0; s < n_steps; ++s) enqueue_step(c, cfl);
  CUDA_TRY(cudaGetLastError());
  Scalars3 h;
  CUDA_TRY(cudaMemcpyAsync(&h, c.sc, sizeof(h), cudaMemcpyDeviceToHost, c.stream));
  CUDA_TRY(cudaStreamSynchronize(c.stream));
  if (h.status) return fail(SMAUG3_ENONFINITE, "non-finite or non-positive dt");
  return SMAUG3_OK;
}

int smaug3_get_state(smaug3_ctx* ctx, void* w) {
  if (!ctx || !w) return fail(SMAUG3_EINVAL, "NULL argument");
  Ctx& c = *CTX(ctx);
  DeviceGuard guard_(c.device);
  const Grid3& g = c.g;
  const size_t nflat = (size_t)NF * g.n[0] * g.n[1] * g.n[2];
  double* staging = c.cf[0].p[0];
  pack3_kernel<<<grid_for(g.n[0], g.n[1], g.n[2]), 128, 0, c.stream>>>(g, nullptr, c.buf[0], 1, staging);
  ++c.launches;
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpyAsync(w, staging, nflat * sizeof(double), cudaMemcpyDefault, c.stream));
  CUDA_TRY(cudaStreamSynchronize(c.stream));
  return SMAUG3_OK;
}

int smaug3_get_time(smaug3_ctx* ctx, double* t, double* last_dt) {
  if (!ctx) return fail(SMAUG3_EINVAL, "NULL ctx");
  Ctx& c = *CTX(ctx);
  DeviceGuard guard_(c.device);
  Scalars3 h;
  CUDA_TRY(cudaMemcpyAsync(&h, c.sc, sizeof(h), cudaMemcpyDeviceToHost, c.stream));
  CUDA_TRY(cudaStreamSynchronize(c.stream));
  if (t) *t = h.t;
  if (last_dt) *last_dt = h.dt;
  return SMAUG3_OK;
}

int smaug3_get_wavespeeds(smaug3_ctx* ctx, double out[5]) {
  if (!ctx || !out) return fail(SMAUG3_EINVAL, "NULL argument");
  Ctx& c = *CTX(ctx);
  DeviceGuard guard_(c.device);
  Scalars3 h;
  CUDA_TRY(cudaMemcpyAsync(&h, c.sc, sizeof(h), cudaMemcpyDeviceToHost, c.stream));
  CUDA_TRY(cudaStreamSynchronize(c.stream));
  for (int k = 0; k < 5; ++k) {
    const unsigned long long u = h.red[c.cur][k];
    double d;
    memcpy(&d, &u, sizeof(d));
    out[k] = d;
  }
  return SMAUG3_OK;
}

int smaug3_get_launch_count(smaug3_ctx* ctx, long long* n) {
  if (!ctx || !n) return fail(SMAUG3_EINVAL, "NULL argument");
  *n = CTX(ctx)->launches;
  return SMAUG3_OK;
}

int smaug3_set_kernel_timing(smaug3_ctx* ctx, int on) {
  if (!ctx) return fail(SMAUG3_EINVAL, "NULL ctx");
  Ctx& c = *CTX(ctx);
  DeviceGuard guard_(c.device);
  CUDA_TRY(cudaStreamSynchronize(c.stream));      // recorded events may still be pending: settle them before the pool is reused
  c.timing = on != 0;
  c.timing_broken = false;
  c.ev_used = 0;
  for (int k = 0; k < 5; ++k) { c.ms[k] = 0; c.nk[k] = 0; }
  return SMAUG3_OK;
}

int smaug3_get_kernel_timing(smaug3_ctx* ctx, double ms[5], long long n[5]) {
  if (!ctx || !ms || !n) return fail(SMAUG3_EINVAL, "NULL argument");
  Ctx& c = *CTX(ctx);
  DeviceGuard guard_(c.device);
  CUDA_TRY(cudaStreamSynchronize(c.stream));
  if (c.timing_broken) return fail(SMAUG3_ECUDA, "kernel timing was abandoned: a CUDA event could not be created or recorded");
  for (size_t e = 0; e + 1 < c.ev_used; e += 2) {
    float t = 0;
    CUDA_TRY(cudaEventElapsedTime(&t, c.ev[e], c.ev[e + 1]));
    c.ms[c.ev_kind[e]] += t;
    c.nk[c.ev_kind[e]] += 1;
  }
  c.ev_used = 0;
  for (int k = 0; k < 5; ++k) { ms[k] = c.ms[k]; n[k] = c.nk[k]; }
  return SMAUG3_OK;
}

}  // extern "C"
