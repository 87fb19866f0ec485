// oracle/smaug3d_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// The three-dimensional form of the scheme ("the 3-dimensional MHD
// equations", "implemented in 3D"): a plain, slow CPU implementation in fp64 -- straight loops over
// ghost-padded volumes, one full-size temporary per intermediate quantity -- of one SMAUG+ time step on an
// nx x ny x nz grid with the eight fields w = (rho, mx, my, mz, e, bx, by, bz), zero background.  It is the
// two-dimensional oracle (smaug_oracle.cpp; readings c-1..c-10 of DESIGN.md section 3) with every sum over
// directions and components running to three; the few places where the third dimension needs a choice are the
// reading c-11 of DESIGN.md section 3 and are marked [c-11] below.  It shares no code with the CUDA path and none
// with smaug_oracle.cpp (a separate translation unit and library, so that the 2-D oracle can serve as a pin).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may load it.
//
// Parity pins (tests/test_oracle3d_pins.py; none re-types a formula of this file):
//   D1  z-invariant data (mz = bz = 0, nz = 1 or 5) reproduces the pinned 2-D oracle cell for cell (rhs, steps, dt,
//       maxima): every x/y term, the RK combine, dt, the ghost fill in x and y
//   D2  cyclic axis permutation x -> y -> z -> x (and the swap x <-> z) of a fully three-dimensional state: rhs and
//       steps of the permuted problem are the permuted results: every term that involves z is the image of a term
//       D1 pins (fluxes, kappa_z, interface and mixed fluxes along / across z, the energy couplings, cmax_z)
//   D3  uniform states are fixed points, bit for bit, for every boundary kind (P1 in 3-D)
//   D4  conservation of all eight sums on a periodic box with hyperdiffusion on (every term is a flux difference)
//   D5  ghost fill against numpy.pad on the padded volume, edges and corners included; fixed ghosts stay frozen
//   D6  closed-form maxima and dt of a uniform magnetised flow (cmax_z and the n = 1 rule in 3-D)
//   D7  central div B is preserved to rounding with hyperdiffusion off (the central operators commute)
//   D8  temporal order 4 and spatial order 4 of a 3-D oblique smooth problem (HD off)
// Against SAC/SMAUG themselves parity is unpinned, as for the 2-D oracle (the paper prints no field values).

#include <algorithm>
#include <cmath>
#include <cstring>
#include <string>
#include <vector>

namespace {

constexpr int NG = 3;
enum { F_RHO = 0, F_MX = 1, F_MY = 2, F_MZ = 3, F_E = 4, F_BX = 5, F_BY = 6, F_BZ = 7, NF = 8 };
enum { BC_PERIODIC = 0, BC_OPEN = 1, BC_FIXED = 2 };
enum {   // parameter keys: 0..12 as in the 2-D interface, 13.. the third dimension
  P_LX = 0, P_LY = 1, P_HD_ON = 2, P_C_RHO = 3, P_C_MOM = 4, P_C_E = 5, P_C_B = 6, P_RK_ORDER = 7,
  P_FIXED_DT = 8, P_GX = 10, P_GY = 11, P_LZ = 13, P_GZ = 14
};
enum { OK = 0, EINVAL_ = -1, ENONFINITE_ = -4 };

typedef std::vector<double> Vol;

struct Ctx {
  int n[3], N[3];           // interior and padded cell counts along x, y, z
  double gamma;
  int bc[6];                // x_lo, x_hi, y_lo, y_hi, z_lo, z_hi
  double L[3] = {1.0, 1.0, 1.0};
  int hd_on = 1;
  double c_rho = 0.02, c_mom = 0.4, c_e = 0.02, c_b = 0.02;
  int rk_order = 4;
  double fixed_dt = 0.0;
  double g[3] = {0.0, 0.0, 0.0};
  Vol w[NF];
  double t = 0.0, last_dt = 0.0;
  int nthreads = 1;
  size_t vsize() const { return (size_t)N[0] * N[1] * N[2]; }
  long stride(int d) const { return d == 0 ? 1 : (d == 1 ? (long)N[0] : (long)N[0] * N[1]); }
  size_t at(int i, int j, int k) const { return ((size_t)(k + NG) * N[1] + (j + NG)) * N[0] + (i + NG); }
  double inv_d(int d) const { return n[d] / L[d]; }
};

thread_local std::string g_err;

int wrap(int i, int n) { return ((i % n) + n) % n; }

// c-8 in three dimensions [c-11]: x over interior (j, k), then y over the full padded x-extent and interior k, then z
// over the full padded x- and y-extents (edges and corners come out of the composition).  periodic: wrap (works for
// n < 3); open: nearest interior cell; fixed: untouched unless `freeze` (set_state: nearest interior value, once).
void fill_ghosts(const Ctx& c, Vol& p, bool freeze) {
  const int nx = c.n[0], ny = c.n[1], nz = c.n[2];
  auto side = [&](int axis, int lo_hi, int g, int& dst, int& src) -> bool {     // ghost layer g = 1..3 of one side
    const int n = c.n[axis], kind = c.bc[2 * axis + lo_hi];
    dst = lo_hi == 0 ? -g : n - 1 + g;
    if (kind == BC_PERIODIC) { src = wrap(dst, n); return true; }
    if (kind == BC_OPEN || freeze) { src = lo_hi == 0 ? 0 : n - 1; return true; }
    return false;
  };
  int dst, src;
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int g = 1; g <= NG; ++g)
        for (int s = 0; s < 2; ++s)
          if (side(0, s, g, dst, src)) p[c.at(dst, j, k)] = p[c.at(src, j, k)];
  for (int k = 0; k < nz; ++k)
    for (int i = -NG; i < nx + NG; ++i)
      for (int g = 1; g <= NG; ++g)
        for (int s = 0; s < 2; ++s)
          if (side(1, s, g, dst, src)) p[c.at(i, dst, k)] = p[c.at(i, src, k)];
  for (int j = -NG; j < ny + NG; ++j)
    for (int i = -NG; i < nx + NG; ++i)
      for (int g = 1; g <= NG; ++g)
        for (int s = 0; s < 2; ++s)
          if (side(2, s, g, dst, src)) p[c.at(i, j, dst)] = p[c.at(i, j, src)];
}

// The arithmetic contract of DESIGN.md section 4 holds here as well: every formula is an explicit sequence of
// IEEE-754 binary64 operations, `fma` is one rounding, the file is compiled with -ffp-contract=off.  Sums over the
// three components are nested x innermost, z outermost [c-11] -- fma(z.., fma(y.., x..)) -- so that with a vanishing
// z-component every value is the 2-D oracle's, bit for bit.
using std::fma;

// c-2 derived quantities (zero background): v = m (1/rho), eps = e - rho v^2/2 - b^2/2 = p_k/(gamma-1),
// p_t = (gamma-1) eps + b^2/2.
struct Derived {
  Vol v[3], ptt, eps;
};

void derived(const Ctx& c, const Vol* w, Derived& d) {
  const size_t n = c.vsize();
  const double gm1 = c.gamma - 1.0;
  for (Vol* p : {&d.v[0], &d.v[1], &d.v[2], &d.ptt, &d.eps}) p->assign(n, 0.0);
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (long q = 0; q < (long)n; ++q) {
    const double rr = 1.0 / w[F_RHO][q];
    const double mx = w[F_MX][q], my = w[F_MY][q], mz = w[F_MZ][q];
    const double vx = mx * rr, vy = my * rr, vz = mz * rr;
    const double bx = w[F_BX][q], by = w[F_BY][q], bz = w[F_BZ][q];
    const double b2h = 0.5 * fma(bz, bz, fma(by, by, bx * bx));
    const double ke = 0.5 * fma(mz, vz, fma(my, vy, mx * vx));
    const double eps = (w[F_E][q] - ke) - b2h;
    d.v[0][q] = vx; d.v[1][q] = vy; d.v[2][q] = vz;
    d.eps[q] = eps;
    d.ptt[q] = fma(gm1, eps, b2h);
  }
}

// c-3 along any axis (stride s): cd12 = 8 (f[+1] - f[-1]) - (f[+2] - f[-2]) = 12 Delta df/dx
inline double cd12(const Vol& f, size_t q, size_t s) {
  return fma(8.0, f[q + s] - f[q - s], -(f[q + 2 * s] - f[q - 2 * s]));
}

// c-2 fluxes of PAPER.md:35 along direction dir at padded cell q (mu0 = 1):
//   F_d(rho) = rho v_d;  F_d(m_l) = m_l v_d - b_l b_d + delta_ld p_t;  F_d(e) = v_d (e + p_t) - b_d (b.v);
//   F_d(b_l) = v_d b_l - b_d v_l (0 for l = d)
double flux(const Vol* w, const Derived& d, int field, int dir, size_t q) {
  const double v[3] = {d.v[0][q], d.v[1][q], d.v[2][q]};
  const double b[3] = {w[F_BX][q], w[F_BY][q], w[F_BZ][q]};
  if (field == F_RHO) return w[F_RHO][q] * v[dir];
  if (field >= F_MX && field <= F_MZ) {
    const int l = field - F_MX;
    const double f = fma(w[F_MX + l][q], v[dir], -(b[l] * b[dir]));
    return l == dir ? f + d.ptt[q] : f;
  }
  if (field == F_E) {
    const double bv = fma(b[2], v[2], fma(b[1], v[1], b[0] * v[0]));
    const double h = w[F_E][q] + d.ptt[q];
    return fma(v[dir], h, -(b[dir] * bv));
  }
  const int l = field - F_BX;
  if (l == dir) return 0.0;
  return fma(v[dir], b[l], -(b[dir] * v[l]));
}

// c-5 hyperviscosity coefficient along dir of the scalar u, stored as kappa = nu / Delta at the
// padded index of the cell left of the interface; computed for interfaces -1 .. n-1 along dir and for every padded
// index across it.  M3 = max |D3| over 3 interfaces, M1 = max |D1| over 5, kappa = cv (M3 / M1), 0 if M1 = 0.
void hyper_kappa(const Ctx& c, const Vol& u, int dir, double cv, Vol& kap) {
  kap.assign(c.vsize(), 0.0);
  const long s = c.stride(dir);
  const int a1 = (dir + 1) % 3, a2 = (dir + 2) % 3;          // the two axes across dir
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int p2 = 0; p2 < c.N[a2]; ++p2)
    for (int p1 = 0; p1 < c.N[a1]; ++p1)
      for (int k = -1; k <= c.n[dir] - 1; ++k) {
        const long q = (long)p2 * c.stride(a2) + (long)p1 * c.stride(a1) + (long)(k + NG) * s;
        double M3 = 0.0, M1 = 0.0;
        for (int o = -1; o <= 1; ++o) {
          const long r = q + o * s;
          const double d3 = fma(3.0, u[r + s] - u[r], -(u[r + 2 * s] - u[r - s]));
          M3 = std::max(M3, std::fabs(d3));
        }
        for (int o = -2; o <= 2; ++o) {
          const long r = q + o * s;
          M1 = std::max(M1, std::fabs(u[r + s] - u[r]));
        }
        kap[q] = M1 > 0.0 ? cv * (M3 / M1) : 0.0;
      }
}

enum { K_RHO = 0, K_V = 1, K_EPS = 4, K_B = 5, NK = 8 };    // K_V + l: of v_l;  K_B + l: of b_l (unused for l = dir)
struct Kappas {
  Vol k[3][NK];      // k[dir][family]
};

// c-5 interface fluxes along dir between cells a and b = a + stride(dir): Phi = g kappa (q_b - q_a) with
//   rho: g = 1;  m_l: g = rho-bar (l = dir) or rho-bar/2 (l != dir), q = v_l;  eps: g = 1;  b_l (l != dir): g = 1;
//   e: Phi(eps) + sum_l vbar_l Phi(m_l) + sum_{l != dir} Bbar_l Phi(b_l)   [c-11: l ascending, v before B]
void hd_interface_fluxes(const Ctx& c, const Vol* w, const Derived& d, const Kappas& K, int dir, long a, double out[NF]) {
  const long b = a + c.stride(dir);
  const Vol* kap = K.k[dir];
  const double rbar = 0.5 * (w[F_RHO][a] + w[F_RHO][b]);
  double e = kap[K_EPS][a] * (d.eps[b] - d.eps[a]);
  out[F_RHO] = kap[K_RHO][a] * (w[F_RHO][b] - w[F_RHO][a]);
  for (int l = 0; l < 3; ++l) {
    const double gl = l == dir ? rbar : 0.5 * rbar;
    const double pm = (gl * kap[K_V + l][a]) * (d.v[l][b] - d.v[l][a]);
    out[F_MX + l] = pm;
    e = fma(0.5 * (d.v[l][a] + d.v[l][b]), pm, e);
  }
  for (int l = 0; l < 3; ++l) {
    if (l == dir) { out[F_BX + l] = 0.0; continue; }
    const Vol& bl = w[F_BX + l];
    const double pb = kap[K_B + l][a] * (bl[b] - bl[a]);
    out[F_BX + l] = pb;
    e = fma(0.5 * (bl[a] + bl[b]), pb, e);
  }
  out[F_E] = e;
}

// c-5 mixed terms [c-11]: the viscous stress tau_kl = (rho/2) [nu_k(v_l) d_k v_l + nu_l(v_k) d_l v_k] and the
// resistive field eps = nu o curl b, written per direction k as cell-centred fluxes built from derivatives along
// each l != k:  G(m_l ; k) = (rho/2) nubar_l(v_k) d^c_l v_k,  G(b_l ; k) = - nubar_l(b_k) d^c_l b_k,
//               G(e ; k) = sum_{l != k} [ v_l G(m_l ; k) + B_l G(b_l ; k) ]      (l ascending)
// They enter as + d^c_k G, i.e. C_k = F_k - G_k.  Defined on [-2, n+2) along k and interior cells across it.
void hd_mixed_fluxes(const Ctx& c, const Vol* w, const Derived& d, const Kappas& K, int k, Vol* G) {
  for (int f = 0; f < NF; ++f) G[f].assign(c.vsize(), 0.0);
  int lo[3] = {0, 0, 0}, hi[3] = {c.n[0], c.n[1], c.n[2]};
  lo[k] = -2; hi[k] = c.n[k] + 2;
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int kk = lo[2]; kk < hi[2]; ++kk)
    for (int j = lo[1]; j < hi[1]; ++j)
      for (int i = lo[0]; i < hi[0]; ++i) {
        const long q = (long)c.at(i, j, kk);
        double ge = 0.0;
        bool first = true;
        for (int l = 0; l < 3; ++l) {
          if (l == k) continue;
          const long sl = c.stride(l);
          const Vol& kv = K.k[l][K_V + k];
          const Vol& kb = K.k[l][K_B + k];
          const double kbar_v = 0.5 * (kv[q - sl] + kv[q]);
          const double kbar_b = 0.5 * (kb[q - sl] + kb[q]);
          const double dv = cd12(d.v[k], (size_t)q, (size_t)sl) * (1.0 / 12.0);
          const double db = cd12(w[F_BX + k], (size_t)q, (size_t)sl) * (1.0 / 12.0);
          const double gm = ((0.5 * w[F_RHO][q]) * kbar_v) * dv;
          const double gb = -(kbar_b * db);
          G[F_MX + l][q] = gm;
          G[F_BX + l][q] = gb;
          if (first) ge = fma(d.v[l][q], gm, w[F_BX + l][q] * gb);
          else ge = fma(w[F_BX + l][q], gb, fma(d.v[l][q], gm, ge));
          first = false;
        }
        G[F_E][q] = ge;
      }
}

// c-4 maxima over interior cells: out = { max(|v_d| + c_f,d) for d = x, y, z, max a^2, max b^2 }
void wavespeeds(const Ctx& c, const Vol* w, double out[5]) {
  double m0 = 0, m1 = 0, m2 = 0, m3 = 0, m4 = 0;
  const double gm1 = c.gamma - 1.0;
#pragma omp parallel for num_threads(c.nthreads) schedule(static) reduction(max : m0, m1, m2, m3, m4)
  for (int k = 0; k < c.n[2]; ++k)
    for (int j = 0; j < c.n[1]; ++j)
      for (int i = 0; i < c.n[0]; ++i) {
        const size_t q = c.at(i, j, k);
        const double rr = 1.0 / w[F_RHO][q];
        const double mx = w[F_MX][q], my = w[F_MY][q], mz = w[F_MZ][q];
        const double vx = mx * rr, vy = my * rr, vz = mz * rr;
        const double Bx = w[F_BX][q], By = w[F_BY][q], Bz = w[F_BZ][q];
        const double B2 = fma(Bz, Bz, fma(By, By, Bx * Bx));
        const double pk = gm1 * ((w[F_E][q] - 0.5 * fma(mz, vz, fma(my, vy, mx * vx))) - 0.5 * B2);
        const double a2 = (c.gamma * pk) * rr;
        const double b2 = B2 * rr;
        const double s = a2 + b2;
        const double fa = (4.0 * a2) * rr;
        const double cfx2 = 0.5 * (s + std::sqrt(std::max(0.0, fma(s, s, -(fa * (Bx * Bx))))));
        const double cfy2 = 0.5 * (s + std::sqrt(std::max(0.0, fma(s, s, -(fa * (By * By))))));
        const double cfz2 = 0.5 * (s + std::sqrt(std::max(0.0, fma(s, s, -(fa * (Bz * Bz))))));
        const double cx = std::fabs(vx) + std::sqrt(cfx2);
        const double cy = std::fabs(vy) + std::sqrt(cfy2);
        const double cz = std::fabs(vz) + std::sqrt(cfz2);
        if (cx > m0) m0 = cx;
        if (cy > m1) m1 = cy;
        if (cz > m2) m2 = cz;
        if (a2 > m3) m3 = a2;
        if (b2 > m4) m4 = b2;
      }
  out[0] = m0; out[1] = m1; out[2] = m2; out[3] = m3; out[4] = m4;
}

// c-6: R(w) = - sum_d d^c_d (F_d - G_d) + rho g (momentum), rho g.v (energy) + sum_d (Phi_d+ - Phi_d-)/Delta_d
void rhs(const Ctx& c, const Vol* w, Vol* R) {
  const size_t n = c.vsize();
  const double id[3] = {c.inv_d(0), c.inv_d(1), c.inv_d(2)};
  Derived d;
  derived(c, w, d);
  Kappas K;
  Vol G[3][NF];
  for (int k = 0; k < 3; ++k)
    for (int f = 0; f < NF; ++f) G[k][f].assign(n, 0.0);
  if (c.hd_on) {
    double ws[5];
    wavespeeds(c, w, ws);
    const double vt = std::sqrt(ws[3]) + std::sqrt(ws[4]);
    const double cv_rho = c.c_rho * vt, cv_mom = c.c_mom * vt, cv_e = c.c_e * vt, cv_b = c.c_b * vt;
    for (int dir = 0; dir < 3; ++dir) {
      hyper_kappa(c, w[F_RHO], dir, cv_rho, K.k[dir][K_RHO]);
      for (int l = 0; l < 3; ++l) hyper_kappa(c, d.v[l], dir, cv_mom, K.k[dir][K_V + l]);
      hyper_kappa(c, d.eps, dir, cv_e, K.k[dir][K_EPS]);
      for (int l = 0; l < 3; ++l) {
        if (l == dir) K.k[dir][K_B + l].assign(n, 0.0);
        else hyper_kappa(c, w[F_BX + l], dir, cv_b, K.k[dir][K_B + l]);
      }
    }
    for (int k = 0; k < 3; ++k) hd_mixed_fluxes(c, w, d, K, k, G[k]);
  }
  Vol C[3];
  for (int k = 0; k < 3; ++k) C[k].assign(n, 0.0);
  for (int f = 0; f < NF; ++f) {
    R[f].assign(n, 0.0);
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
    for (long q = 0; q < (long)n; ++q)
      for (int k = 0; k < 3; ++k) C[k][q] = flux(w, d, f, k, (size_t)q) - G[k][f][q];
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
    for (int k = 0; k < c.n[2]; ++k)
      for (int j = 0; j < c.n[1]; ++j)
        for (int i = 0; i < c.n[0]; ++i) {
          const size_t q = c.at(i, j, k);
          R[f][q] = fma(cd12(C[0], q, 1), id[0],
                        fma(cd12(C[1], q, (size_t)c.stride(1)), id[1], cd12(C[2], q, (size_t)c.stride(2)) * id[2])) *
                    (-1.0 / 12.0);
        }
  }
  if (c.g[0] != 0.0 || c.g[1] != 0.0 || c.g[2] != 0.0) {      // c-10 with a zero background: rho g, rho g.v
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
    for (int k = 0; k < c.n[2]; ++k)
      for (int j = 0; j < c.n[1]; ++j)
        for (int i = 0; i < c.n[0]; ++i) {
          const size_t q = c.at(i, j, k);
          const double rt = w[F_RHO][q];
          for (int l = 0; l < 3; ++l) R[F_MX + l][q] = fma(rt, c.g[l], R[F_MX + l][q]);
          R[F_E][q] = fma(rt, fma(c.g[2], d.v[2][q], fma(c.g[1], d.v[1][q], c.g[0] * d.v[0][q])), R[F_E][q]);
        }
  }
  if (c.hd_on) {
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
    for (int k = 0; k < c.n[2]; ++k)
      for (int j = 0; j < c.n[1]; ++j)
        for (int i = 0; i < c.n[0]; ++i) {
          const long q = (long)c.at(i, j, k);
          double lo[NF], hi[NF];
          for (int dir = 0; dir < 3; ++dir) {
            hd_interface_fluxes(c, w, d, K, dir, q - c.stride(dir), lo);
            hd_interface_fluxes(c, w, d, K, dir, q, hi);
            for (int f = 0; f < NF; ++f) R[f][q] = fma(hi[f] - lo[f], id[dir], R[f][q]);
          }
        }
  }
}

// c-7: dt = cfl min_d (Delta_d / cmax_d) over the axes with more than one cell
double cfl_dt(const Ctx& c, const Vol* w, double cfl) {
  double ws[5];
  wavespeeds(c, w, ws);
  double m = INFINITY;
  for (int d = 0; d < 3; ++d)
    if (c.n[d] > 1) m = std::min(m, (c.L[d] / c.n[d]) / ws[d]);
  return cfl * m;
}

void finish_stage(const Ctx& c, const Vol* wn, Vol* ws) {     // ghosts from w^n (keeps frozen fixed ghosts), then refill
  for (int f = 0; f < NF; ++f) {
    for (int k = -NG; k < c.n[2] + NG; ++k)
      for (int j = -NG; j < c.n[1] + NG; ++j)
        for (int i = -NG; i < c.n[0] + NG; ++i)
          if (i < 0 || i >= c.n[0] || j < 0 || j >= c.n[1] || k < 0 || k >= c.n[2]) ws[f][c.at(i, j, k)] = wn[f][c.at(i, j, k)];
    fill_ghosts(c, ws[f], false);
  }
}

// c-6 classical RK4 in stage-state form (see smaug_oracle.cpp): w1 = w^n + dt/2 R(w^n), w2 = w^n + dt/2 R(w1),
// w3 = w^n + dt R(w2), acc = (w1 - w^n) + 2 w2, w^{n+1} = w3 + (acc - 2 w3)/3 + dt/6 R(w3); order 2 = midpoint, 1 = Euler.
void rk_step(Ctx& c, double dt) {
  const size_t n = c.vsize();
  Vol R[NF], w1[NF], w2[NF], w3[NF], wnew[NF];
  Vol* wn = c.w;
  auto interior = [&](auto&& body) {
    for (int k = 0; k < c.n[2]; ++k)
      for (int j = 0; j < c.n[1]; ++j)
        for (int i = 0; i < c.n[0]; ++i) body(c.at(i, j, k));
  };
  auto axpy = [&](double a, Vol* out) {
    for (int f = 0; f < NF; ++f) {
      out[f].assign(n, 0.0);
      interior([&](size_t q) { out[f][q] = fma(a, R[f][q], wn[f][q]); });
    }
    finish_stage(c, wn, out);
  };
  for (int f = 0; f < NF; ++f) fill_ghosts(c, wn[f], false);
  rhs(c, wn, R);
  if (c.rk_order == 1) {
    axpy(dt, wnew);
  } else if (c.rk_order == 2) {
    axpy(0.5 * dt, w1);
    rhs(c, w1, R);
    axpy(dt, wnew);
  } else {
    axpy(0.5 * dt, w1);
    rhs(c, w1, R);
    axpy(0.5 * dt, w2);
    rhs(c, w2, R);
    axpy(dt, w3);
    rhs(c, w3, R);
    const double dt6 = (1.0 / 6.0) * dt;
    for (int f = 0; f < NF; ++f) {
      wnew[f].assign(n, 0.0);
      interior([&](size_t q) {
        const double acc = fma(2.0, w2[f][q], w1[f][q] - wn[f][q]);
        wnew[f][q] = fma(dt6, R[f][q], fma(fma(-2.0, w3[f][q], acc), 1.0 / 3.0, w3[f][q]));
      });
    }
    finish_stage(c, wn, wnew);
  }
  for (int f = 0; f < NF; ++f) c.w[f].swap(wnew[f]);
  c.t += dt;
  c.last_dt = dt;
}

}  // namespace

// C ABI (host pointers only).  State layout [field][nz][ny][nx], x fastest, interior cells, fp64.
typedef struct oracle3_ctx oracle3_ctx;
#define CTX(p) (reinterpret_cast<Ctx*>(p))

extern "C" {

const char* oracle3_last_error(void) { return g_err.c_str(); }

int oracle3_create(int nx, int ny, int nz, double gamma, const int bc[6], oracle3_ctx** out) {
  if (!out || !bc) { g_err = "NULL argument"; return EINVAL_; }
  *out = nullptr;
  if (nx < 1 || ny < 1 || nz < 1) { g_err = "nx, ny, nz must be >= 1"; return EINVAL_; }
  if (!(gamma > 1.0)) { g_err = "gamma must be > 1"; return EINVAL_; }
  for (int s = 0; s < 6; ++s)
    if (bc[s] < 0 || bc[s] > 2) { g_err = "unknown boundary kind"; return EINVAL_; }
  for (int a = 0; a < 3; ++a)
    if ((bc[2 * a] == BC_PERIODIC) != (bc[2 * a + 1] == BC_PERIODIC)) {
      g_err = "periodic must be set on both sides of an axis";
      return EINVAL_;
    }
  Ctx* c = new Ctx();
  c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
  for (int d = 0; d < 3; ++d) c->N[d] = c->n[d] + 2 * NG;
  c->gamma = gamma;
  for (int s = 0; s < 6; ++s) c->bc[s] = bc[s];
  for (int f = 0; f < NF; ++f) c->w[f].assign(c->vsize(), 0.0);
  *out = reinterpret_cast<oracle3_ctx*>(c);
  return OK;
}

void oracle3_destroy(oracle3_ctx* p) { delete CTX(p); }

int oracle3_set_param(oracle3_ctx* p, int key, double v) {
  if (!p) { g_err = "NULL ctx"; return EINVAL_; }
  Ctx& c = *CTX(p);
  switch (key) {
    case P_LX: if (!(v > 0)) break; c.L[0] = v; return OK;
    case P_LY: if (!(v > 0)) break; c.L[1] = v; return OK;
    case P_LZ: if (!(v > 0)) break; c.L[2] = v; return OK;
    case P_HD_ON: c.hd_on = v != 0.0; return OK;
    case P_C_RHO: if (!(v >= 0)) break; c.c_rho = v; return OK;
    case P_C_MOM: if (!(v >= 0)) break; c.c_mom = v; return OK;
    case P_C_E: if (!(v >= 0)) break; c.c_e = v; return OK;
    case P_C_B: if (!(v >= 0)) break; c.c_b = v; return OK;
    case P_RK_ORDER: if (v != 1 && v != 2 && v != 4) break; c.rk_order = (int)v; return OK;
    case P_FIXED_DT: if (!(v >= 0)) break; c.fixed_dt = v; return OK;
    case P_GX: if (!std::isfinite(v)) break; c.g[0] = v; return OK;
    case P_GY: if (!std::isfinite(v)) break; c.g[1] = v; return OK;
    case P_GZ: if (!std::isfinite(v)) break; c.g[2] = v; return OK;
    default: g_err = "unknown parameter key"; return EINVAL_;
  }
  g_err = "parameter value out of range";
  return EINVAL_;
}

int oracle3_set_threads(oracle3_ctx* p, int n) {
  if (!p || n < 1) { g_err = "bad argument"; return EINVAL_; }
  CTX(p)->nthreads = n;
  return OK;
}

static void copy_interior(Ctx& c, Vol* vols, double* flat, bool to_flat) {
  for (int f = 0; f < NF; ++f)
    for (int k = 0; k < c.n[2]; ++k)
      for (int j = 0; j < c.n[1]; ++j)
        for (int i = 0; i < c.n[0]; ++i) {
          const size_t o = (((size_t)f * c.n[2] + k) * c.n[1] + j) * c.n[0] + i;
          if (to_flat) flat[o] = vols[f][c.at(i, j, k)];
          else vols[f][c.at(i, j, k)] = flat[o];
        }
}

int oracle3_set_state(oracle3_ctx* p, const double* w) {
  if (!p || !w) { g_err = "NULL argument"; return EINVAL_; }
  Ctx& c = *CTX(p);
  copy_interior(c, c.w, const_cast<double*>(w), false);
  for (int f = 0; f < NF; ++f) fill_ghosts(c, c.w[f], true);
  c.t = 0.0; c.last_dt = 0.0;
  return OK;
}

int oracle3_get_state(oracle3_ctx* p, double* w) {
  if (!p || !w) { g_err = "NULL argument"; return EINVAL_; }
  copy_interior(*CTX(p), CTX(p)->w, w, true);
  return OK;
}

int oracle3_get_time(oracle3_ctx* p, double* t, double* last_dt) {
  if (!p) { g_err = "NULL ctx"; return EINVAL_; }
  if (t) *t = CTX(p)->t;
  if (last_dt) *last_dt = CTX(p)->last_dt;
  return OK;
}

int oracle3_step(oracle3_ctx* p, int n_steps, double cfl) {
  if (!p || n_steps < 0) { g_err = "bad argument"; return EINVAL_; }
  Ctx& c = *CTX(p);
  if (c.fixed_dt <= 0.0 && !(cfl > 0.0)) { g_err = "cfl must be > 0"; return EINVAL_; }
  for (int s = 0; s < n_steps; ++s) {
    const double dt = c.fixed_dt > 0.0 ? c.fixed_dt : cfl_dt(c, c.w, cfl);
    if (!(dt > 0.0) || !std::isfinite(dt)) { g_err = "non-finite or non-positive dt"; return ENONFINITE_; }
    rk_step(c, dt);
  }
  return OK;
}

int oracle3_rhs(oracle3_ctx* p, double* R) {       // R(w) of the current state, [8][nz][ny][nx]
  if (!p || !R) { g_err = "NULL argument"; return EINVAL_; }
  Ctx& c = *CTX(p);
  Vol k[NF];
  for (int f = 0; f < NF; ++f) fill_ghosts(c, c.w[f], false);
  rhs(c, c.w, k);
  copy_interior(c, k, R, true);
  return OK;
}

int oracle3_wavespeeds(oracle3_ctx* p, double out[5]) {
  if (!p || !out) { g_err = "NULL argument"; return EINVAL_; }
  wavespeeds(*CTX(p), CTX(p)->w, out);
  return OK;
}

int oracle3_get_padded(oracle3_ctx* p, int f, double* out) {     // the padded volume of field f as it currently is
  if (!p || !out || f < 0 || f >= NF) { g_err = "bad argument"; return EINVAL_; }
  std::memcpy(out, CTX(p)->w[f].data(), CTX(p)->vsize() * sizeof(double));
  return OK;
}

}  // extern "C"
