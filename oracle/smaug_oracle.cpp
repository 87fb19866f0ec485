// oracle/smaug_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, obviously-correct CPU implementation (C++17, fp64, straight loops over
// ghost-padded arrays, one full-size temporary per intermediate quantity) of one SMAUG+ time step
// on a 2-D grid, written from the paper (/root/reference/PAPER.md = "PAPER.md" below) and from the
// readings listed in DESIGN.md section 3 (= SURVEY.md section 8(c), "c-1".."c-9").  It shares no code
// with the CUDA path under paper_1710_06423_b200/csrc/ and neither includes the other.  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
//
// Parity pins (tests/test_oracle_pins.py, none of them re-types a formula of this file):
//   fill_ghosts            P5 (ny=1 == ny=8), P3 (periodic wrap keeps the OT point symmetry), brute force
//   central differences    P4 (numerical phase speed k*), P6 (4th-order convergence), exact on cubics
//   fluxes / split form    P1, P2 (conservation), P4 (sound/Alfven/fast/slow phase speeds), split==unsplit
//   hyper_kappa            P8 (unit-step worked example 1,2,2,2,1), P9 (closed form on a sine), P10 (bound 4)
//   hyper_div              P1, P2 (conservation incl. energy couplings), P3, P5 (x<->y transposition)
//   wavespeeds / dt        P11 (closed-form Brio-Wu and Orszag-Tang maxima and dt0)
//   rk4_step               P6 (temporal order 4), P4 (RK4 amplification factor), P12 (restart)
//   gravity (c-10)         G1 (hydrostatic background stays exactly static), G2 (free fall: closed form),
//                          G3 (hydrostatic balance of PAPER.md:35 to 4th order), G4 (split == unsplit, 4th order)
// Round-2 pins (tests/test_oracle_pins_r2.py; each fails on the seeded mistake named in its docstring):
//   hd_mixed_fluxes, energy   M1 (uniform drift U: viscous R_e contains U * closed-form mixed R_mx; x<->y mirror),
//                             M2 (uniform B0: ohmic R_e contains B0 * closed-form mixed R_bx; mirror)
//   fill_ghosts during steps  F1 (fixed ghost strips incl. corners bitwise frozen while a pulse runs into them; the
//                             interior differs from the open run), F2 (frozen values == np.pad 'edge' of the set_state data)
//   flux / rhs (non-linear)   R1 (rhs of a flowing magnetised state == PAPER.md:35 differentiated analytically, order 4)
// "Parity unpinned" against the SAC/SMAUG codes themselves: the paper prints no field values and its
// figures are not in the container.
//
// Notation: interior cells i=0..nx-1 (x, fastest), j=0..ny-1; ghost width ng=3;
// perturbed state w=(rho~, mx, my, e~, bx~, by~); static background (rho_b, e_b, Bbx, Bby).

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int NG = 3;
enum { F_RHO = 0, F_MX = 1, F_MY = 2, F_E = 3, F_BX = 4, F_BY = 5, NF = 6 };
enum { BG_RHO = 0, BG_E = 1, BG_BX = 2, BG_BY = 3, NBG = 4 };
enum { BC_PERIODIC = 0, BC_OPEN = 1, BC_FIXED = 2 };
enum { SIDE_XLO = 0, SIDE_XHI = 1, SIDE_YLO = 2, SIDE_YHI = 3 };
enum {
  P_LX = 0, P_LY = 1, P_HD_ON = 2, P_C_RHO = 3, P_C_MOM = 4, P_C_E = 5, P_C_B = 6, P_RK_ORDER = 7,
  P_FIXED_DT = 8, P_GX = 10, P_GY = 11   // (9 is the CUDA library's kernel selector; unused here)
};
enum { OK = 0, EINVAL_ = -1, ENOMEM_ = -2, ECUDA_ = -3, ENONFINITE_ = -4 };

typedef std::vector<double> Plane;

struct Ctx {
  int nx, ny, NX, NY;
  double gamma;
  int bc[4];
  double Lx = 1.0, Ly = 1.0;
  int hd_on = 1;
  double c_rho = 0.02, c_mom = 0.4, c_e = 0.02, c_b = 0.02;
  int rk_order = 4;
  double fixed_dt = 0.0;
  double gx = 0.0, gy = 0.0;     // uniform gravitational acceleration g, c-10
  Plane bg[NBG];
  Plane w[NF];
  double t = 0.0, last_dt = 0.0;
  int nthreads = 1;
  double dx() const { return Lx / nx; }
  double dy() const { return Ly / ny; }
  size_t psize() const { return (size_t)NX * NY; }
  // padded index of cell (i,j); i in [-3,nx+3), j in [-3,ny+3)
  size_t at(int i, int j) const { return (size_t)(j + NG) * NX + (i + NG); }
};

thread_local std::string g_err;

// ---------------------------------------------------------------------------------------------
// c-8 ghost fill (PAPER.md:59 "halo layers", :101 "periodic at each boundary"; open/fixed: north_star).
// x first over interior rows, then y over the full padded width (this fills the corners).
// periodic: index modulo n (works for n < ng);  open: nearest interior cell;  fixed: left untouched
// (unless `freeze`, which writes the nearest interior cell once, at set_state time).
// ---------------------------------------------------------------------------------------------
int wrap(int i, int n) { return ((i % n) + n) % n; }

void fill_ghosts(const Ctx& c, Plane& p, bool freeze) {
  const int nx = c.nx, ny = c.ny;
  for (int j = 0; j < ny; ++j) {
    for (int g = 1; g <= NG; ++g) {
      int kind = c.bc[SIDE_XLO];
      if (kind == BC_PERIODIC) p[c.at(-g, j)] = p[c.at(wrap(-g, nx), j)];
      else if (kind == BC_OPEN || freeze) p[c.at(-g, j)] = p[c.at(0, j)];
      kind = c.bc[SIDE_XHI];
      if (kind == BC_PERIODIC) p[c.at(nx - 1 + g, j)] = p[c.at(wrap(nx - 1 + g, nx), j)];
      else if (kind == BC_OPEN || freeze) p[c.at(nx - 1 + g, j)] = p[c.at(nx - 1, j)];
    }
  }
  for (int i = -NG; i < nx + NG; ++i) {
    for (int g = 1; g <= NG; ++g) {
      int kind = c.bc[SIDE_YLO];
      if (kind == BC_PERIODIC) p[c.at(i, -g)] = p[c.at(i, wrap(-g, ny))];
      else if (kind == BC_OPEN || freeze) p[c.at(i, -g)] = p[c.at(i, 0)];
      kind = c.bc[SIDE_YHI];
      if (kind == BC_PERIODIC) p[c.at(i, ny - 1 + g)] = p[c.at(i, wrap(ny - 1 + g, ny))];
      else if (kind == BC_OPEN || freeze) p[c.at(i, ny - 1 + g)] = p[c.at(i, ny - 1)];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// ARITHMETIC CONTRACT.  The scheme's hyperviscosity ratio max|D3|/max|D1| is not
// smooth, and it amplifies rounding-level differences by ~6x per step for the first ~10 steps (measured:
// this file built with and without FMA contraction differs by 4e-8 after 40 steps on a 200^2
// Orszag-Tang run).  A 1e-10 parity bar after 50..1000 steps is therefore only reachable if both
// implementations evaluate every value with the SAME sequence of IEEE-754 operations.  So each formula
// below is written as an explicit operation sequence -- `fma(a,b,c)` is one correctly rounded a*b+c,
// every other +,-,*,/ and sqrt is one correctly rounded operation, evaluation order is as parenthesised
// -- and the file is compiled with -ffp-contract=off so the compiler adds no contraction of its own.
// The CUDA path implements the same sequences independently (built with -fmad=false).  Terms that are
// exactly zero for a zero background (x - 0, 0 + x, fma(0,y,0*z)) may be dropped without changing bits.
// ---------------------------------------------------------------------------------------------
using std::fma;

// ---------------------------------------------------------------------------------------------
// c-2 derived quantities on every padded cell (PAPER.md:39-43 with the SAC background split).
//   rho = rho_b + rho~,  v = m/rho (as m * (1/rho)),  B = B_b + b~
//   p~_k = (gamma-1)(e~ - rho v^2/2 - B_b.b~ - b~^2/2),  p~_t = p~_k + B_b.b~ + b~^2/2
//   eps~ = p~_k/(gamma-1)   (thermal-energy perturbation, the scalar the energy hyperdiffusion acts on)
// ---------------------------------------------------------------------------------------------
struct Derived {
  Plane rho, vx, vy, Bx, By, ptt, eps;
};

void derived(const Ctx& c, const Plane* w, Derived& d) {
  const size_t n = c.psize();
  const double gm1 = c.gamma - 1.0;
  for (Plane* p : {&d.rho, &d.vx, &d.vy, &d.Bx, &d.By, &d.ptt, &d.eps}) p->assign(n, 0.0);
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (long q = 0; q < (long)n; ++q) {
    const double rho = c.bg[BG_RHO][q] + w[F_RHO][q];
    const double rr = 1.0 / rho;
    const double mx = w[F_MX][q], my = w[F_MY][q];
    const double vx = mx * rr, vy = my * rr;
    const double bbx = c.bg[BG_BX][q], bby = c.bg[BG_BY][q];
    const double bx = w[F_BX][q], by = w[F_BY][q];
    const double b2h = 0.5 * fma(by, by, bx * bx);         // b~^2/2
    const double cross = fma(bby, by, bbx * bx);            // B_b . b~
    const double ke = 0.5 * fma(my, vy, mx * vx);           // rho v^2/2
    const double eps = ((w[F_E][q] - ke) - cross) - b2h;
    d.rho[q] = rho;
    d.vx[q] = vx;
    d.vy[q] = vy;
    d.Bx[q] = bbx + bx;
    d.By[q] = bby + by;
    d.eps[q] = eps;
    d.ptt[q] = fma(gm1, eps, cross + b2h);
  }
}

// c-3 fourth-order central difference, stride s = 1 (x) or NX (y):
//   cd12 = 12 * Delta * df/dx = 8 (f[+1] - f[-1]) - (f[+2] - f[-2]);   df/dx = cd12 * (1/Delta) * (1/12).
inline double cd12(const Plane& f, size_t q, size_t s) {
  return fma(8.0, f[q + s] - f[q - s], -(f[q + 2 * s] - f[q - 2 * s]));
}

// ---------------------------------------------------------------------------------------------
// c-2 fluxes of the split equations in direction dir (0 = x, 1 = y) at padded cell q.  With a zero
// background these are exactly the fluxes of PAPER.md:35 (mu0 = 1):
//   F_d(rho~) = rho v_d
//   F_d(m_l)  = m_l v_d - b~_l b~_d - b~_l B_b,d - B_b,l b~_d + delta_ld p~_t
//   F_d(e~)   = v_d (e~ + e_b + p~_t) - b~_d (b~.v) - b~_d (B_b.v) - B_b,d (b~.v)
//   F_d(b~_l) = v_d B_l - B_d v_l                     (total B; identically 0 for l = d)
// ---------------------------------------------------------------------------------------------
double flux(const Ctx& c, const Plane* w, const Derived& d, int field, int dir, size_t q) {
  const double v[2] = {d.vx[q], d.vy[q]};
  const double m[2] = {w[F_MX][q], w[F_MY][q]};
  const double bt[2] = {w[F_BX][q], w[F_BY][q]};             // b~
  const double Bb[2] = {c.bg[BG_BX][q], c.bg[BG_BY][q]};     // B_b
  const double B[2] = {d.Bx[q], d.By[q]};                    // total
  switch (field) {
    case F_RHO:
      return d.rho[q] * v[dir];
    case F_MX:
    case F_MY: {
      const int l = field - F_MX;
      const double f = (fma(m[l], v[dir], -(bt[l] * bt[dir])) - bt[l] * Bb[dir]) - Bb[l] * bt[dir];
      return l == dir ? f + d.ptt[q] : f;
    }
    case F_E: {
      const double btv = fma(bt[1], v[1], bt[0] * v[0]);     // b~ . v
      const double Bbv = fma(Bb[1], v[1], Bb[0] * v[0]);     // B_b . v
      const double h = (w[F_E][q] + c.bg[BG_E][q]) + d.ptt[q];
      return (fma(v[dir], h, -(bt[dir] * btv)) - bt[dir] * Bbv) - Bb[dir] * btv;
    }
    case F_BX:
    case F_BY: {
      const int l = field - F_BX;
      if (l == dir) return 0.0;
      return fma(v[dir], B[l], -(B[dir] * v[l]));
    }
  }
  return 0.0;
}

// ---------------------------------------------------------------------------------------------
// c-5 hyperviscosity coefficient ("the ratio of the forward difference of a parameter
// to third order and first order"; "require the estimation of maximum wave speed").
// For scalar u along direction dir, at interface k+1/2 (stored at the padded index of cell k):
//   D1_k = u_{k+1} - u_k,   D3_k = 3 (u_{k+1} - u_k) - (u_{k+2} - u_{k-1})
//   M3 = max |D3| over interfaces k-1, k, k+1;   M1 = max |D1| over interfaces k-2 .. k+2
//   nu_{k+1/2} = c_u * Delta * v_t * M3 / M1   if M1 > 0, else 0.
// Stored is kappa = nu / Delta = (c_u v_t) * (M3 / M1): every use of nu below is nu/Delta * (difference)
// or nu * (derivative), in which Delta cancels.  Valid (and computed) for k = -1 .. n-1 along dir and
// for every padded index across dir; other entries are 0.
// ---------------------------------------------------------------------------------------------
void hyper_kappa(const Ctx& c, const Plane& u, int dir, double cv, Plane& kap) {
  kap.assign(c.psize(), 0.0);
  const long s = dir == 0 ? 1 : c.NX;
  const int n_along = dir == 0 ? c.nx : c.ny;
  const int n_across = dir == 0 ? c.NY : c.NX;   // padded extent across dir
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int a = 0; a < n_across; ++a) {
    for (int k = -1; k <= n_along - 1; ++k) {
      const long q = dir == 0 ? (long)a * c.NX + (k + NG) : (long)(k + NG) * c.NX + a;
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
}

enum { K_RHO = 0, K_VX = 1, K_VY = 2, K_EPS = 3, K_B = 4, NK = 5 };
struct Kappas {
  Plane x[NK];   // along x, of rho~, vx, vy, eps~, by~
  Plane y[NK];   // along y, of rho~, vx, vy, eps~, bx~
};

// c-5 interface (diffusive) fluxes of all fields at the interface between cells a and b = a + s along
// dir, Phi = g * nu * (q_b - q_a)/Delta = g * kappa * (q_b - q_a):
//   rho~ : g = 1, q = rho~                     eps~ -> e : g = 1, q = eps~
//   m_l  : g = rho-bar (l = dir) or rho-bar/2 (l != dir), q = v_l      (tau_kl = rho/2 [nu_k d_k v_l + nu_l d_l v_k])
//   b~_l : g = 1, q = b~_l, only l != dir                              (eps_z = nu_x(by) d_x by - nu_y(bx) d_y bx)
//   e    : eps~ flux + vbar_x Phi(mx) + vbar_y Phi(my) + Bbar_l Phi(b_l)   (viscous work, ohmic coupling; total B)
// out[F_*]; out[F_B{dir}] = 0.
void hd_interface_fluxes(const Ctx& c, const Plane* w, const Derived& d, const Kappas& K, int dir, long a,
                         double out[NF]) {
  const long s = dir == 0 ? 1 : c.NX, b = a + s;
  const Plane* kap = dir == 0 ? K.x : K.y;
  const int lt = 1 - dir;                                    // the transverse magnetic component
  const Plane& bq = w[F_BX + lt];
  const Plane& Bq = lt == 0 ? d.Bx : d.By;
  const double rbar = 0.5 * (d.rho[a] + d.rho[b]);
  const double g_mx = dir == 0 ? rbar : 0.5 * rbar;
  const double g_my = dir == 1 ? rbar : 0.5 * rbar;
  const double p_rho = kap[K_RHO][a] * (w[F_RHO][b] - w[F_RHO][a]);
  const double p_mx = (g_mx * kap[K_VX][a]) * (d.vx[b] - d.vx[a]);
  const double p_my = (g_my * kap[K_VY][a]) * (d.vy[b] - d.vy[a]);
  const double p_eps = kap[K_EPS][a] * (d.eps[b] - d.eps[a]);
  const double p_b = kap[K_B][a] * (bq[b] - bq[a]);
  const double vxbar = 0.5 * (d.vx[a] + d.vx[b]);
  const double vybar = 0.5 * (d.vy[a] + d.vy[b]);
  const double Bbar = 0.5 * (Bq[a] + Bq[b]);
  out[F_RHO] = p_rho;
  out[F_MX] = p_mx;
  out[F_MY] = p_my;
  out[F_E] = fma(Bbar, p_b, fma(vybar, p_my, fma(vxbar, p_mx, p_eps)));
  out[F_BX + lt] = p_b;
  out[F_BX + dir] = 0.0;
}

// c-5 mixed (cross) terms: cell-centred fluxes along direction k built from derivatives along l != k,
//   G(m_l ; k) = (rho/2) nubar_l(v_k) d^c_l v_k       G(b_l ; k) = - nubar_l(b~_k) d^c_l b~_k
//   G(e ; k)   = v_l G(m_l;k) + B_l G(b_l;k)           nubar_l = (nu_{l-1/2} + nu_{l+1/2})/2, d^c = c-3
// [note the roles: the flux of m_l along k uses the coefficient and derivative ALONG l of the k-component].
// They enter the RHS as + d^c_k G, i.e. they are subtracted from F_k before the central difference.
// Defined on cells interior along l and [-2, n+2) along k; G planes are 0 elsewhere.  Gk[F_*].
void hd_mixed_fluxes(const Ctx& c, const Plane* w, const Derived& d, const Kappas& K, int k, Plane* G) {
  for (int f = 0; f < NF; ++f) G[f].assign(c.psize(), 0.0);
  const int l = 1 - k;
  const long sl = l == 0 ? 1 : c.NX;
  const Plane* kap = l == 0 ? K.x : K.y;             // coefficients along l
  const Plane& vk = k == 0 ? d.vx : d.vy;            // k-component of v  (kappa family K_VX + k)
  const Plane& bk = w[F_BX + k];                     // k-component of b~ (kappa family K_B along l)
  const Plane& vl = l == 0 ? d.vx : d.vy;
  const Plane& Bl = l == 0 ? d.Bx : d.By;
  const int lo_i = (k == 0) ? -2 : 0, hi_i = (k == 0) ? c.nx + 2 : c.nx;
  const int lo_j = (k == 1) ? -2 : 0, hi_j = (k == 1) ? c.ny + 2 : c.ny;
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int j = lo_j; j < hi_j; ++j)
    for (int i = lo_i; i < hi_i; ++i) {
      const long q = (long)c.at(i, j);
      const double kbar_v = 0.5 * (kap[K_VX + k][q - sl] + kap[K_VX + k][q]);
      const double kbar_b = 0.5 * (kap[K_B][q - sl] + kap[K_B][q]);
      const double dv = cd12(vk, (size_t)q, (size_t)sl) * (1.0 / 12.0);
      const double db = cd12(bk, (size_t)q, (size_t)sl) * (1.0 / 12.0);
      const double gm = ((0.5 * d.rho[q]) * kbar_v) * dv;
      const double gb = -(kbar_b * db);
      G[F_MX + l][q] = gm;
      G[F_BX + l][q] = gb;
      G[F_E][q] = fma(vl[q], gm, Bl[q] * gb);
    }
}

// c-4 maxima over interior cells of the state w:
//   a^2 = gamma p_k / rho with total p_k = (gamma-1)(e - rho v^2/2 - B^2/2), e = e_b + e~;  b^2 = B^2/rho
//   c_f,d^2 = ( a^2+b^2 + sqrt(max(0, (a^2+b^2)^2 - 4 a^2 B_d^2/rho)) ) / 2
//   out = { max(|vx|+c_f,x), max(|vy|+c_f,y), max a^2, max b^2 };  maxima start at 0, NaNs are skipped.
void wavespeeds(const Ctx& c, const Plane* w, double out[4]) {
  double m0 = 0, m1 = 0, m2 = 0, m3 = 0;
  const double gm1 = c.gamma - 1.0;
#pragma omp parallel for num_threads(c.nthreads) schedule(static) reduction(max : m0, m1, m2, m3)
  for (int j = 0; j < c.ny; ++j)
    for (int i = 0; i < c.nx; ++i) {
      const size_t q = c.at(i, j);
      const double rho = c.bg[BG_RHO][q] + w[F_RHO][q];
      const double rr = 1.0 / rho;
      const double mx = w[F_MX][q], my = w[F_MY][q];
      const double vx = mx * rr, vy = my * rr;
      const double Bx = c.bg[BG_BX][q] + w[F_BX][q], By = c.bg[BG_BY][q] + w[F_BY][q];
      const double e = c.bg[BG_E][q] + w[F_E][q];
      const double B2 = fma(By, By, Bx * Bx);
      const double pk = gm1 * ((e - 0.5 * fma(my, vy, mx * vx)) - 0.5 * B2);
      const double a2 = (c.gamma * pk) * rr;
      const double b2 = B2 * rr;
      const double s = a2 + b2;
      const double fa = (4.0 * a2) * rr;
      const double cfx2 = 0.5 * (s + std::sqrt(std::max(0.0, fma(s, s, -(fa * (Bx * Bx))))));
      const double cfy2 = 0.5 * (s + std::sqrt(std::max(0.0, fma(s, s, -(fa * (By * By))))));
      const double cx = std::fabs(vx) + std::sqrt(cfx2);
      const double cy = std::fabs(vy) + std::sqrt(cfy2);
      if (cx > m0) m0 = cx;
      if (cy > m1) m1 = cy;
      if (a2 > m2) m2 = a2;
      if (b2 > m3) m3 = b2;
    }
  out[0] = m0; out[1] = m1; out[2] = m2; out[3] = m3;
}

// c-6: R(w) = -sum_d d^c_d (F_d - G_d) + S + sum_d (Phi_{d,+} - Phi_{d,-})/Delta_d; ghosts of w must be
// filled.  v_t = sqrt(max a^2) + sqrt(max b^2) of the state being differentiated (c-5).
void rhs(const Ctx& c, const Plane* w, Plane* R) {
  const size_t n = c.psize();
  const double inv_dx = c.nx / c.Lx, inv_dy = c.ny / c.Ly;
  Derived d;
  derived(c, w, d);
  Kappas K;
  Plane Gx[NF], Gy[NF];
  for (int f = 0; f < NF; ++f) { Gx[f].assign(n, 0.0); Gy[f].assign(n, 0.0); }
  if (c.hd_on) {
    double ws[4];
    wavespeeds(c, w, ws);
    const double vt = std::sqrt(ws[2]) + std::sqrt(ws[3]);
    const double cv_rho = c.c_rho * vt, cv_mom = c.c_mom * vt, cv_e = c.c_e * vt, cv_b = c.c_b * vt;
    hyper_kappa(c, w[F_RHO], 0, cv_rho, K.x[K_RHO]);  hyper_kappa(c, w[F_RHO], 1, cv_rho, K.y[K_RHO]);
    hyper_kappa(c, d.vx, 0, cv_mom, K.x[K_VX]);       hyper_kappa(c, d.vx, 1, cv_mom, K.y[K_VX]);
    hyper_kappa(c, d.vy, 0, cv_mom, K.x[K_VY]);       hyper_kappa(c, d.vy, 1, cv_mom, K.y[K_VY]);
    hyper_kappa(c, d.eps, 0, cv_e, K.x[K_EPS]);       hyper_kappa(c, d.eps, 1, cv_e, K.y[K_EPS]);
    hyper_kappa(c, w[F_BY], 0, cv_b, K.x[K_B]);       hyper_kappa(c, w[F_BX], 1, cv_b, K.y[K_B]);
    hd_mixed_fluxes(c, w, d, K, 0, Gx);
    hd_mixed_fluxes(c, w, d, K, 1, Gy);
  }
  // flux divergence of C_d = F_d - G_d, fourth-order central (c-3)
  Plane Cx(n), Cy(n);
  for (int f = 0; f < NF; ++f) {
    R[f].assign(n, 0.0);
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
    for (long q = 0; q < (long)n; ++q) {
      Cx[q] = flux(c, w, d, f, 0, (size_t)q) - Gx[f][q];
      Cy[q] = flux(c, w, d, f, 1, (size_t)q) - Gy[f][q];
    }
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
    for (int j = 0; j < c.ny; ++j)
      for (int i = 0; i < c.nx; ++i) {
        const size_t q = c.at(i, j);
        R[f][q] = fma(cd12(Cx, q, 1), inv_dx, cd12(Cy, q, (size_t)c.NX) * inv_dy) * (-1.0 / 12.0);
      }
  }
  // c-2 energy source (zero when the background is zero; gravity: c-10 below):
  //   S_e = -p_tb (dvx/dx + dvy/dy) + sum_{k,l} B_b,k B_b,l d_k v_l,  p_tb = (gamma-1)(e_b - B_b^2/2) + B_b^2/2
  const double gm1 = c.gamma - 1.0;
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int j = 0; j < c.ny; ++j)
    for (int i = 0; i < c.nx; ++i) {
      const size_t q = c.at(i, j);
      const double bbx = c.bg[BG_BX][q], bby = c.bg[BG_BY][q];
      const double bb2h = 0.5 * fma(bby, bby, bbx * bbx);
      const double ptb = fma(gm1, c.bg[BG_E][q] - bb2h, bb2h);
      const double dxvx = (cd12(d.vx, q, 1) * inv_dx) * (1.0 / 12.0);
      const double dyvx = (cd12(d.vx, q, (size_t)c.NX) * inv_dy) * (1.0 / 12.0);
      const double dxvy = (cd12(d.vy, q, 1) * inv_dx) * (1.0 / 12.0);
      const double dyvy = (cd12(d.vy, q, (size_t)c.NX) * inv_dy) * (1.0 / 12.0);
      const double S = fma(-ptb, dxvx + dyvy,
                           fma(bby * bby, dyvy, fma(bbx * bby, dxvy + dyvx, (bbx * bbx) * dxvx)));
      R[F_E][q] = R[F_E][q] + S;
    }
  // c-10 gravity ("rho g" in the momentum equation, "rho g.v" in the energy equation), in the
  // split form: the background is taken to be in magneto-hydrostatic balance,
  //   grad p_tb - (B_b.grad) B_b = rho_b g,
  // so the background part of "rho g" cancels the background pressure gradient and the background part of
  // "rho g.v" cancels v.grad p_tb (which is how S_e above arises); what is left acts on the PERTURBED density:
  //   S(m) = rho~ g,   S(e~) = rho~ (g.v)        [g uniform; with a zero background rho~ = rho: PAPER.md:35 as printed]
  // Applied only when g != 0 (fma(x, 0, -0.0) would turn a -0 into +0).
  if (c.gx != 0.0 || c.gy != 0.0) {
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
    for (int j = 0; j < c.ny; ++j)
      for (int i = 0; i < c.nx; ++i) {
        const size_t q = c.at(i, j);
        const double rt = w[F_RHO][q];
        R[F_MX][q] = fma(rt, c.gx, R[F_MX][q]);
        R[F_MY][q] = fma(rt, c.gy, R[F_MY][q]);
        R[F_E][q] = fma(rt, fma(c.gy, d.vy[q], c.gx * d.vx[q]), R[F_E][q]);
      }
  }
  // c-5 interface fluxes, x then y
  if (c.hd_on) {
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
    for (int j = 0; j < c.ny; ++j)
      for (int i = 0; i < c.nx; ++i) {
        const long q = (long)c.at(i, j);
        double lo[NF], hi[NF];
        hd_interface_fluxes(c, w, d, K, 0, q - 1, lo);
        hd_interface_fluxes(c, w, d, K, 0, q, hi);
        for (int f = 0; f < NF; ++f) R[f][q] = fma(hi[f] - lo[f], inv_dx, R[f][q]);
        hd_interface_fluxes(c, w, d, K, 1, q - c.NX, lo);
        hd_interface_fluxes(c, w, d, K, 1, q, hi);
        for (int f = 0; f < NF; ++f) R[f][q] = fma(hi[f] - lo[f], inv_dy, R[f][q]);
      }
  }
}

// c-7: dt = cfl * min_d (Delta_d / cmax_d); an axis with n = 1 is excluded.
double cfl_dt(const Ctx& c, const Plane* w, double cfl) {
  double ws[4];
  wavespeeds(c, w, ws);
  double m = INFINITY;
  if (c.nx > 1) m = std::min(m, (c.Lx / c.nx) / ws[0]);
  if (c.ny > 1) m = std::min(m, (c.Ly / c.ny) / ws[1]);
  return cfl * m;
}

// A stage state: interior from `interior`, ghosts copied from wn (keeps frozen "fixed" ghosts), then
// refilled on periodic/open sides.
void finish_stage(const Ctx& c, const Plane* wn, Plane* ws) {
  for (int f = 0; f < NF; ++f) {
    for (int j = -NG; j < c.ny + NG; ++j)
      for (int i = -NG; i < c.nx + NG; ++i)
        if (i < 0 || i >= c.nx || j < 0 || j >= c.ny) ws[f][c.at(i, j)] = wn[f][c.at(i, j)];
    fill_ghosts(c, ws[f], false);
  }
}

// c-6 one step of the classical fourth-order Runge-Kutta scheme, dt frozen over the step,
// written in stage-state form (algebraically the classical update w^{n+1} = w^n + dt/6 (k1+2k2+2k3+k4),
// since k1 = 2(w1-w^n)/dt, k2 = 2(w2-w^n)/dt, k3 = (w3-w^n)/dt):
//   w1 = w^n + (dt/2) R(w^n),  w2 = w^n + (dt/2) R(w1),  w3 = w^n + dt R(w2),
//   acc = (w1 - w^n) + 2 w2,   w^{n+1} = w3 + (acc - 2 w3)/3 + (dt/6) R(w3)      [= (w1+2w2+w3-w^n)/3 + dt/6 k4;
//   this grouping returns w^n bit for bit when every R is 0, pin P1].
// rk_order 2 = midpoint (w1 as above, w^{n+1} = w^n + dt R(w1)), 1 = forward Euler.
void rk_step(Ctx& c, double dt) {
  const size_t n = c.psize();
  Plane R[NF], w1[NF], w2[NF], w3[NF], wnew[NF];
  Plane* wn = c.w;
  auto axpy = [&](double a, Plane* out) {           // out = w^n + a R on interior cells
    for (int f = 0; f < NF; ++f) {
      out[f].assign(n, 0.0);
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) {
          const size_t q = c.at(i, j);
          out[f][q] = fma(a, R[f][q], wn[f][q]);
        }
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
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) {
          const size_t q = c.at(i, j);
          const double acc = fma(2.0, w2[f][q], w1[f][q] - wn[f][q]);
          wnew[f][q] = fma(dt6, R[f][q], fma(fma(-2.0, w3[f][q], acc), 1.0 / 3.0, w3[f][q]));
        }
    }
    finish_stage(c, wn, wnew);
  }
  for (int f = 0; f < NF; ++f) c.w[f].swap(wnew[f]);
  c.t += dt;
  c.last_dt = dt;
}

}  // namespace

// =============================================================================================
// C ABI.  Same shape as include/smaug.h so that one harness drives both, plus
// a few entry points that expose the pieces to the pin tests.  Host pointers only.
// State / background layout: [field][ny][nx], x fastest, interior only, fp64.
// =============================================================================================
typedef struct oracle_ctx oracle_ctx;
#define CTX(p) (reinterpret_cast<Ctx*>(p))

extern "C" {

const char* oracle_last_error(void) { return g_err.c_str(); }

int oracle_create(int nx, int ny, double gamma, const int bc[4], const double* bg, oracle_ctx** out) {
  if (!out || !bc) { g_err = "NULL argument"; return EINVAL_; }
  *out = nullptr;
  if (nx < 1 || ny < 1) { g_err = "nx, ny must be >= 1"; return EINVAL_; }
  if (!(gamma > 1.0)) { g_err = "gamma must be > 1"; return EINVAL_; }
  for (int s = 0; s < 4; ++s)
    if (bc[s] < 0 || bc[s] > 2) { g_err = "unknown boundary kind"; return EINVAL_; }
  for (int a = 0; a < 2; ++a)
    if ((bc[2 * a] == BC_PERIODIC) != (bc[2 * a + 1] == BC_PERIODIC)) {
      g_err = "periodic must be set on both sides of an axis";
      return EINVAL_;
    }
  Ctx* c = new Ctx();
  c->nx = nx; c->ny = ny; c->NX = nx + 2 * NG; c->NY = ny + 2 * NG; c->gamma = gamma;
  for (int s = 0; s < 4; ++s) c->bc[s] = bc[s];
  for (int b = 0; b < NBG; ++b) {
    c->bg[b].assign(c->psize(), 0.0);
    if (bg) {
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) c->bg[b][c->at(i, j)] = bg[((size_t)b * ny + j) * nx + i];
      fill_ghosts(*c, c->bg[b], true);   // c-8: periodic -> wrap, else edge copy, once
    }
  }
  for (int f = 0; f < NF; ++f) c->w[f].assign(c->psize(), 0.0);
  *out = reinterpret_cast<oracle_ctx*>(c);
  return OK;
}

void oracle_destroy(oracle_ctx* p) { delete CTX(p); }

int oracle_set_param(oracle_ctx* p, int key, double v) {
  if (!p) { g_err = "NULL ctx"; return EINVAL_; }
  Ctx& c = *CTX(p);
  switch (key) {
    case P_LX: if (!(v > 0)) break; c.Lx = v; return OK;
    case P_LY: if (!(v > 0)) break; c.Ly = v; return OK;
    case P_HD_ON: c.hd_on = v != 0.0; return OK;
    case P_C_RHO: if (!(v >= 0)) break; c.c_rho = v; return OK;
    case P_C_MOM: if (!(v >= 0)) break; c.c_mom = v; return OK;
    case P_C_E: if (!(v >= 0)) break; c.c_e = v; return OK;
    case P_C_B: if (!(v >= 0)) break; c.c_b = v; return OK;
    case P_RK_ORDER: if (v != 1 && v != 2 && v != 4) break; c.rk_order = (int)v; return OK;
    case P_FIXED_DT: if (!(v >= 0)) break; c.fixed_dt = v; return OK;
    case P_GX: if (!std::isfinite(v)) break; c.gx = v; return OK;
    case P_GY: if (!std::isfinite(v)) break; c.gy = v; return OK;
    default: g_err = "unknown parameter key"; return EINVAL_;
  }
  g_err = "parameter value out of range";
  return EINVAL_;
}

int oracle_set_threads(oracle_ctx* p, int n) {   // result-neutral OpenMP over rows (no sum reductions)
  if (!p || n < 1) { g_err = "bad argument"; return EINVAL_; }
  CTX(p)->nthreads = n;
  return OK;
}

int oracle_set_state(oracle_ctx* p, const double* w) {
  if (!p || !w) { g_err = "NULL argument"; return EINVAL_; }
  Ctx& c = *CTX(p);
  for (int f = 0; f < NF; ++f) {
    for (int j = 0; j < c.ny; ++j)
      for (int i = 0; i < c.nx; ++i) c.w[f][c.at(i, j)] = w[((size_t)f * c.ny + j) * c.nx + i];
    fill_ghosts(c, c.w[f], true);        // fixed sides: frozen here at the nearest interior value
  }
  c.t = 0.0; c.last_dt = 0.0;
  return OK;
}

int oracle_get_state(oracle_ctx* p, double* w) {
  if (!p || !w) { g_err = "NULL argument"; return EINVAL_; }
  Ctx& c = *CTX(p);
  for (int f = 0; f < NF; ++f)
    for (int j = 0; j < c.ny; ++j)
      for (int i = 0; i < c.nx; ++i) w[((size_t)f * c.ny + j) * c.nx + i] = c.w[f][c.at(i, j)];
  return OK;
}

int oracle_get_time(oracle_ctx* p, double* t, double* last_dt) {
  if (!p) { g_err = "NULL ctx"; return EINVAL_; }
  if (t) *t = CTX(p)->t;
  if (last_dt) *last_dt = CTX(p)->last_dt;
  return OK;
}

int oracle_step(oracle_ctx* p, int n_steps, double cfl) {
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

// ---- pieces, for the pin tests ------------------------------------------------------------------
// R(w) of the current state, [6][ny][nx].
int oracle_rhs(oracle_ctx* p, double* R) {
  if (!p || !R) { g_err = "NULL argument"; return EINVAL_; }
  Ctx& c = *CTX(p);
  Plane k[NF];
  for (int f = 0; f < NF; ++f) fill_ghosts(c, c.w[f], false);
  rhs(c, c.w, k);
  for (int f = 0; f < NF; ++f)
    for (int j = 0; j < c.ny; ++j)
      for (int i = 0; i < c.nx; ++i) R[((size_t)f * c.ny + j) * c.nx + i] = k[f][c.at(i, j)];
  return OK;
}

// out = { cmax_x, cmax_y, max a^2, max b^2 } of the current state (c-4).
int oracle_wavespeeds(oracle_ctx* p, double out[4]) {
  if (!p || !out) { g_err = "NULL argument"; return EINVAL_; }
  wavespeeds(*CTX(p), CTX(p)->w, out);
  return OK;
}

// The padded plane of field f (rows of nx+6, ny+6 rows), ghosts as they currently are.
int oracle_get_padded(oracle_ctx* p, int f, double* out) {
  if (!p || !out || f < 0 || f >= NF) { g_err = "bad argument"; return EINVAL_; }
  std::memcpy(out, CTX(p)->w[f].data(), CTX(p)->psize() * sizeof(double));
  return OK;
}

// c-5 coefficient on a 1-D line: u has n+6 entries (3 ghosts each side, already filled);
// nu_out has n+1 entries, the interfaces -1/2 .. n-1/2.
int oracle_hyper_nu_1d(const double* u, int n, double coef, double delta, double vt, double* nu_out) {
  if (!u || !nu_out || n < 1) { g_err = "bad argument"; return EINVAL_; }
  const int bc[4] = {BC_OPEN, BC_OPEN, BC_PERIODIC, BC_PERIODIC};
  oracle_ctx* h = nullptr;
  int rc = oracle_create(n, 1, 2.0, bc, nullptr, &h);
  if (rc) return rc;
  Ctx& c = *CTX(h);
  c.Lx = delta * n;
  Plane up(c.psize(), 0.0), kap;
  for (int j = -NG; j < 1 + NG; ++j)
    for (int i = -NG; i < n + NG; ++i) up[c.at(i, j)] = u[i + NG];
  hyper_kappa(c, up, 0, coef * vt, kap);
  for (int k = -1; k <= n - 1; ++k) nu_out[k + 1] = kap[c.at(k, 0)] * delta;   // nu = kappa * Delta
  oracle_destroy(h);
  return OK;
}

// c-3 on a 1-D line: f has n+4 entries (2 extra each side); out has n entries.
int oracle_central_diff_1d(const double* f, int n, double h, double* out) {
  if (!f || !out || n < 1) { g_err = "bad argument"; return EINVAL_; }
  Plane fp(f, f + n + 4);
  for (int i = 0; i < n; ++i) out[i] = (cd12(fp, (size_t)i + 2, 1) * (1.0 / h)) * (1.0 / 12.0);
  return OK;
}

}  // extern "C"
