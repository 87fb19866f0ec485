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
//   hyper_nu               P8 (unit-step worked example 1,2,2,2,1), P9 (closed form on a sine), P10 (bound 4)
//   hyper_div              P1, P2 (conservation incl. energy couplings), P3, P5 (x<->y transposition)
//   wavespeeds / dt        P11 (closed-form Brio-Wu and Orszag-Tang maxima and dt0)
//   rk4_step               P6 (temporal order 4), P4 (RK4 amplification factor), P12 (restart)
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
  P_FIXED_DT = 8
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
// c-2 derived quantities on every padded cell (PAPER.md:39-43 with the SAC background split).
//   rho = rho_b + rho~,  v = m/rho,  B = B_b + b~
//   p~_k = (gamma-1)(e~ - rho v^2/2 - B_b.b~ - b~^2/2),  p~_t = p~_k + B_b.b~ + b~^2/2
//   eps~ = p~_k/(gamma-1)   (thermal-energy perturbation, the scalar the energy hyperdiffusion acts on)
// ---------------------------------------------------------------------------------------------
struct Derived {
  Plane rho, vx, vy, Bx, By, ptt, eps;
};

void derived(const Ctx& c, const Plane* w, Derived& d) {
  const size_t n = c.psize();
  for (Plane* p : {&d.rho, &d.vx, &d.vy, &d.Bx, &d.By, &d.ptt, &d.eps}) p->assign(n, 0.0);
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (long q = 0; q < (long)n; ++q) {
    const double rho = c.bg[BG_RHO][q] + w[F_RHO][q];
    const double vx = w[F_MX][q] / rho;
    const double vy = w[F_MY][q] / rho;
    const double bbx = c.bg[BG_BX][q], bby = c.bg[BG_BY][q];
    const double bx = w[F_BX][q], by = w[F_BY][q];
    const double cross = bbx * bx + bby * by;        // B_b . b~
    const double b2h = 0.5 * (bx * bx + by * by);    // b~^2/2
    const double eps = w[F_E][q] - 0.5 * rho * (vx * vx + vy * vy) - cross - b2h;
    d.rho[q] = rho;
    d.vx[q] = vx;
    d.vy[q] = vy;
    d.Bx[q] = bbx + bx;
    d.By[q] = bby + by;
    d.eps[q] = eps;
    d.ptt[q] = (c.gamma - 1.0) * eps + cross + b2h;
  }
}

// c-3 fourth-order central difference, stride s = 1 (x) or NX (y), spacing h.
inline double cdiff(const Plane& f, size_t q, size_t s, double h) {
  return (8.0 * (f[q + s] - f[q - s]) - (f[q + 2 * s] - f[q - 2 * s])) / (12.0 * h);
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
      double f = m[l] * v[dir] - bt[l] * bt[dir] - bt[l] * Bb[dir] - Bb[l] * bt[dir];
      if (l == dir) f += d.ptt[q];
      return f;
    }
    case F_E: {
      const double btv = bt[0] * v[0] + bt[1] * v[1];        // b~ . v
      const double Bbv = Bb[0] * v[0] + Bb[1] * v[1];        // B_b . v
      return v[dir] * (w[F_E][q] + c.bg[BG_E][q] + d.ptt[q]) - bt[dir] * btv - bt[dir] * Bbv -
             Bb[dir] * btv;
    }
    case F_BX:
    case F_BY: {
      const int l = field - F_BX;
      if (l == dir) return 0.0;
      return v[dir] * B[l] - B[dir] * v[l];
    }
  }
  return 0.0;
}

// R_f -= d/dx F_x(f) + d/dy F_y(f) on interior cells; R planes are padded, interior entries used.
void flux_div(const Ctx& c, const Plane* w, const Derived& d, Plane* R) {
  const size_t n = c.psize();
  Plane F(n);
  for (int field = 0; field < NF; ++field) {
    for (int dir = 0; dir < 2; ++dir) {
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
      for (long q = 0; q < (long)n; ++q) F[q] = flux(c, w, d, field, dir, (size_t)q);
      const size_t s = dir == 0 ? 1 : (size_t)c.NX;
      const double h = dir == 0 ? c.dx() : c.dy();
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) {
          const size_t q = c.at(i, j);
          R[field][q] -= cdiff(F, q, s, h);
        }
    }
  }
}

// c-2 energy source (zero when the background is zero; gravity absent):
//   S_e = -p_tb (dvx/dx + dvy/dy) + sum_{k,l} B_b,k B_b,l d_k v_l,
//   p_tb = (gamma-1)(e_b - B_b^2/2) + B_b^2/2.
void sources(const Ctx& c, const Derived& d, Plane* R) {
  const size_t sx = 1, sy = (size_t)c.NX;
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int j = 0; j < c.ny; ++j)
    for (int i = 0; i < c.nx; ++i) {
      const size_t q = c.at(i, j);
      const double bbx = c.bg[BG_BX][q], bby = c.bg[BG_BY][q];
      const double bb2h = 0.5 * (bbx * bbx + bby * bby);
      const double ptb = (c.gamma - 1.0) * (c.bg[BG_E][q] - bb2h) + bb2h;
      const double dxvx = cdiff(d.vx, q, sx, c.dx()), dyvx = cdiff(d.vx, q, sy, c.dy());
      const double dxvy = cdiff(d.vy, q, sx, c.dx()), dyvy = cdiff(d.vy, q, sy, c.dy());
      R[F_E][q] += -ptb * (dxvx + dyvy) +
                   (bbx * bbx * dxvx + bbx * bby * dxvy + bby * bbx * dyvx + bby * bby * dyvy);
    }
}

// ---------------------------------------------------------------------------------------------
// c-5 hyperviscosity coefficient ("the ratio of the forward difference of a parameter
// to third order and first order"; "require the estimation of maximum wave speed").
// For scalar u along direction dir, at interface k+1/2 (stored at the padded index of cell k):
//   D1_k = u_{k+1} - u_k,   D3_k = 3 (u_{k+1} - u_k) - (u_{k+2} - u_{k-1})
//   M3 = max |D3| over interfaces k-1, k, k+1;   M1 = max |D1| over interfaces k-2 .. k+2
//   nu_{k+1/2} = coef * Delta * v_t * M3 / M1   if M1 > 0, else 0.
// Valid (and computed) for k = -1 .. n-1 along dir and for every padded index across dir; other
// entries are 0.
// ---------------------------------------------------------------------------------------------
void hyper_nu(const Ctx& c, const Plane& u, int dir, double coef, double vt, Plane& nu) {
  nu.assign(c.psize(), 0.0);
  const long s = dir == 0 ? 1 : c.NX;
  const double delta = dir == 0 ? c.dx() : c.dy();
  const int n_along = dir == 0 ? c.nx : c.ny;
  const int n_across = dir == 0 ? c.NY : c.NX;   // padded extent across dir
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int a = 0; a < n_across; ++a) {
    for (int k = -1; k <= n_along - 1; ++k) {
      const long q = dir == 0 ? (long)a * c.NX + (k + NG) : (long)(k + NG) * c.NX + a;
      double M3 = 0.0, M1 = 0.0;
      for (int o = -1; o <= 1; ++o) {
        const long r = q + o * s;
        const double d3 = 3.0 * (u[r + s] - u[r]) - (u[r + 2 * s] - u[r - s]);
        M3 = std::max(M3, std::fabs(d3));
      }
      for (int o = -2; o <= 2; ++o) {
        const long r = q + o * s;
        M1 = std::max(M1, std::fabs(u[r + s] - u[r]));
      }
      nu[q] = M1 > 0.0 ? coef * delta * vt * (M3 / M1) : 0.0;
    }
  }
}

// Interface operator of c-5, direction dir, added to R on interior cells:
//   Phi_{k+1/2} = g_{k+1/2} * nu_{k+1/2} * (qv_{k+1} - qv_k)/Delta * fac
//   R    += (Phi_{k+1/2} - Phi_{k-1/2}) / Delta
//   R_e  += (cj_{k+1/2} Phi_{k+1/2} - cj_{k-1/2} Phi_{k-1/2}) / Delta   (if conj != nullptr)
// g = 1 (gw == nullptr) or the interface average (gw_k + gw_{k+1})/2; cj_{k+1/2} is the interface
// average of the conjugate factor (v_l for a momentum flux, total B_l for a magnetic flux).
void hyper_interface(const Ctx& c, const Plane& nu, const Plane& qv, const Plane* gw, double fac,
                     int dir, Plane& R, const Plane* conj, Plane* Re) {
  const long s = dir == 0 ? 1 : c.NX;
  const double delta = dir == 0 ? c.dx() : c.dy();
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int j = 0; j < c.ny; ++j)
    for (int i = 0; i < c.nx; ++i) {
      const long q = (long)c.at(i, j);
      double phi[2], cj[2];
      for (int side = 0; side < 2; ++side) {
        const long a = q + (side - 1) * s, b = a + s;   // interface between cells a and b
        const double g = gw ? 0.5 * ((*gw)[a] + (*gw)[b]) : 1.0;
        phi[side] = g * nu[a] * (qv[b] - qv[a]) / delta * fac;
        cj[side] = conj ? 0.5 * ((*conj)[a] + (*conj)[b]) : 0.0;
      }
      R[q] += (phi[1] - phi[0]) / delta;
      if (conj) (*Re)[q] += (cj[1] * phi[1] - cj[0] * phi[0]) / delta;
    }
}

// Mixed (cross) term of c-5: cell-centred flux along direction k built from a derivative along l != k,
//   G = fac * gw * nubar_l(u) * d^c_l qv,   nubar_l = (nu_{l-1/2} + nu_{l+1/2})/2,   d^c = c-3,
//   R   += d^c_k G,    R_e += d^c_k (conj * G)     (conj cell-centred).
// G is needed at cells +-1, +-2 along k (ghost cells there), interior along l.
void hyper_mixed(const Ctx& c, const Plane& nu_l, const Plane& qv, const Plane* gw, double fac, int l,
                 Plane& R, const Plane& conj, Plane& Re) {
  const int k = 1 - l;
  const long sl = l == 0 ? 1 : c.NX, sk = k == 0 ? 1 : c.NX;
  const double hl = l == 0 ? c.dx() : c.dy(), hk = k == 0 ? c.dx() : c.dy();
  Plane G(c.psize(), 0.0), GE(c.psize(), 0.0);
  // cells: interior along l, [-2, n+2) along k
  const int lo_i = (k == 0) ? -2 : 0, hi_i = (k == 0) ? c.nx + 2 : c.nx;
  const int lo_j = (k == 1) ? -2 : 0, hi_j = (k == 1) ? c.ny + 2 : c.ny;
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int j = lo_j; j < hi_j; ++j)
    for (int i = lo_i; i < hi_i; ++i) {
      const long q = (long)c.at(i, j);
      const double nubar = 0.5 * (nu_l[q - sl] + nu_l[q]);
      const double g = gw ? (*gw)[q] : 1.0;
      G[q] = fac * g * nubar * cdiff(qv, (size_t)q, (size_t)sl, hl);
      GE[q] = conj[q] * G[q];
    }
#pragma omp parallel for num_threads(c.nthreads) schedule(static)
  for (int j = 0; j < c.ny; ++j)
    for (int i = 0; i < c.nx; ++i) {
      const size_t q = c.at(i, j);
      R[q] += cdiff(G, q, (size_t)sk, hk);
      Re[q] += cdiff(GE, q, (size_t)sk, hk);
    }
}

// c-4 maxima over interior cells of the (ghost-filled or not: interior only) state w:
//   a^2 = gamma p_k / rho with total p_k = (gamma-1)(e - rho v^2/2 - B^2/2), e = e_b + e~;  b^2 = B^2/rho
//   c_f,d^2 = ( a^2+b^2 + sqrt(max(0, (a^2+b^2)^2 - 4 a^2 B_d^2/rho)) ) / 2
//   out = { max(|vx|+c_f,x), max(|vy|+c_f,y), max a^2, max b^2 };  maxima start at 0, NaNs are skipped.
void wavespeeds(const Ctx& c, const Plane* w, double out[4]) {
  double m0 = 0, m1 = 0, m2 = 0, m3 = 0;
#pragma omp parallel for num_threads(c.nthreads) schedule(static) reduction(max : m0, m1, m2, m3)
  for (int j = 0; j < c.ny; ++j)
    for (int i = 0; i < c.nx; ++i) {
      const size_t q = c.at(i, j);
      const double rho = c.bg[BG_RHO][q] + w[F_RHO][q];
      const double vx = w[F_MX][q] / rho, vy = w[F_MY][q] / rho;
      const double Bx = c.bg[BG_BX][q] + w[F_BX][q], By = c.bg[BG_BY][q] + w[F_BY][q];
      const double e = c.bg[BG_E][q] + w[F_E][q];
      const double B2 = Bx * Bx + By * By;
      const double pk = (c.gamma - 1.0) * (e - 0.5 * rho * (vx * vx + vy * vy) - 0.5 * B2);
      const double a2 = c.gamma * pk / rho;
      const double b2 = B2 / rho;
      const double s = a2 + b2;
      const double cfx2 = 0.5 * (s + std::sqrt(std::max(0.0, s * s - 4.0 * a2 * Bx * Bx / rho)));
      const double cfy2 = 0.5 * (s + std::sqrt(std::max(0.0, s * s - 4.0 * a2 * By * By / rho)));
      const double cx = std::fabs(vx) + std::sqrt(cfx2);
      const double cy = std::fabs(vy) + std::sqrt(cfy2);
      if (cx > m0) m0 = cx;
      if (cy > m1) m1 = cy;
      if (a2 > m2) m2 = a2;
      if (b2 > m3) m3 = b2;
    }
  out[0] = m0; out[1] = m1; out[2] = m2; out[3] = m3;
}

// c-5 all hyperdiffusive increments D(w; v_t) added to R (interior cells).
void hyper_div(const Ctx& c, const Plane* w, const Derived& d, double vt, Plane* R) {
  Plane nu;
  const Plane* vel[2] = {&d.vx, &d.vy};
  const Plane* Btot[2] = {&d.Bx, &d.By};
  // D_rho = sum_d H_d[rho~, rho~; 1];   D_e gets sum_d H_d[eps~, eps~; 1]
  for (int dir = 0; dir < 2; ++dir) {
    hyper_nu(c, w[F_RHO], dir, c.c_rho, vt, nu);
    hyper_interface(c, nu, w[F_RHO], nullptr, 1.0, dir, R[F_RHO], nullptr, nullptr);
    hyper_nu(c, d.eps, dir, c.c_e, vt, nu);
    hyper_interface(c, nu, d.eps, nullptr, 1.0, dir, R[F_E], nullptr, nullptr);
  }
  // D_{m_l} = H_l[v_l,v_l;rho-bar] + 1/2 H_k[v_l,v_l;rho-bar] + d^c_k{ 1/2 rho nubar_l(v_k) d^c_l v_k },  k != l
  // (= div tau, tau_kl = rho/2 [nu_k(v_l) d_k v_l + nu_l(v_k) d_l v_k]); viscous work v_l * flux -> R_e.
  for (int l = 0; l < 2; ++l) {
    const int k = 1 - l;
    Plane& Rm = R[F_MX + l];
    hyper_nu(c, *vel[l], l, c.c_mom, vt, nu);
    hyper_interface(c, nu, *vel[l], &d.rho, 1.0, l, Rm, vel[l], &R[F_E]);
    hyper_nu(c, *vel[l], k, c.c_mom, vt, nu);
    hyper_interface(c, nu, *vel[l], &d.rho, 0.5, k, Rm, vel[l], &R[F_E]);
    hyper_nu(c, *vel[k], l, c.c_mom, vt, nu);
    hyper_mixed(c, nu, *vel[k], &d.rho, 0.5, l, Rm, *vel[l], R[F_E]);
  }
  // D_bx = H_y[bx~,bx~;1] - d^c_y{ nubar_x(by~) d^c_x by~ },  D_by = H_x[by~,by~;1] - d^c_x{ nubar_y(bx~) d^c_y bx~ }
  // (= -curl(eps_z), eps_z = nu_x(by) d_x by~ - nu_y(bx) d_y bx~); ohmic coupling B_l(total) * flux -> R_e.
  for (int l = 0; l < 2; ++l) {
    const int k = 1 - l;
    Plane& Rb = R[F_BX + l];
    hyper_nu(c, w[F_BX + l], k, c.c_b, vt, nu);
    hyper_interface(c, nu, w[F_BX + l], nullptr, 1.0, k, Rb, Btot[l], &R[F_E]);
    hyper_nu(c, w[F_BX + k], l, c.c_b, vt, nu);
    hyper_mixed(c, nu, w[F_BX + k], nullptr, -1.0, l, Rb, *Btot[l], R[F_E]);
  }
}

// c-6: R(w) = -sum_d d^c_d F_d + S + D(w; v_t(w)); ghosts of w must be filled.  R planes are zeroed here.
// v_t = sqrt(max a^2) + sqrt(max b^2) of the state being differentiated (c-5).
void rhs(const Ctx& c, const Plane* w, Plane* R) {
  Derived d;
  derived(c, w, d);
  for (int f = 0; f < NF; ++f) R[f].assign(c.psize(), 0.0);
  flux_div(c, w, d, R);
  sources(c, d, R);
  if (c.hd_on) {
    double ws[4];
    wavespeeds(c, w, ws);
    const double vt = std::sqrt(ws[2]) + std::sqrt(ws[3]);
    hyper_div(c, w, d, vt, R);
  }
}

// c-7: dt = cfl * min_d (Delta_d / cmax_d); an axis with n = 1 is excluded.
double cfl_dt(const Ctx& c, const Plane* w, double cfl) {
  double ws[4];
  wavespeeds(c, w, ws);
  double dt = INFINITY;
  if (c.nx > 1) dt = std::min(dt, c.dx() / ws[0]);
  if (c.ny > 1) dt = std::min(dt, c.dy() / ws[1]);
  return cfl * dt;
}

// stage state ws = wn + a * K on interior cells; ghosts: copy of wn's (keeps frozen "fixed" ghosts),
// then refilled on periodic/open sides.
void stage_state(const Ctx& c, const Plane* wn, double a, const Plane* K, Plane* ws) {
  for (int f = 0; f < NF; ++f) {
    ws[f] = wn[f];
    for (int j = 0; j < c.ny; ++j)
      for (int i = 0; i < c.nx; ++i) {
        const size_t q = c.at(i, j);
        ws[f][q] = wn[f][q] + a * K[f][q];
      }
    fill_ghosts(c, ws[f], false);
  }
}

// c-6 one step of the classical Runge-Kutta scheme, dt frozen over the step:
//   k1 = R(w^n), k2 = R(w^n + dt/2 k1), k3 = R(w^n + dt/2 k2), k4 = R(w^n + dt k3),
//   w^{n+1} = w^n + dt/6 (k1 + 2 k2 + 2 k3 + k4).       rk_order 2 = midpoint, 1 = forward Euler.
void rk_step(Ctx& c, double dt) {
  Plane k1[NF], k2[NF], k3[NF], k4[NF], ws[NF];
  Plane* wn = c.w;
  for (int f = 0; f < NF; ++f) fill_ghosts(c, wn[f], false);
  rhs(c, wn, k1);
  if (c.rk_order == 1) {
    stage_state(c, wn, dt, k1, ws);
  } else if (c.rk_order == 2) {
    stage_state(c, wn, 0.5 * dt, k1, ws);
    rhs(c, ws, k2);
    stage_state(c, wn, dt, k2, ws);
  } else {
    stage_state(c, wn, 0.5 * dt, k1, ws);
    rhs(c, ws, k2);
    stage_state(c, wn, 0.5 * dt, k2, ws);
    rhs(c, ws, k3);
    stage_state(c, wn, dt, k3, ws);
    rhs(c, ws, k4);
    for (int f = 0; f < NF; ++f) {
      ws[f] = wn[f];
      for (int j = 0; j < c.ny; ++j)
        for (int i = 0; i < c.nx; ++i) {
          const size_t q = c.at(i, j);
          ws[f][q] = wn[f][q] + dt / 6.0 * (k1[f][q] + 2.0 * k2[f][q] + 2.0 * k3[f][q] + k4[f][q]);
        }
      fill_ghosts(c, ws[f], false);
    }
  }
  for (int f = 0; f < NF; ++f) c.w[f].swap(ws[f]);
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
  Plane up(c.psize(), 0.0), nu;
  for (int j = -NG; j < 1 + NG; ++j)
    for (int i = -NG; i < n + NG; ++i) up[c.at(i, j)] = u[i + NG];
  hyper_nu(c, up, 0, coef, vt, nu);
  for (int k = -1; k <= n - 1; ++k) nu_out[k + 1] = nu[c.at(k, 0)];
  oracle_destroy(h);
  return OK;
}

// c-3 on a 1-D line: f has n+4 entries (2 extra each side); out has n entries.
int oracle_central_diff_1d(const double* f, int n, double h, double* out) {
  if (!f || !out || n < 1) { g_err = "bad argument"; return EINVAL_; }
  Plane fp(f, f + n + 4);
  for (int i = 0; i < n; ++i) out[i] = cdiff(fp, (size_t)i + 2, 1, h);
  return OK;
}

}  // extern "C"
