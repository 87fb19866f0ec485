// smaug_split_kernel.cuh -- the role-split streaming form of the fused stage kernel (hyperdiffusion on; BG = false:
// zero background, the benchmark configurations; BG = true: a background, with or without gravity).  Same
// arithmetic contract as every other stage kernel: bit-identical to the oracle.
//
// One CTA owns a strip of NC columns (NC - 8 of them produce output, 4 halo columns on each side so that
// column pairs are 16-byte aligned) and marches down a chunk of rows, newest ("head") row r, output ("tail")
// row j = r - 3.  The work of a row is split between two kinds of warps:
//
//   X warps (NC/2 threads, TWO adjacent columns per thread) do everything that is local to the head row or
//   differences along x:  derived quantities, F_x, F_y, the five kappa_x / Phi_x (the |D1| / |D3| windows of
//   the two interfaces of a pair share their differences and partial maxima, neighbours come in as 128-bit
//   shared-memory loads), the mixed fluxes G(.;y), C_y = F_y - G.  They read the input rows (128-bit loads, one row
//   ahead, held in registers) and hold no row history at all.
//   Y warps (NC threads, one column each) do everything that differences along y or assembles the result:
//   six-row register histories of rho, vx, vy, eps, bx, the five kappa_y / Phi_y, the mixed fluxes G(.;x),
//   C_x = F_x - G, the central differences of C_x and C_y, R, the RK combine, the store, the wave-speed maxima.
//
// X is a pure producer for Y; the hand-over goes through shared memory: one-row planes UP (derived head row)
// and PK (Phi_x, kappa_x), and thread-column rings CXR/BYR (F_x -> C_x, by; 5 rows), DXR (Phi_x differences;
// 4 rows), CYR (C_y; 6 rows).  Two CTA-wide barriers per row (A: UP/CXR published, B: PK/C_x published) order
// every write against every read (ring depths chosen so that a slot is never rewritten in the barrier
// interval in which it is read).  12 warps per SM at <= 168 registers instead of 8 at 240.
//
// BG = true adds: the four background planes of the head row in the landing zone; total density / total By planes
// beside the perturbed ones in UP; the totals of the tail rows rebuilt in the Y role from background values it
// loads itself; the energy source S_e from a two-buffer exchange of the tail row's vx, vy; gravity; and -- to make
// room for all that -- the C_y ring in TENSOR MEMORY (thread-private columns, tcgen05.st / tcgen05.ld) with a
// two-row staging buffer in shared memory.
#pragma once
#include <type_traits>

#include "smaug_stage_common.cuh"

#ifndef SMAUG_SPLIT_DECOUPLE
#define SMAUG_SPLIT_DECOUPLE 1
#endif
#ifndef SMAUG_SPLIT_TMEM
#define SMAUG_SPLIT_TMEM 0      // 1: the C_y ring of the Y role lives in tensor memory (thread-private columns), shared
#endif                          //    memory keeps a two-row staging buffer only (needs SMAUG_SPLIT_DECOUPLE): 25.6 KB
                                //    less shared memory per CTA, bit-identical, 3.35 instead of 3.31 ms per stage at
                                //    8000^2 -- a capacity lever (room for the background planes), not a speed-up

namespace smaug {

template <int NC, bool BG = false>
struct SplitSmem {
  static constexpr int PW = NC + 8;                     // padded plane width (index c + 4)
  // DEC (SMAUG_SPLIT_DECOUPLE): the X warps may run one row ahead of the Y warps (producer / consumer
  // barriers instead of the CTA-wide barrier A); the rings X writes after barrier B are one row deeper then,
  // and UP is single-buffered (X waits until Y has read it).
  static constexpr bool DEC = SMAUG_SPLIT_DECOUPLE != 0;
  static constexpr int NUP = DEC ? 1 : 2;               // UP buffers
  static constexpr int ND = DEC ? 5 : 4;                // rows in DXR
  static constexpr bool TM = BG || SMAUG_SPLIT_TMEM != 0;     // the background form needs the room
  static_assert(!TM || DEC, "SMAUG_SPLIT_TMEM needs SMAUG_SPLIT_DECOUPLE");
  static constexpr int NY = TM ? 2 : (DEC ? 7 : 6);     // rows in CYR (TM: a two-row staging buffer)
  static constexpr int NUPP = BG ? 8 : 6;               // planes of one UP buffer
  static constexpr int NIN = BG ? NF + NBG : NF;        // fields in the landing zone
  static constexpr int OFF_UP = 0;                      // NUP x NUPP planes: rho, vx, vy, eps, by~, bx~ of the head row
                                                        // (BG: rho is the total density; + rho~, total By)
  static constexpr int OFF_PK = OFF_UP + NUP * NUPP * PW;  // 7 planes: Phi_x[5], kappa_x(vy), kappa_x(by)
  static constexpr int OFF_CXR = OFF_PK + 7 * PW;       // ring 5 rows x 5 planes: F_x, then C_x
  static constexpr int OFF_BYR = OFF_CXR + 25 * PW;     // ring 5 rows: by~
  static constexpr int OFF_DXR = OFF_BYR + 5 * NC;      // ring ND rows x 5: Phi_x differences
  static constexpr int OFF_CYR = OFF_DXR + ND * 5 * NC; // ring NY rows x 5: C_y
  static constexpr int OFF_VJ = OFF_CYR + NY * 5 * NC;  // BG: 2 buffers x 2 planes: vx, vy of the tail row (for S_e)
  static constexpr int OFF_INR = OFF_VJ + (BG ? 4 * PW : 0);  // cp.async landing zone of the next input row
  static constexpr int OFF_RED = OFF_INR;               // block reduction scratch (after the march: INR is dead)
  static constexpr int OFF_MBAR = OFF_INR + (NIN * NC > 4 * 32 ? NIN * NC : 4 * 32);   // one mbarrier (barrier B of Y)
  static constexpr int TOTAL = OFF_MBAR + 2;
  static constexpr int CTAS_PER_SM = NC <= 64 ? 4 : (NC <= 128 ? 2 : 1);
  static constexpr size_t BYTES = (size_t)TOTAL * sizeof(double);
};

__device__ __forceinline__ void cp_async16(double* smem_dst, const double* gsrc) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ double2 lds2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void sts2(double* p, double x, double y) { *reinterpret_cast<double2*>(p) = make_double2(x, y); }
template <int NTHREADS>
__device__ __forceinline__ void cta_barrier() { asm volatile("bar.sync 0, %0;" ::"n"(NTHREADS) : "memory"); }
// producer / consumer halves of a named barrier over NTHREADS threads: the arriving threads do not wait
template <int ID, int NTHREADS>
__device__ __forceinline__ void bar_arrive() { asm volatile("bar.arrive %0, %1;" ::"n"(ID), "n"(NTHREADS) : "memory"); }
// barrier among the NTHREADS threads of one role (named barrier ID > 0)
template <int ID, int NTHREADS>
__device__ __forceinline__ void role_barrier() { asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(NTHREADS) : "memory"); }

// split-phase barrier (mbarrier): arrive when this thread's data is published, wait -- later -- for everyone's
__device__ __forceinline__ void mbar_init(double* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(double* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(double* bar, int parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra MBAR_DONE;\n"
      "bra MBAR_WAIT;\n"
      "MBAR_DONE:\n"
      "}" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
// Tensor memory as thread-private fp64 storage: a double is two 32-bit columns of the thread's own lane
// (32x32b shape: lane = 32 * (warp % 4) + lane id).  .sync.aligned: whole warps execute these together.
__device__ __forceinline__ void tm_st(unsigned taddr, double v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(__double2loint(v)),
               "r"(__double2hiint(v)) : "memory");
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_ld4(unsigned taddr, double (&v)[4]) {     // four consecutive doubles
  unsigned r0, r1, r2, r3, r4, r5, r6, r7;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3), "=r"(r4), "=r"(r5), "=r"(r6), "=r"(r7) : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
  v[0] = __hiloint2double(r1, r0); v[1] = __hiloint2double(r3, r2);
  v[2] = __hiloint2double(r5, r4); v[3] = __hiloint2double(r7, r6);
}
constexpr int SPLIT_TMEM_COLS = 128;     // 5 components x 10 slots x 2 columns = 100 -> next power of two

#ifndef SMAUG_SPLIT_MBAR
#define SMAUG_SPLIT_MBAR 0      // barrier B of the Y role: 0 bar.sync; 1 split-phase mbarrier (arrive after publishing
                                // C_x, wait after the y-differences) -- measured: no gain (3.310 vs 3.302 ms per stage)
#endif

// the operand of larger magnitude (max and abs are exact, so |amax| chains equal max-of-abs chains bit for bit;
// the comparisons take |.| as a free source modifier)
__device__ __forceinline__ double amax(double a, double b) { return fabs(a) > fabs(b) ? a : b; }

// kappa = cv * M3 / M1 in two forms with the same bits wherever both apply (c-5):
//   GUARD = true : kappa_ratio -- zero guard and the 2^200 rescue for tiny / denormal M1;
//   GUARD = false: the plain exact division, valid when M1 is an ordinary number (exponent field >= 100);
//                  `lo` collects the smallest high word of the M1 seen, so that the caller can tell afterwards
//                  whether every ratio of the row step was ordinary.  Where M1 is not, the unguarded result is
//                  garbage (possibly NaN) and the caller recomputes the whole section with GUARD = true:
//                  speculate on the common case, keep every division of a step in one basic block.
template <bool GUARD>
__device__ __forceinline__ double kappa_q(double m3, double m1, double cv, int& lo) {
  if (GUARD) return kappa_ratio(m3, m1, cv);
  lo = min(lo, __double2hiint(m1));
  return cv * ddiv(m3, m1);
}
constexpr int ORDINARY_HI = 0x06400000;     // high word of 2^-923: below it ratio_div rescales

#ifndef SMAUG_KAPPA_FAST
#define SMAUG_KAPPA_FAST 1      // 1: the guarded kappa of a family is the plain exact division, redone with the zero
#endif                          //    guard and the 2^200 rescue only when a warp vote finds an M1 below 2^-923 (same
                                //    bits: the rescue scales by 1.0 above that); the redo is a few lines, not a section.
                                //    8000^2: 3.30 -> 3.24 ms per stage without a background; the background form loses
                                //    4.6 % with it (1.067 -> 1.116 ms at 4000^2), so it is taken for BG = false only
// kappa of N ratios of one family (N = 2: the two interfaces of a column pair; N = 1: one y-interface)
template <int N, bool FAST>
__device__ __forceinline__ void kappa_family(const double (&m3)[N], const double (&m1)[N], double cv, double (&k)[N]) {
  if constexpr (FAST) {
  int lo = __double2hiint(m1[0]);
#pragma unroll
  for (int q = 1; q < N; ++q) lo = min(lo, __double2hiint(m1[q]));
#pragma unroll
  for (int q = 0; q < N; ++q) k[q] = cv * ddiv(m3[q], m1[q]);
  // Only a TINY M1 needs the redo.  A non-finite M1 (infinite or NaN: a blown-up state) passes this test, and rightly so:
  // kappa_ratio would leave it as it is (it is not zero) and scale by 1.0 (it is not tiny), i.e. form the same
  // cv * ddiv(m3, m1) from the same operands, so both forms return the same bits there too.  (An upper bound in the vote
  // was measured: +2.4 % per stage at 8000^2 for no difference in any result.)
  if (__any_sync(0xffffffffu, lo < ORDINARY_HI)) {
#pragma unroll
    for (int q = 0; q < N; ++q) k[q] = kappa_ratio(m3[q], m1[q], cv);
  }
  } else {
#pragma unroll
  for (int q = 0; q < N; ++q) k[q] = kappa_ratio(m3[q], m1[q], cv);
  }
}

// kappa at the TWO adjacent interfaces (u[2] | u[3]) and (u[3] | u[4]) of the seven cells u[0..6] (c-5).
// d0, d1: the first differences across the two interfaces.
template <bool GUARD, bool FAST = false>
__device__ __forceinline__ void kappa7(const double u[7], double cv, double& k0, double& k1, double& d0,
                                       double& d1, int& lo) {
  double a[6], t[4];
#pragma unroll
  for (int k = 0; k < 6; ++k) a[k] = u[k + 1] - u[k];
#pragma unroll
  for (int k = 0; k < 4; ++k) t[k] = fma(3.0, a[k + 1], -(u[k + 3] - u[k]));
  const double tm = amax(t[1], t[2]);
  const double am = amax(amax(a[1], a[2]), amax(a[3], a[4]));
  const double m3_0 = dabs(amax(t[0], tm)), m3_1 = dabs(amax(tm, t[3]));
  const double m1_0 = dabs(amax(a[0], am)), m1_1 = dabs(amax(am, a[5]));
  if (GUARD) {
    const double m3[2] = {m3_0, m3_1}, m1[2] = {m1_0, m1_1};
    double k[2];
    kappa_family<2, FAST>(m3, m1, cv, k);
    k0 = k[0]; k1 = k[1];
  } else {
    k0 = kappa_q<GUARD>(m3_0, m1_0, cv, lo);
    k1 = kappa_q<GUARD>(m3_1, m1_1, cv, lo);
  }
  d0 = a[2];
  d1 = a[3];
}

// kappa at ONE interface from six cells, max chains with free |.| modifiers (same value as kappa6)
template <bool GUARD, bool FAST = false>
__device__ __forceinline__ double kappa6m(double u0, double u1, double u2, double u3, double u4, double u5,
                                          double cv, double& d1_mid, int& lo) {
  const double a0 = u1 - u0, a1 = u2 - u1, a2 = u3 - u2, a3 = u4 - u3, a4 = u5 - u4;
  const double t0 = fma(3.0, a1, -(u3 - u0));
  const double t1 = fma(3.0, a2, -(u4 - u1));
  const double t2 = fma(3.0, a3, -(u5 - u2));
  const double m3 = dabs(amax(amax(t0, t1), t2));
  const double m1 = dabs(amax(amax(amax(a0, a1), amax(a2, a3)), a4));
  d1_mid = a2;
  if (GUARD) {
    const double m3a[1] = {m3}, m1a[1] = {m1};
    double k[1];
    kappa_family<1, FAST>(m3a, m1a, cv, k);
    return k[0];
  }
  return kappa_q<GUARD>(m3, m1, cv, lo);
}

// M3 = max |D3| over the three interfaces around (u[2] | u[3]), M1 = max |D1| over the five (c-5), and the
// first difference across the interface itself.
__device__ __forceinline__ void maxima6(const double u[6], double& m3, double& m1, double& d_mid) {
  const double a0 = u[1] - u[0], a1 = u[2] - u[1], a2 = u[3] - u[2], a3 = u[4] - u[3], a4 = u[5] - u[4];
  const double t0 = fma(3.0, a1, -(u[3] - u[0]));
  const double t1 = fma(3.0, a2, -(u[4] - u[1]));
  const double t2 = fma(3.0, a3, -(u[5] - u[2]));
  m3 = dabs(amax(amax(t0, t1), t2));
  m1 = dabs(amax(amax(amax(a0, a1), amax(a2, a3)), a4));
  d_mid = a2;
}

// kappa[k] = cv[k] * M3[k] / M1[k] (0 where M1 == 0) for N ratios at once.  Almost always every M1 of a
// warp is an ordinary number (exponent field >= 100): then the plain exact division is taken, without the
// zero guard and the 2^200 rescue of kappa_ratio.  One warp-uniform vote decides for all N ratios, so the
// divisions stay in one basic block and interleave.  Both paths give the same bits where both apply.
template <int N>
__device__ __forceinline__ void kappa_batch(const double (&m3)[N], const double (&m1)[N], const double (&cv)[N],
                                            double (&kap)[N]) {
#ifdef SMAUG_NO_KBATCH
#pragma unroll
  for (int k = 0; k < N; ++k) kap[k] = kappa_ratio(m3[k], m1[k], cv[k]);
  return;
#endif
  int lo = __double2hiint(m1[0]);
#pragma unroll
  for (int k = 1; k < N; ++k) lo = min(lo, __double2hiint(m1[k]));
  if (__any_sync(0xffffffffu, lo < 0x06400000)) {
#pragma unroll
    for (int k = 0; k < N; ++k) kap[k] = kappa_ratio(m3[k], m1[k], cv[k]);
  } else {
#pragma unroll
    for (int k = 0; k < N; ++k) kap[k] = cv[k] * ddiv(m3[k], m1[k]);
  }
}

#ifndef SMAUG_SPLIT_LATELOAD
#define SMAUG_SPLIT_LATELOAD 0   // RK operands of the tail row: 0 loaded at the top of the step, 1 after barrier B,
#endif                           // 2 after barrier B with an L2 prefetch at the top
__device__ __forceinline__ void prefetch_l2(const double* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
#ifndef SMAUG_SPLIT_SPEC
#define SMAUG_SPLIT_SPEC 0
#endif
#ifndef SMAUG_SPLIT_KY
#define SMAUG_SPLIT_KY 0      // 0: one kappa at a time (guarded division), 1: batched with a fast path
#endif
#ifndef SMAUG_SPLIT_YUNROLL
#define SMAUG_SPLIT_YUNROLL 2
#endif
constexpr int SPLIT_YUNROLL = SMAUG_SPLIT_YUNROLL;   // row steps of the Y role per loop trip

#ifndef SMAUG_SPLIT_WSFILTER
#define SMAUG_SPLIT_WSFILTER 1
#endif
#ifndef SMAUG_SPLIT_JIN3
#define SMAUG_SPLIT_JIN3 1
#endif
// Wave-speed maxima of one written cell folded into the running maxima m[4] (c-4): the same operation sequence
// as cell_wavespeeds, with two changes that leave every reduced value unchanged:
//  * a candidate enters with `c > m ? c : m` against a running maximum that is >= 0, which drops NaNs and
//    negative values exactly like the clamp fmax(c, 0) followed by a max;
//  * FULL: the two fast speeds (four square roots) are evaluated only where they can still raise a maximum.
//    thr[d] is any lower bound of the final max(|v_d| + c_f,d) (the running maximum of this thread or the value
//    other CTAs have already published).  With a^2 >= 0, b^2 >= 0:  c_f,d^2 <= s = a^2 + b^2, and in floating
//    point |v_d| + sqrt(c_f,d^2) <= (|v_d| + sqrt(s) (1 + 2u)) (1 + u), u = 2^-53.  So with t = thr - |v_d|,
//    t > thr 2^-10 and t^2 >= s (1 + 2^-40) prove the cell cannot exceed thr (the margin 2^-40 covers the
//    rounding of t, t^2 and the bound by ten orders of magnitude; t > thr 2^-10 keeps the cancellation in t
//    harmless).  Skipped cells therefore never held the maximum: the reduced values are bit-identical.
template <int WS>
__device__ __forceinline__ void split_wavespeeds(const double (&o)[NF], double gamma, double (&m)[4], double thr0,
                                                 double thr1) {
  const double rr = drcp(o[F_RHO]);
  const double vx = o[F_MX] * rr, vy = o[F_MY] * rr;
  const double B2 = fma(o[F_BY], o[F_BY], o[F_BX] * o[F_BX]);
  const double pk = (gamma - 1.0) * ((o[F_E] - 0.5 * fma(o[F_MY], vy, o[F_MX] * vx)) - 0.5 * B2);
  const double a2 = (gamma * pk) * rr;
  const double b2 = B2 * rr;
  m[2] = a2 > m[2] ? a2 : m[2];
  m[3] = b2 > m[3] ? b2 : m[3];
  if (WS == WS_FULL) {
    const double s = a2 + b2;
#if SMAUG_SPLIT_WSFILTER
    const double t0 = thr0 - fabs(vx), t1 = thr1 - fabs(vy);
    const double sm = s * (1.0 + 0x1p-40);
    const bool skip = a2 >= 0.0 && b2 >= 0.0 && t0 > thr0 * 0x1p-10 && t1 > thr1 * 0x1p-10 && t0 * t0 >= sm &&
                      t1 * t1 >= sm;
    if (skip) return;
#endif
    const double fa = (4.0 * a2) * rr;
    const double d0 = fma(s, s, -(fa * (o[F_BX] * o[F_BX]))), d1 = fma(s, s, -(fa * (o[F_BY] * o[F_BY])));
    const double cfx2 = 0.5 * (s + sqrt(d0 > 0.0 ? d0 : 0.0));
    const double cfy2 = 0.5 * (s + sqrt(d1 > 0.0 ? d1 : 0.0));
    const double c0 = fabs(vx) + sqrt(cfx2), c1 = fabs(vy) + sqrt(cfy2);
    m[0] = c0 > m[0] ? c0 : m[0];
    m[1] = c1 > m[1] ? c1 : m[1];
  }
}

template <int NC, int COMBINE, int WS, bool BG = false, bool GRAV = false>   // GRAV: gravity without a background
#ifdef SMAUG_SPLIT_MAXNREG
__global__ void __maxnreg__(SMAUG_SPLIT_MAXNREG) split_kernel
#else
__global__ void __launch_bounds__(NC + NC / 2, SplitSmem<NC, BG>::CTAS_PER_SM) split_kernel
#endif
(const StageArgs a, const MarchGeom mg) {
  using S = SplitSmem<NC, BG>;
  constexpr bool TM = S::TM;
  constexpr bool KFAST = SMAUG_KAPPA_FAST != 0 && !BG;
  constexpr int PW = S::PW, NXT = NC / 2, NTH = NC + NC / 2;
  extern __shared__ __align__(16) double smem[];
  double* const UP = smem + S::OFF_UP;
  double* const PK = smem + S::OFF_PK;
  double* const CXR = smem + S::OFF_CXR;
  double* const BYR = smem + S::OFF_BYR;
  double* const DXR = smem + S::OFF_DXR;
  double* const CYR = smem + S::OFF_CYR;
  double* const INR = smem + S::OFF_INR;
  double* const red_sh = smem + S::OFF_RED;
  const Grid& g = a.g;
  const int tid = threadIdx.x;
  constexpr int W = NC - 8;
  const int x0 = blockIdx.x * W;
  const int ystart = blockIdx.y * mg.rows_per_cta;
  const int yend = min(ystart + mg.rows_per_cta, g.ny);
  double wsmax[4] = {0.0, 0.0, 0.0, 0.0};
  double* const MBAR = smem + S::OFF_MBAR;
#if SMAUG_SPLIT_MBAR
  if (tid == 0) mbar_init(MBAR, NC);
  __syncthreads();
#endif
  unsigned tm_base = 0;
  if constexpr (TM) {
  unsigned* const tm_base_sh = reinterpret_cast<unsigned*>(MBAR + 1);
  if (tid < 32) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                     (unsigned)__cvta_generic_to_shared(tm_base_sh)), "n"(SPLIT_TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  tm_base = *tm_base_sh;
  }

  if (tid < NXT) {
    // =================================================================== X role: columns c0, c0 + 1
    const int c0 = 2 * tid, tp = c0 + 4;
    const double gm1 = a.prm.gamma - 1.0;
    const double vt = sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][2])) +
                      sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][3]));
    const double cv_rho = a.prm.c_rho * vt, cv_mom = a.prm.c_mom * vt, cv_e = a.prm.c_e * vt, cv_b = a.prm.c_b * vt;
    const int gcol = min(x0 - 4 + c0 + XOFF, g.pitch - 2);            // even => 16-byte aligned pairs
    const long long colbase = (long long)NG * g.pitch + gcol;
    // the input rows arrive one step ahead through cp.async (16 bytes per field and thread) into a
    // thread-private landing zone: no registers are held while a row is in flight, and the copy cannot be
    // sunk towards its use by the compiler (which exposed the HBM latency when the rows were plain loads).
    // The copy of row r + 1 is issued after every value of row r has been consumed from the landing zone.
    double* const inr = INR + c0;
    auto fetch_row = [&](int row) {
      const long long ga = colbase + (long long)min(row, g.ny + NG - 1) * g.pitch;
#pragma unroll
      for (int f = 0; f < NF; ++f) cp_async16(inr + f * NC, a.in.p[f] + ga);
      if constexpr (BG) {
#pragma unroll
        for (int k = 0; k < NBG; ++k) cp_async16(inr + (NF + k) * NC, a.bg.p[k] + ga);
      }
      cp_async_commit();
    };
    fetch_row(ystart - NG);
    int s4 = 0, s5 = 0, s6 = 0;     // ring slots of row r (mod ND, 5, NY)
    int par = 0;                    // UP buffer of row r
    constexpr bool DEC = S::DEC;
    constexpr int ND = S::ND, NY = S::NY;

#pragma unroll 1
    for (int r = ystart - NG; r < yend + NG; ++r) {
      double rho[2], mx[2], my[2], et[2], bx[2], by[2];
      cp_async_wait<0>();
      {
        const double2 q0 = lds2(inr + F_RHO * NC), q1 = lds2(inr + F_MX * NC), q2 = lds2(inr + F_MY * NC);
        const double2 q3 = lds2(inr + F_E * NC), q4 = lds2(inr + F_BX * NC), q5 = lds2(inr + F_BY * NC);
        rho[0] = q0.x; rho[1] = q0.y; mx[0] = q1.x; mx[1] = q1.y; my[0] = q2.x; my[1] = q2.y;
        et[0] = q3.x; et[1] = q3.y; bx[0] = q4.x; bx[1] = q4.y; by[0] = q5.x; by[1] = q5.y;
      }
      double* const UPr = UP + par * S::NUPP * PW;
      // ---------------------------------------------------------------- derived quantities, F_x, F_y of row r
      // (BG: c-2 with the background terms; rho[] becomes the total density, rhot[] keeps the perturbation,
      //  Bxt / Byt are the total field; without a background these coincide and the extra terms are exact zeros)
      double vx[2], vy[2], eps[2], cyn[2][5], fx[2][5];
      [[maybe_unused]] double rhot[2] = {rho[0], rho[1]}, Bxt[2] = {bx[0], bx[1]}, Byt[2] = {by[0], by[1]};
      if constexpr (BG) {
        const double2 g0 = lds2(inr + (NF + BG_RHO) * NC), g1 = lds2(inr + (NF + BG_E) * NC);
        const double2 g2 = lds2(inr + (NF + BG_BX) * NC), g3 = lds2(inr + (NF + BG_BY) * NC);
        const double rb[2] = {g0.x, g0.y}, eb[2] = {g1.x, g1.y}, Bbx[2] = {g2.x, g2.y}, Bby[2] = {g3.x, g3.y};
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          rho[q] = rb[q] + rhot[q];
          const double rr = drcp(rho[q]);
          vx[q] = mx[q] * rr; vy[q] = my[q] * rr;
          const double b2h = 0.5 * fma(by[q], by[q], bx[q] * bx[q]);
          const double cross = fma(Bby[q], by[q], Bbx[q] * bx[q]);
          const double ke = 0.5 * fma(my[q], vy[q], mx[q] * vx[q]);
          eps[q] = ((et[q] - ke) - cross) - b2h;
          const double ptt = fma(gm1, eps[q], cross + b2h);
          Bxt[q] = Bbx[q] + bx[q]; Byt[q] = Bby[q] + by[q];
          const double btv = fma(by[q], vy[q], bx[q] * vx[q]);
          const double Bbv = fma(Bby[q], vy[q], Bbx[q] * vx[q]);
          const double h = (et[q] + eb[q]) + ptt;
          cyn[q][C_RHO] = rho[q] * vy[q];
          cyn[q][C_MX] = (fma(mx[q], vy[q], -(bx[q] * by[q])) - bx[q] * Bby[q]) - Bbx[q] * by[q];
          cyn[q][C_MY] = ((fma(my[q], vy[q], -(by[q] * by[q])) - by[q] * Bby[q]) - Bby[q] * by[q]) + ptt;
          cyn[q][C_E] = (fma(vy[q], h, -(by[q] * btv)) - by[q] * Bbv) - Bby[q] * btv;
          cyn[q][C_B] = fma(vy[q], Bxt[q], -(Byt[q] * vx[q]));
          fx[q][C_RHO] = rho[q] * vx[q];
          fx[q][C_MX] = ((fma(mx[q], vx[q], -(bx[q] * bx[q])) - bx[q] * Bbx[q]) - Bbx[q] * bx[q]) + ptt;
          fx[q][C_MY] = (fma(my[q], vx[q], -(by[q] * bx[q])) - by[q] * Bbx[q]) - Bby[q] * bx[q];
          fx[q][C_E] = (fma(vx[q], h, -(bx[q] * btv)) - bx[q] * Bbv) - Bbx[q] * btv;
          fx[q][C_B] = fma(vx[q], Byt[q], -(Bxt[q] * vy[q]));
        }
      } else {
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const double rr = drcp(rho[q]);
        vx[q] = mx[q] * rr; vy[q] = my[q] * rr;
        const double b2h = 0.5 * fma(by[q], by[q], bx[q] * bx[q]);
        const double ke = 0.5 * fma(my[q], vy[q], mx[q] * vx[q]);
        eps[q] = (et[q] - ke) - b2h;
        const double ptt = fma(gm1, eps[q], b2h);
        const double btv = fma(by[q], vy[q], bx[q] * vx[q]);
        const double h = et[q] + ptt;
        cyn[q][C_RHO] = rho[q] * vy[q];
        cyn[q][C_MX] = fma(mx[q], vy[q], -(bx[q] * by[q]));
        cyn[q][C_MY] = fma(my[q], vy[q], -(by[q] * by[q])) + ptt;
        cyn[q][C_E] = fma(vy[q], h, -(by[q] * btv));
        cyn[q][C_B] = fma(vy[q], bx[q], -(by[q] * vx[q]));
        fx[q][C_RHO] = rho[q] * vx[q];
        fx[q][C_MX] = fma(mx[q], vx[q], -(bx[q] * bx[q])) + ptt;
        fx[q][C_MY] = fma(my[q], vx[q], -(by[q] * bx[q]));
        fx[q][C_E] = fma(vx[q], h, -(bx[q] * btv));
        fx[q][C_B] = fma(vx[q], by[q], -(bx[q] * vy[q]));
      }
      }
      if (DEC) role_barrier<4, NTH>();      // ---- E: every warp is done with UP of the previous row
      sts2(UPr + 0 * PW + tp, rho[0], rho[1]); sts2(UPr + 1 * PW + tp, vx[0], vx[1]);
      sts2(UPr + 2 * PW + tp, vy[0], vy[1]);   sts2(UPr + 3 * PW + tp, eps[0], eps[1]);
      sts2(UPr + 4 * PW + tp, by[0], by[1]);   sts2(UPr + 5 * PW + tp, bx[0], bx[1]);
      if constexpr (BG) { sts2(UPr + 6 * PW + tp, rhot[0], rhot[1]); sts2(UPr + 7 * PW + tp, Byt[0], Byt[1]); }
#pragma unroll
      for (int f = 0; f < 5; ++f) sts2(CXR + (s5 * 5 + f) * PW + tp, fx[0][f], fx[1][f]);
      sts2(BYR + s5 * NC + c0, by[0], by[1]);
      fetch_row(r + 1);     // the stores above depend on every value read from the landing zone
      if (DEC) {
        bar_arrive<3, NTH>();                                         // ---- F: head row published for Y
        role_barrier<5, NXT>();                                       // ---- A among the X warps
      } else {
        cta_barrier<NTH>();                                           // ---- A (both roles)
      }

      // ---------------------------------------------------------------- x-interfaces (c0|c0+1), (c0+1|c0+2)
      double px[2][5], kxv[2], kxb[2], dcx_vy[2], dcx_by[2];
      auto x_interfaces = [&](auto GUARD_) {
        constexpr bool GUARD = decltype(GUARD_)::value;
        int lo = 0x7fffffff;
        double u[7], k0, k1, d0, d1;
        auto gather = [&](int plane, double o0, double o1) {
          const double2 l = lds2(UPr + plane * PW + tp - 2), rgt = lds2(UPr + plane * PW + tp + 2);
          u[0] = l.x; u[1] = l.y; u[2] = o0; u[3] = o1; u[4] = rgt.x; u[5] = rgt.y;
          u[6] = UPr[plane * PW + tp + 4];
        };
        // kappa_x(rho~) on the perturbed density; the interface weights rho-bar use the total density
        if constexpr (BG) gather(6, rhot[0], rhot[1]); else gather(0, rho[0], rho[1]);
        kappa7<GUARD, KFAST>(u, cv_rho, k0, k1, d0, d1, lo);
        const double rho_r = BG ? UPr[0 * PW + tp + 2] : u[4];           // total density of the cell right of the pair
        const double rbar0 = 0.5 * (rho[0] + rho[1]), rbar1 = 0.5 * (rho[1] + rho_r);
        px[0][C_RHO] = k0 * d0; px[1][C_RHO] = k1 * d1;
        gather(1, vx[0], vx[1]);
        kappa7<GUARD, KFAST>(u, cv_mom, k0, k1, d0, d1, lo);
        px[0][C_MX] = (rbar0 * k0) * d0; px[1][C_MX] = (rbar1 * k1) * d1;
        const double vxbar0 = 0.5 * (u[2] + u[3]), vxbar1 = 0.5 * (u[3] + u[4]);
        gather(2, vy[0], vy[1]);
        kappa7<GUARD, KFAST>(u, cv_mom, kxv[0], kxv[1], d0, d1, lo);
        px[0][C_MY] = ((0.5 * rbar0) * kxv[0]) * d0; px[1][C_MY] = ((0.5 * rbar1) * kxv[1]) * d1;
        const double vybar0 = 0.5 * (u[2] + u[3]), vybar1 = 0.5 * (u[3] + u[4]);
        dcx_vy[0] = cd12v(u[0], u[1], u[3], u[4]); dcx_vy[1] = cd12v(u[1], u[2], u[4], u[5]);
        gather(3, eps[0], eps[1]);
        kappa7<GUARD, KFAST>(u, cv_e, k0, k1, d0, d1, lo);
        const double p_eps0 = k0 * d0, p_eps1 = k1 * d1;
        gather(4, by[0], by[1]);
        kappa7<GUARD, KFAST>(u, cv_b, kxb[0], kxb[1], d0, d1, lo);
        px[0][C_B] = kxb[0] * d0; px[1][C_B] = kxb[1] * d1;
        dcx_by[0] = cd12v(u[0], u[1], u[3], u[4]); dcx_by[1] = cd12v(u[1], u[2], u[4], u[5]);
        // ohmic coupling with the TOTAL transverse field (u[] holds by~ here)
        const double By_r = BG ? UPr[7 * PW + tp + 2] : u[4];
        px[0][C_E] = fma(0.5 * (Byt[0] + Byt[1]), px[0][C_B], fma(vybar0, px[0][C_MY], fma(vxbar0, px[0][C_MX], p_eps0)));
        px[1][C_E] = fma(0.5 * (Byt[1] + By_r), px[1][C_B], fma(vybar1, px[1][C_MY], fma(vxbar1, px[1][C_MX], p_eps1)));
        return lo;
      };
      // SMAUG_SPLIT_SPEC: speculate that every M1 of this warp's row step is an ordinary number and redo the
      // section otherwise (measured slower on B200: 3.87 vs 3.57 ms per stage at 8000^2 -- larger loop bodies)
#if SMAUG_SPLIT_SPEC
      if (__any_sync(0xffffffffu, x_interfaces(std::false_type{}) < ORDINARY_HI)) x_interfaces(std::true_type{});
#else
      x_interfaces(std::true_type{});
#endif
#pragma unroll
      for (int f = 0; f < 5; ++f) sts2(PK + f * PW + tp, px[0][f], px[1][f]);
      sts2(PK + 5 * PW + tp, kxv[0], kxv[1]);
      sts2(PK + 6 * PW + tp, kxb[0], kxb[1]);
      role_barrier<1, NXT>();                                         // ---- B (X warps only)

      // ---------------------------------------------------------------- Phi_x differences, G(.;y), C_y of row r
      {
        const double kvl = PK[5 * PW + tp - 1], kbl = PK[6 * PW + tp - 1];
#pragma unroll
        for (int f = 0; f < 5; ++f)
          sts2(DXR + (s4 * 5 + f) * NC + c0, px[0][f] - PK[f * PW + tp - 1], px[1][f] - px[0][f]);
        const double kv0 = 0.5 * (kvl + kxv[0]), kv1 = 0.5 * (kxv[0] + kxv[1]);
        const double kb0 = 0.5 * (kbl + kxb[0]), kb1 = 0.5 * (kxb[0] + kxb[1]);
        const double gm0 = ((0.5 * rho[0]) * kv0) * (dcx_vy[0] * (1.0 / 12.0));      // G(mx ; y)
        const double gm1_ = ((0.5 * rho[1]) * kv1) * (dcx_vy[1] * (1.0 / 12.0));
        const double gb0 = -(kb0 * (dcx_by[0] * (1.0 / 12.0)));                       // G(bx ; y)
        const double gb1 = -(kb1 * (dcx_by[1] * (1.0 / 12.0)));
        double* cy = CYR + s6 * 5 * NC + c0;
        sts2(cy + C_RHO * NC, cyn[0][C_RHO], cyn[1][C_RHO]);
        sts2(cy + C_MX * NC, cyn[0][C_MX] - gm0, cyn[1][C_MX] - gm1_);
        sts2(cy + C_MY * NC, cyn[0][C_MY], cyn[1][C_MY]);
        sts2(cy + C_E * NC, cyn[0][C_E] - fma(vx[0], gm0, Bxt[0] * gb0), cyn[1][C_E] - fma(vx[1], gm1_, Bxt[1] * gb1));
        sts2(cy + C_B * NC, cyn[0][C_B] - gb0, cyn[1][C_B] - gb1);
      }
      s4 = s4 == ND - 1 ? 0 : s4 + 1;
      s5 = s5 == 4 ? 0 : s5 + 1;
      s6 = s6 == NY - 1 ? 0 : s6 + 1;
      if (!DEC) par ^= 1;
    }
    cp_async_wait<0>();
  } else {
    // =================================================================== Y role: column c
    const int c = tid - NXT, tp = c + 4;
    const int ci = x0 - 4 + c;
    const int cl = min(ci, g.nx + NG - 1);
    const bool col_out = c >= 4 && c < NC - 4 && ci < g.nx;
    const double gamma = a.prm.gamma;
    const double idx_ = a.prm.inv_dx, idy_ = a.prm.inv_dy;
    const double vt = sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][2])) +
                      sqrt(__longlong_as_double((long long)a.sc->red[a.red_in][3]));
    const double cv_rho = a.prm.c_rho * vt, cv_mom = a.prm.c_mom * vt, cv_e = a.prm.c_e * vt, cv_b = a.prm.c_b * vt;
    const double cdt = a.c * a.sc->dt;
    // element offset of (cl, row j) inside a plane, advanced by one row per step (a plane has fewer than
    // 2^31 elements: smaug_create checks); rows above the chunk are never dereferenced
    unsigned gj = (unsigned)(ystart + NG) * (unsigned)g.pitch + (unsigned)(cl + XOFF);
    const unsigned upitch = (unsigned)g.pitch;
    // six-row histories (index 0 = row r-5 ... 5 = row r)
    double hr[6], hvx[6], hvy[6], he[6], hbx[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) { hr[k] = 1.0; hvx[k] = 0.0; hvy[k] = 0.0; he[k] = 0.0; hbx[k] = 0.0; }
    double py_prev[5] = {0.0, 0.0, 0.0, 0.0, 0.0};        // Phi_y at interface (j-1 | j)
    double kyv_prev = 0.0, kyb_prev = 0.0;                 // kappa_y(vx), kappa_y(bx) at (j-1 | j)
    constexpr bool DEC = S::DEC;
    constexpr int ND = S::ND, NY = S::NY;
    int s4 = ND - 3, s5 = 2, s6 = 0;                       // slots of row j in DXR, CXR; of row r in CYR
    int par = 0;                                           // UP buffer of row r
    [[maybe_unused]] int mph = 0;                          // phase parity of barrier B (mbarrier)
    // (TM) C_y ring in tensor memory: component f at columns 20 f .. 20 f + 19 = ten slots of one double; row k is
    // written to slots (k mod 5) and (k mod 5) + 5, so that any four consecutive rows are four consecutive slots
    [[maybe_unused]] const unsigned tm_y = tm_base + ((unsigned)(((tid >> 5) & 3) * 32) << 16);
    [[maybe_unused]] int p5 = 4;                           // slot class of row r - 1
    [[maybe_unused]] int yst = 1;                          // staging buffer holding C_y(r - 1)
    [[maybe_unused]] double cyv[5] = {0.0, 0.0, 0.0, 0.0, 0.0};   // C_y(r - 1) of this column
    [[maybe_unused]] double* const VJ = smem + S::OFF_VJ;  // BG: vx, vy of the tail row, two buffers
    [[maybe_unused]] int vjb = 0;
    [[maybe_unused]] const double gm1y = a.prm.gamma - 1.0;
    if (DEC) bar_arrive<4, NTH>();                         // E for the first row: nothing to wait for
    // (row r starts in slot 0 of every ring; row j = r - 3 is then at -3 mod 4 = 1 and -3 mod 5 = 2)

#pragma unroll SPLIT_YUNROLL
    for (int r = ystart - NG; r < yend + NG; ++r) {
      const int j = r - NG;
      const bool tail_on = j >= ystart;
      const bool ky_on = r >= ystart + NG - 1;
      // operands of the RK combine for row j: issued here, consumed at the end of the step
      double jbase[NF], jacc[NF], jin[NF];
      // the stage input at row j: rho~, bx~ are in the histories and by~ in the by ring (the same values X read
      // from global memory), so only mx, my, e~ are loaded
      auto load_jin = [&]() {
#if SMAUG_SPLIT_JIN3
        jin[F_MX] = a.in.p[F_MX][gj]; jin[F_MY] = a.in.p[F_MY][gj]; jin[F_E] = a.in.p[F_E][gj];
#else
#pragma unroll
        for (int f = 0; f < NF; ++f) jin[f] = a.in.p[f][gj];
#endif
      };
      // maxima other CTAs have already published for this launch: lower bounds of the final maxima (any stale
      // value is one too), used by split_wavespeeds to skip cells that cannot raise them
      double gthr0 = 0.0, gthr1 = 0.0;
      if (WS == WS_FULL && tail_on) {
        gthr0 = __longlong_as_double((long long)__ldcg(&a.sc->red[a.red_out][0]));
        gthr1 = __longlong_as_double((long long)__ldcg(&a.sc->red[a.red_out][1]));
      }
      auto load_operands = [&]() {
        if (COMBINE == COMBINE_FINAL) {
#pragma unroll
          for (int f = 0; f < NF; ++f) jacc[f] = a.acc_in.p[f][gj];
          load_jin();
        } else {
#pragma unroll
          for (int f = 0; f < NF; ++f) jbase[f] = a.base.p[f][gj];
          if (COMBINE == COMBINE_ACC) load_jin();
        }
      };
#if SMAUG_SPLIT_LATELOAD == 0
      if (tail_on) load_operands();
#elif SMAUG_SPLIT_LATELOAD == 2 || SMAUG_SPLIT_LATELOAD == 3
      if (tail_on) {     // bring the lines into L2; the loads themselves are issued after barrier B
        if (COMBINE == COMBINE_FINAL) {
#pragma unroll
          for (int f = 0; f < NF; ++f) { prefetch_l2(a.in.p[f] + gj); prefetch_l2(a.acc_in.p[f] + gj); }
        } else {
#pragma unroll
          for (int f = 0; f < NF; ++f) prefetch_l2(a.base.p[f] + gj);
          if (COMBINE == COMBINE_ACC) {
#pragma unroll
            for (int f = 0; f < NF; ++f) prefetch_l2(a.in.p[f] + gj);
          }
        }
      }
#endif
      // BG: background of rows j and j + 1 at this column (L2 hits: X fetched these rows three steps ago); the
      // totals are rebuilt with the oracle's own operations (rho = rho_b + rho~, B = B_b + b~)
      [[maybe_unused]] double rb0 = 0.0, rb1 = 0.0, Bbx0 = 0.0, Bbx1 = 0.0, eb0 = 0.0, Bby0 = 0.0;
      if constexpr (BG) {
        if (ky_on) {
          const unsigned gq = tail_on ? gj : gj - upitch;            // (cl, row j)
          rb0 = a.bg.p[BG_RHO][gq]; rb1 = a.bg.p[BG_RHO][gq + upitch];
          Bbx0 = a.bg.p[BG_BX][gq]; Bbx1 = a.bg.p[BG_BX][gq + upitch];
          if (tail_on) { eb0 = a.bg.p[BG_E][gq]; Bby0 = a.bg.p[BG_BY][gq]; }
        }
      }
      if (DEC) role_barrier<3, NTH>();                                // ---- F: head row r is published
      else cta_barrier<NTH>();                                        // ---- A (both roles)
      const double* const UPr = UP + par * S::NUPP * PW;
#pragma unroll
      for (int k = 0; k < 5; ++k) { hr[k] = hr[k + 1]; hvx[k] = hvx[k + 1]; hvy[k] = hvy[k + 1]; he[k] = he[k + 1]; hbx[k] = hbx[k + 1]; }
      hr[5] = UPr[(BG ? 6 : 0) * PW + tp]; hvx[5] = UPr[1 * PW + tp]; hvy[5] = UPr[2 * PW + tp]; he[5] = UPr[3 * PW + tp];
      hbx[5] = UPr[5 * PW + tp];
      if constexpr (TM) {
        // C_y(r - 1), which X wrote at the end of its step r - 1, from the staging buffer into the ring
#pragma unroll
        for (int f = 0; f < 5; ++f) cyv[f] = CYR[(yst * 5 + f) * NC + c];
        asm volatile("" ::"d"(cyv[0]), "d"(cyv[1]), "d"(cyv[2]), "d"(cyv[3]), "d"(cyv[4]) : "memory");
      }
      if (DEC) {
        // E: UP may be overwritten (the loads above must have landed: consume them first)
        asm volatile("" ::"d"(hr[5]), "d"(hvx[5]), "d"(hvy[5]), "d"(he[5]), "d"(hbx[5]) : "memory");
        if (r + 1 < yend + NG) bar_arrive<4, NTH>();
      }
      if constexpr (TM) {
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          tm_st(tm_y + 20 * f + 2 * p5, cyv[f]);
          tm_st(tm_y + 20 * f + 2 * p5 + 10, cyv[f]);
        }
        tm_wait_st();
      }

      // ---------------------------------------------------------------- y-interface (j | j+1)
      double py[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      double kyv = 0.0, kyb = 0.0;
      auto y_interface = [&](auto GUARD_) {
        constexpr bool GUARD = decltype(GUARD_)::value;
        int lo = 0x7fffffff;
        double d_rho, d_vx, d_vy, d_e, d_bx;
        const double k_rho = kappa6m<GUARD, KFAST>(hr[0], hr[1], hr[2], hr[3], hr[4], hr[5], cv_rho, d_rho, lo);
        kyv = kappa6m<GUARD, KFAST>(hvx[0], hvx[1], hvx[2], hvx[3], hvx[4], hvx[5], cv_mom, d_vx, lo);
        const double k_vy = kappa6m<GUARD, KFAST>(hvy[0], hvy[1], hvy[2], hvy[3], hvy[4], hvy[5], cv_mom, d_vy, lo);
        const double k_e = kappa6m<GUARD, KFAST>(he[0], he[1], he[2], he[3], he[4], he[5], cv_e, d_e, lo);
        kyb = kappa6m<GUARD, KFAST>(hbx[0], hbx[1], hbx[2], hbx[3], hbx[4], hbx[5], cv_b, d_bx, lo);
        const double rbar = BG ? 0.5 * ((rb0 + hr[2]) + (rb1 + hr[3])) : 0.5 * (hr[2] + hr[3]);
        const double p_rho = k_rho * d_rho;
        const double p_mx = ((0.5 * rbar) * kyv) * d_vx;
        const double p_my = (rbar * k_vy) * d_vy;
        const double p_eps = k_e * d_e;
        const double p_b = kyb * d_bx;
        py[C_RHO] = p_rho; py[C_MX] = p_mx; py[C_MY] = p_my; py[C_B] = p_b;
        const double Bbar = BG ? 0.5 * ((Bbx0 + hbx[2]) + (Bbx1 + hbx[3])) : 0.5 * (hbx[2] + hbx[3]);
        py[C_E] = fma(Bbar, p_b,
                      fma(0.5 * (hvy[2] + hvy[3]), p_my, fma(0.5 * (hvx[2] + hvx[3]), p_mx, p_eps)));
        return lo;
      };
      if (ky_on) {
#if SMAUG_SPLIT_SPEC
        if (__any_sync(0xffffffffu, y_interface(std::false_type{}) < ORDINARY_HI)) y_interface(std::true_type{});
#else
        y_interface(std::true_type{});
#endif
      }
#if SMAUG_SPLIT_LATELOAD == 3 || SMAUG_SPLIT_LATELOAD == 4
      if (tail_on) load_operands();     // after the register-hungry kappa phase, one barrier ahead of their use
#endif
      if (tail_on) {
        // G(my ; x), G(by ; x) and their energy companion at row j (histories index 2); C_x = F_x - G
        const double kv = 0.5 * (kyv_prev + kyv);
        const double kb = 0.5 * (kyb_prev + kyb);
        const double rho_j = BG ? rb0 + hr[2] : hr[2];               // total density of the tail cell
        const double gm = ((0.5 * rho_j) * kv) * (cd12v(hvx[0], hvx[1], hvx[3], hvx[4]) * (1.0 / 12.0));
        const double gb = -(kb * (cd12v(hbx[0], hbx[1], hbx[3], hbx[4]) * (1.0 / 12.0)));
        double* cx = CXR + s5 * 5 * PW + tp;
        const double jby = BYR[s5 * NC + c];
#if SMAUG_SPLIT_JIN3
        if (COMBINE != COMBINE_BASE) { jin[F_RHO] = hr[2]; jin[F_BX] = hbx[2]; jin[F_BY] = jby; }
#endif
        cx[C_MY * PW] = cx[C_MY * PW] - gm;
        cx[C_E * PW] = cx[C_E * PW] - fma(hvy[2], gm, (BG ? Bby0 + jby : jby) * gb);
        cx[C_B * PW] = cx[C_B * PW] - gb;
        if constexpr (BG) {       // vx, vy of the tail row for the x-derivatives of S_e (read after barrier B)
          VJ[(vjb * 2 + 0) * PW + tp] = hvx[2];
          VJ[(vjb * 2 + 1) * PW + tp] = hvy[2];
        }
      }
#if SMAUG_SPLIT_MBAR
      mbar_arrive(MBAR);                                              // ---- B (Y warps only): C_x(j) published
#else
      role_barrier<2, NC>();                                          // ---- B (Y warps only)
#endif

      // ---------------------------------------------------------------- assemble R(j), combine, write
      // (everything that does not need the neighbours' C_x comes before the wait of barrier B)
      double cdyi[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (tail_on) {
        // rows j-2, j-1, j+1, j+2 = r-5, r-4, r-2, r-1 in the mod-NY ring
        auto back = [&](int k) { const int q = s6 + (NY - k); return q >= NY ? q - NY : q; };   // slot of row r - k
        const int jm2 = back(5), jm1 = back(4), jp1 = back(2), jp2 = back(1);
        if constexpr (TM) {
          const int q5 = p5 == 4 ? 0 : p5 + 1;            // slot of row r - 5; rows r-5 .. r-2 follow each other
#pragma unroll
          for (int f = 0; f < 5; ++f) {
            double v[4];
            tm_ld4(tm_y + 20 * f + 2 * q5, v);
            cdyi[f] = cd12v(v[0], v[1], v[3], cyv[f]) * idy_;
          }
        } else {
#pragma unroll
          for (int f = 0; f < 5; ++f)
            cdyi[f] = cd12v(CYR[(jm2 * 5 + f) * NC + c], CYR[(jm1 * 5 + f) * NC + c], CYR[(jp1 * 5 + f) * NC + c],
                            CYR[(jp2 * 5 + f) * NC + c]) * idy_;
        }
      }
#if SMAUG_SPLIT_MBAR
      mbar_wait(MBAR, mph);
      mph ^= 1;
#endif
      if (tail_on) {
#if SMAUG_SPLIT_LATELOAD == 1 || SMAUG_SPLIT_LATELOAD == 2
        if (COMBINE == COMBINE_FINAL) {
#pragma unroll
          for (int f = 0; f < NF; ++f) { jin[f] = a.in.p[f][gj]; jacc[f] = a.acc_in.p[f][gj]; }
        } else {
#pragma unroll
          for (int f = 0; f < NF; ++f) jbase[f] = a.base.p[f][gj];
          if (COMBINE == COMBINE_ACC) {
#pragma unroll
            for (int f = 0; f < NF; ++f) jin[f] = a.in.p[f][gj];
          }
        }
#endif
        const double* cx = CXR + s5 * 5 * PW + tp;
        double R[NF];
        {
          double cdx[5];
#pragma unroll
          for (int f = 0; f < 5; ++f) cdx[f] = cd12v(cx[f * PW - 2], cx[f * PW - 1], cx[f * PW + 1], cx[f * PW + 2]);
          R[F_RHO] = fma(cdx[C_RHO], idx_, cdyi[C_RHO]) * (-1.0 / 12.0);
          R[F_MX] = fma(cdx[C_MX], idx_, cdyi[C_MX]) * (-1.0 / 12.0);
          R[F_MY] = fma(cdx[C_MY], idx_, cdyi[C_MY]) * (-1.0 / 12.0);
          R[F_E] = fma(cdx[C_E], idx_, cdyi[C_E]) * (-1.0 / 12.0);
          R[F_BX] = cdyi[C_B] * (-1.0 / 12.0);
          R[F_BY] = fma(cdx[C_B], idx_, 0.0) * (-1.0 / 12.0);
        }
        if constexpr (BG) {
          // energy source S_e = -p_tb div v + B_b B_b : grad v (c-2) at the tail cell; then gravity (c-10)
          const double* vxj = VJ + (vjb * 2 + 0) * PW + tp;
          const double* vyj = VJ + (vjb * 2 + 1) * PW + tp;
          const double dxvx = (cd12v(vxj[-2], vxj[-1], vxj[1], vxj[2]) * idx_) * (1.0 / 12.0);
          const double dxvy = (cd12v(vyj[-2], vyj[-1], vyj[1], vyj[2]) * idx_) * (1.0 / 12.0);
          const double dyvx = (cd12v(hvx[0], hvx[1], hvx[3], hvx[4]) * idy_) * (1.0 / 12.0);
          const double dyvy = (cd12v(hvy[0], hvy[1], hvy[3], hvy[4]) * idy_) * (1.0 / 12.0);
          const double bb2h = 0.5 * fma(Bby0, Bby0, Bbx0 * Bbx0);
          const double ptb = fma(gm1y, eb0 - bb2h, bb2h);
          const double S = fma(-ptb, dxvx + dyvy,
                               fma(Bby0 * Bby0, dyvy, fma(Bbx0 * Bby0, dxvy + dyvx, (Bbx0 * Bbx0) * dxvx)));
          R[F_E] = R[F_E] + S;
          if (a.prm.grav_on) {
            const double rt = hr[2];
            R[F_MX] = fma(rt, a.prm.gx, R[F_MX]);
            R[F_MY] = fma(rt, a.prm.gy, R[F_MY]);
            R[F_E] = fma(rt, fma(a.prm.gy, hvy[2], a.prm.gx * hvx[2]), R[F_E]);
          }
        }
        if constexpr (!BG && GRAV) {      // gravity on a zero background (c-10: rho~ is the total density)
          const double rt = hr[2];
          R[F_MX] = fma(rt, a.prm.gx, R[F_MX]);
          R[F_MY] = fma(rt, a.prm.gy, R[F_MY]);
          R[F_E] = fma(rt, fma(a.prm.gy, hvy[2], a.prm.gx * hvx[2]), R[F_E]);
        }
        const double* dx = DXR + s4 * 5 * NC + c;
        R[F_RHO] = fma(dx[C_RHO * NC], idx_, R[F_RHO]);
        R[F_MX] = fma(dx[C_MX * NC], idx_, R[F_MX]);
        R[F_MY] = fma(dx[C_MY * NC], idx_, R[F_MY]);
        R[F_E] = fma(dx[C_E * NC], idx_, R[F_E]);
        R[F_BY] = fma(dx[C_B * NC], idx_, R[F_BY]);
        R[F_RHO] = fma(py[C_RHO] - py_prev[C_RHO], idy_, R[F_RHO]);
        R[F_MX] = fma(py[C_MX] - py_prev[C_MX], idy_, R[F_MX]);
        R[F_MY] = fma(py[C_MY] - py_prev[C_MY], idy_, R[F_MY]);
        R[F_E] = fma(py[C_E] - py_prev[C_E], idy_, R[F_E]);
        R[F_BX] = fma(py[C_B] - py_prev[C_B], idy_, R[F_BX]);
        double o[NF];
        if (COMBINE == COMBINE_FINAL) {
#pragma unroll
          for (int f = 0; f < NF; ++f) o[f] = fma(cdt, R[f], fma(fma(-2.0, jin[f], jacc[f]), 1.0 / 3.0, jin[f]));
        } else {
#pragma unroll
          for (int f = 0; f < NF; ++f) o[f] = fma(cdt, R[f], jbase[f]);
        }
        if (col_out && j < yend) {
          const unsigned go = gj;      // an output column has cl == ci
#pragma unroll
          for (int f = 0; f < NF; ++f) a.out.p[f][go] = o[f];
          if (COMBINE == COMBINE_ACC) {
#pragma unroll
            for (int f = 0; f < NF; ++f) a.acc_out.p[f][go] = fma(2.0, o[f], jin[f] - jbase[f]);
          }
          if (WS != WS_NONE) {
            double thr0 = wsmax[0], thr1 = wsmax[1];
            if (WS == WS_FULL) {
              thr0 = gthr0 > thr0 ? gthr0 : thr0;
              thr1 = gthr1 > thr1 ? gthr1 : thr1;
            }
            if constexpr (BG) {
              const double ot[NF] = {rb0 + o[F_RHO], o[F_MX], o[F_MY], eb0 + o[F_E], Bbx0 + o[F_BX], Bby0 + o[F_BY]};
              split_wavespeeds<WS>(ot, gamma, wsmax, thr0, thr1);
            } else {
              split_wavespeeds<WS>(o, gamma, wsmax, thr0, thr1);
            }
          }
        }
      }
#pragma unroll
      for (int f = 0; f < 5; ++f) py_prev[f] = py[f];
      kyv_prev = kyv; kyb_prev = kyb;
      if (tail_on) gj += upitch;
      s4 = s4 == ND - 1 ? 0 : s4 + 1;
      s5 = s5 == 4 ? 0 : s5 + 1;
      s6 = s6 == NY - 1 ? 0 : s6 + 1;
      if (!DEC) par ^= 1;
      if constexpr (TM) {
        p5 = p5 == 4 ? 0 : p5 + 1;
        yst ^= 1;
      }
      if constexpr (BG) vjb ^= 1;
    }
  }
  if (WS != WS_NONE) {
    __syncthreads();      // red_sh aliases the landing zone of the X warps
    block_max4_atomic(wsmax, red_sh, a.sc->red[a.red_out], WS == WS_FULL ? 0 : 2);
  }
  if constexpr (TM) {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (tid < 32)
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm_base), "n"(SPLIT_TMEM_COLS) : "memory");
  }
}

}  // namespace smaug
