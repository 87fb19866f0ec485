/* smaug3d.h -- C ABI of the three-dimensional form of the SMAUG+ hot path.
 *
 * What the library computes (PAPER.md = /root/reference/PAPER.md; readings: DESIGN.md section 3):
 *   PAPER.md:33 "the 3-dimensional MHD equations", "implemented in 3D": one full time step of the scheme of
 *   smaug.h on an nx x ny x nz grid -- the ideal-MHD fluxes of PAPER.md:35-43 for the eight fields
 *   w = (rho, mx, my, mz, e, bx, by, bz), fourth-order central differences (c-3), hyperdiffusion and
 *   hyper-resistivity along all three axes with the coefficient of PAPER.md:45-49 (c-5, and c-11 for the terms that
 *   exist only in three dimensions), classical RK4 / midpoint / Euler (c-6), ghost fill periodic / open / fixed on six
 *   sides (c-8), the maximum wave speeds and the CFL step over three axes (c-4, c-7), uniform gravity (c-10).
 *   Zero background only (the split form with a stratified background is built in two dimensions: smaug.h).
 * Every step runs in fp64 CUDA kernels for sm_100a (smaug3d.cu); there is no CPU fallback: smaug3_create fails
 * with SMAUG3_ECUDA when no CUDA device is usable.
 *
 * Conventions (as smaug.h unless stated)
 *   - state w [8][nz][ny][nx], fp64, x fastest, INTERIOR CELLS ONLY, order rho, mx, my, mz, e, bx, by, bz.  Pointers may
 *     be HOST or DEVICE memory (copies are cudaMemcpyDefault); the caller owns them; nothing is retained.
 *   - bc[6] = x_lo, x_hi, y_lo, y_hi, z_lo, z_hi, each SMAUG3_BC_*; periodic must be set on both sides of an axis.
 *   - cell centres x_i = (i + 1/2) Lx / nx, likewise y, z; Lx = Ly = Lz = 1 by default; ghost width 3.
 *   - a context lives on the device current at smaug3_create and owns its device memory (cudaMalloc; about
 *     94 padded volumes of (nx + 19 rounded up to 16) x (ny + 6) x (nz + 6) doubles -- smaug3_workspace_bytes tells);
 *     every entry point makes that device current for the call and restores the caller's.
 *   - all work is enqueued on the stream given at creation (0 = the legacy default stream); smaug3_step,
 *     smaug3_get_state, smaug3_get_time and smaug3_get_wavespeeds synchronise it before returning.
 *   - return value 0 = SMAUG3_OK, negative = error, message in smaug3_last_error() (thread-local).  No exception
 *     crosses the ABI.  A context is not thread-safe.
 *   - NaN behaviour: the maxima skip NaNs (c-4), so a NaN state leaves dt finite; SMAUG3_ENONFINITE reports a
 *     non-finite or non-positive time step only.
 */
#ifndef SMAUG3D_H_
#define SMAUG3D_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct smaug3_ctx smaug3_ctx; /* opaque, library-owned */

enum { SMAUG3_BC_PERIODIC = 0, SMAUG3_BC_OPEN = 1, SMAUG3_BC_FIXED = 2 };
enum { SMAUG3_OK = 0, SMAUG3_EINVAL = -1, SMAUG3_ENOMEM = -2, SMAUG3_ECUDA = -3, SMAUG3_ENONFINITE = -4 };

enum { /* keys of smaug3_set_param: 0..11 mean what they mean in smaug.h */
  SMAUG3_PARAM_LX = 0, SMAUG3_PARAM_LY = 1,
  SMAUG3_PARAM_HD_ON = 2,    /* 0: no hyperdiffusion; else on (default) */
  SMAUG3_PARAM_C_RHO = 3, SMAUG3_PARAM_C_MOM = 4, SMAUG3_PARAM_C_E = 5, SMAUG3_PARAM_C_B = 6, /* defaults 0.02 0.4 0.02 0.02 */
  SMAUG3_PARAM_RK_ORDER = 7, /* 4 (default), 2, 1 */
  SMAUG3_PARAM_FIXED_DT = 8, /* > 0: this dt instead of the CFL step */
  SMAUG3_PARAM_GX = 10, SMAUG3_PARAM_GY = 11,
  SMAUG3_PARAM_LZ = 13,      /* domain length in z, > 0 (default 1) */
  SMAUG3_PARAM_GZ = 14,      /* third component of the uniform gravitational acceleration */
  SMAUG3_PARAM_KERNEL = 15   /* 1 (default): cell-centred fluxes and assembly fused in one kernel (C_d in shared memory);
                                0: two kernels with the C_d volumes in HBM.  Same bits; the switch is for tests / profiling */
};

/* Thread-local message of the last failed call (never NULL). */
const char* smaug3_last_error(void);

/* Device bytes a context of this size allocates. */
size_t smaug3_workspace_bytes(int nx, int ny, int nz);

/* Create a context on the current device.  nx, ny, nz >= 1 (an axis with one cell is excluded from the CFL minimum,
 * c-7); gamma > 1; bc[6] as above; stream: a cudaStream_t passed as void* (NULL = legacy default stream).
 * Errors: EINVAL (arguments; a padded volume of 2^31 elements or more), ENOMEM, ECUDA. */
int smaug3_create(int nx, int ny, int nz, double gamma, const int bc[6], void* stream, smaug3_ctx** out);

/* Free the context and its device memory (NULL is allowed). */
void smaug3_destroy(smaug3_ctx* ctx);

/* Set a parameter (keys above).  EINVAL for an unknown key or a value out of range. */
int smaug3_set_param(smaug3_ctx* ctx, int key, double value);

/* Load the state w[8][nz][ny][nx] (host or device), fill the ghost cells (fixed sides are frozen here at the
 * nearest interior value), reduce the wave-speed maxima, reset t to 0. */
int smaug3_set_state(smaug3_ctx* ctx, const void* w);

/* Advance n_steps time steps with dt = cfl min_d(Delta_d / cmax_d) (or the fixed dt): per step one dt launch and,
 * per RK stage, ghost fill (state and derived quantities) -> kappa / interface fluxes along x, y, z -> cell-centred
 * fluxes C_d = F_d - G_d, assembly, RK combine, derived quantities of the result and wave-speed reduction (one tile
 * kernel; SMAUG3_PARAM_KERNEL = 0: two kernels).  dt and the maxima stay on the device.
 * ENONFINITE if a time step was non-finite or <= 0. */
int smaug3_step(smaug3_ctx* ctx, int n_steps, double cfl);

/* Copy the state into w[8][nz][ny][nx] (host or device). */
int smaug3_get_state(smaug3_ctx* ctx, void* w);

/* Simulated time and the last time step (either pointer may be NULL). */
int smaug3_get_time(smaug3_ctx* ctx, double* t, double* last_dt);

/* out[5] = max(|vx| + c_f,x), max(|vy| + c_f,y), max(|vz| + c_f,z), max a^2, max b^2 of the current state (c-4). */
int smaug3_get_wavespeeds(smaug3_ctx* ctx, double out[5]);

/* Kernel launches enqueued by this context so far. */
int smaug3_get_launch_count(smaug3_ctx* ctx, long long* n);

/* Per-kernel timing with CUDA events on the context's stream (for bench.py's roofline pass): on != 0 starts a fresh
 * accumulation.  smaug3_get_kernel_timing synchronises and returns, for the kinds 0 ghost fill, 1 derived quantities,
 * 2 kappa / interface fluxes, 3 cell-centred fluxes, 4 assembly, the accumulated milliseconds ms[5] and launch
 * counts n[5]. */
int smaug3_set_kernel_timing(smaug3_ctx* ctx, int on);
int smaug3_get_kernel_timing(smaug3_ctx* ctx, double ms[5], long long n[5]);

#ifdef __cplusplus
}
#endif
#endif /* SMAUG3D_H_ */
