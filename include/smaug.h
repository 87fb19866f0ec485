/* smaug.h -- C ABI of the B200-native SMAUG+ hot path: one full 2-D MHD time step on one GPU.
 *
 * What the library computes (citations: /root/reference/PAPER.md = "PAPER.md"; DESIGN.md section 3 lists
 * every reading "c-1".."c-9" taken where the paper is silent):
 *   - the SAC/VAC-style split ideal-MHD right-hand side for the perturbed variables
 *     w = (rho~, mx, my, e~, bx~, by~) on a static background (rho_b, e_b, Bbx, Bby)   PAPER.md:35-43, c-2
 *   - 4th-order central differences of the flux components                                PAPER.md:45,    c-3
 *   - hyperdiffusion / hyper-resistivity with the coefficient "ratio of the forward
 *     difference ... to third order and first order" times the max wave speed             PAPER.md:45-49, c-5
 *   - the Runge-Kutta stage updates (classical RK4; 2 = midpoint, 1 = Euler)              PAPER.md:45,    c-6
 *   - ghost-cell (halo) fill, periodic / open / fixed, in device memory                   PAPER.md:59,101, c-8
 *   - the max-wavespeed reduction and the CFL time step                                   PAPER.md:45,    c-4, c-7
 *   - uniform gravity acting on the perturbed density (stratified backgrounds)           PAPER.md:35,    c-10
 * Every step of that path runs in hand-written fp64 CUDA kernels for sm_100a; there is no CPU fallback
 * (every entry point fails with SMAUG_ECUDA when no CUDA device is usable).
 *
 * Conventions
 *   - Arrays are fp64, SoA, field-major, row-major with x fastest, INTERIOR CELLS ONLY:
 *       state      w  [6][ny][nx]  order rho~, mx, my, e~, bx~, by~
 *       background bg [4][ny][nx]  order rho_b, e_b, Bbx, Bby          (NULL = zero background)
 *     Pointers may be HOST or DEVICE memory (unified addressing: the copies are cudaMemcpyDefault); the
 *     caller owns them and the library copies; nothing is retained after the call returns.
 *   - Device: a context lives on the device of its workspace (smaug_create: the device current at the call);
 *     every entry point makes that device current for the duration of the call and restores the caller's.
 *   - Grid: cell centres x_i = (i+1/2) Lx/nx, y_j = (j+1/2) Ly/ny; Lx = Ly = 1 by default.  Ghost width 3.
 *   - Return value: 0 = SMAUG_OK, negative = error; smaug_last_error() gives a thread-local message.
 *     No exception crosses the ABI.  No global state except that message.
 *   - A context is not thread-safe; use one context per host thread (or lock).
 *   - All work is enqueued on the context's stream (default: the legacy default stream 0; pass torch's
 *     current stream with smaug_set_stream).  smaug_step / smaug_get_state / smaug_get_time synchronise
 *     that stream before returning; smaug_step_async does not.
 */
#ifndef SMAUG_H_
#define SMAUG_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct smaug_ctx smaug_ctx;     /* opaque, library-owned */
typedef struct smaug_group smaug_group; /* opaque: a px x py decomposition of one grid into contexts (see below) */

enum { SMAUG_BC_PERIODIC = 0, SMAUG_BC_OPEN = 1, SMAUG_BC_FIXED = 2 };

enum {
  SMAUG_OK = 0,
  SMAUG_EINVAL = -1,    /* bad argument: nx<1, ny<1, gamma<=1, unknown bc, periodic on one side only, NULL */
  SMAUG_ENOMEM = -2,    /* device allocation failed / workspace too small */
  SMAUG_ECUDA = -3,     /* CUDA runtime error (message in smaug_last_error), incl. "no device" */
  SMAUG_ENONFINITE = -4 /* a time step was non-finite or <= 0; the state is then unspecified */
};

enum { /* keys of smaug_set_param */
  SMAUG_PARAM_LX = 0,       /* domain length in x, > 0 (default 1) */
  SMAUG_PARAM_LY = 1,       /* domain length in y, > 0 (default 1) */
  SMAUG_PARAM_HD_ON = 2,    /* 0 = no hyperdiffusion ("Without HD" column of PAPER.md Table 1), else on (default) */
  SMAUG_PARAM_C_RHO = 3,    /* hyperdiffusion coefficients c_u of c-5, >= 0; defaults 0.02, */
  SMAUG_PARAM_C_MOM = 4,    /*   0.4, */
  SMAUG_PARAM_C_E = 5,      /*   0.02, */
  SMAUG_PARAM_C_B = 6,      /*   0.02 */
  SMAUG_PARAM_RK_ORDER = 7, /* 4 (default), 2 (midpoint) or 1 (forward Euler) */
  SMAUG_PARAM_FIXED_DT = 8, /* > 0: use this dt instead of the CFL step; 0 (default): CFL */
  SMAUG_PARAM_KERNEL = 9,   /* which fused stage kernel runs.  2 (default): the fastest applicable form -- the role-split
                               streaming kernel (hyperdiffusion on), the streaming flux kernel (off), and for a
                               one-dimensional problem (ny = 1, nx <= 976, y-boundary not fixed, no background, RK4 / RK2) the small-grid path:
                               whole time steps in one persistent cluster launch.  3: as 2 without the small-grid path.
                               1: single-role streaming kernel where applicable (no background).  0: always the tiled
                               kernel.  All forms are bit-identical; the switch exists for tests and profiling. */
  SMAUG_PARAM_GX = 10,      /* uniform gravitational acceleration g = (GX, GY) of PAPER.md:35 ("rho g", "rho g.v"); */
  SMAUG_PARAM_GY = 11,      /*   default 0.  Split form (c-10): the background is taken to be in magneto-hydrostatic
                               balance  grad p_tb - (B_b.grad)B_b = rho_b g,  so gravity acts on the perturbed
                               density: S(m) = rho~ g, S(e~) = rho~ g.v.  With a zero background rho~ is the total
                               density and these are the printed source terms.  Any finite value. */
  SMAUG_PARAM_GRAPH = 12    /* 1 (default): smaug_step replays whole time steps as CUDA graphs (captured on first use for
                               calls of >= 8 steps, re-captured when a parameter, the stream or cfl changes);
                               0: plain kernel launches.  Same kernels, same results; only the launch path differs. */
};

/* Bytes of device memory a context for an nx-by-ny grid needs (has_bg != 0: a background is given).
 * Returns 0 if nx or ny is < 1. */
size_t smaug_workspace_bytes(int nx, int ny, int has_bg);

/* Create a context.  bc = {x_lo, x_hi, y_lo, y_hi}; periodic must be set on both sides of an axis.
 * bg: background [4][ny][nx] (host or device) or NULL.  Its ghosts are filled once (periodic -> wrap,
 * else nearest interior cell).  The library allocates device memory with cudaMalloc. */
int smaug_create(int nx, int ny, double gamma, const int bc[4], const double* bg, smaug_ctx** out);

/* Same, but all device memory is carved out of `workspace` (DEVICE pointer, 256-byte aligned, at least
 * smaug_workspace_bytes(nx, ny, bg != NULL) bytes, e.g. a torch uint8 tensor) which the caller keeps
 * alive until smaug_destroy.  `stream` is a cudaStream_t (NULL = default stream). */
int smaug_create_in_workspace(int nx, int ny, double gamma, const int bc[4], const double* bg,
                              void* workspace, size_t workspace_bytes, void* stream, smaug_ctx** out);

/* cudaStream_t on which all later work of this context is enqueued. */
int smaug_set_stream(smaug_ctx* ctx, void* stream);

int smaug_set_param(smaug_ctx* ctx, int key, double value);

/* Load the perturbed state w [6][ny][nx] (host or device), fill its ghosts (fixed sides are frozen at
 * the nearest-interior value from now on), reduce its wave-speed maxima, reset t = 0. */
int smaug_set_state(smaug_ctx* ctx, const double* w);

/* Advance n_steps time steps: per step  dt = cfl * min_d(Delta_d / cmax_d)  (c-7; an axis with n = 1 is
 * excluded; or SMAUG_PARAM_FIXED_DT), then the RK stages, each = ghost fill + fused RHS/hyperdiffusion/
 * RK-combine/wavespeed-reduction kernel.  dt and the maxima stay on the device; the host synchronises
 * once, at the end, to read the status.  Returns SMAUG_ENONFINITE if any dt was non-finite or <= 0.
 * Non-finite CELLS are not detected as such: the wave-speed maxima start at 0 and skip NaNs and negative values
 * (c-4), so a local blow-up (NaN cells, negative pressure) leaves dt finite and the call returns SMAUG_OK with a
 * state that contains NaNs; callers that need the check test the state they read back.  Bit-identity with the
 * oracle is claimed for finite states only. */
int smaug_step(smaug_ctx* ctx, int n_steps, double cfl);

/* Same, but only enqueues the work; the status is picked up by the next synchronising call. */
int smaug_step_async(smaug_ctx* ctx, int n_steps, double cfl);

/* Copy the perturbed state out, [6][ny][nx] (host or device). */
int smaug_get_state(smaug_ctx* ctx, double* w);

/* Simulated time and the last dt used (either pointer may be NULL). */
int smaug_get_time(smaug_ctx* ctx, double* t, double* last_dt);

/* out = { max(|vx|+c_fx), max(|vy|+c_fy), max a^2, max b^2 } of the current state (c-4). */
int smaug_get_wavespeeds(smaug_ctx* ctx, double out[4]);

/* Number of kernels this context has launched so far (for bench.py's gpu_launches). */
int smaug_get_launch_count(smaug_ctx* ctx, long long* n);

/* Algorithmic / launch facts of the fused stage kernel, for the roofline report:
 * out = { tile_w, tile_h, threads, dynamic_smem_bytes, ctas_last_launch }; the streaming kernel reports
 * its strip width as tile_w and 1 as tile_h (it marches row by row). */
int smaug_get_kernel_info(smaug_ctx* ctx, int out[5]);

/* Name of the fused stage kernel the context's current parameters select (static string, never NULL;
 * "?" for a NULL context): "split_kernel<128>" (role-split streaming form), "march_kernel<256>"
 * (single-role streaming form), "flux_kernel<128>" or "flux_kernel<256>" (streaming form without hyperdiffusion; the
 * strip width is picked per grid),
 * "line_step_kernel<128>" (small-grid path) or "stage_kernel<32,8,512>" (tiled form: SMAUG_PARAM_KERNEL = 0). */
const char* smaug_get_kernel_name(smaug_ctx* ctx);

/* Device time, in milliseconds, spent in the fused stage kernels (summed over launches) and the number of
 * those launches, measured with CUDA events on the context's stream when enabled with
 * smaug_set_kernel_timing(ctx, 1).  Reading synchronises the stream.  */
int smaug_set_kernel_timing(smaug_ctx* ctx, int on);
int smaug_get_kernel_timing(smaug_ctx* ctx, double* stage_ms, long long* stage_launches);

/* Exactness self-test of the library's branch-free fp64 division helpers ("Division"): on
 * about `draws` seeded operand sets with binary exponents uniform in [exp_lo, exp_hi] (values below 2^-1022 are
 * denormals), counts the results that differ in any bit from the compiler's IEEE-754 `/`:
 *   out[0] ddiv(a, b) vs a / b,   out[1] drcp(b) vs 1 / b,   out[2] ratio_div(m3, m1) vs m3 / m1 and
 *   out[3] kappa_ratio(m3, m1, cv) vs (m1 > 0 ? cv * (m3 / m1) : 0) on ratio-like operands 0 <= m3 <= 4 m1 (incl.
 *   m1 = 0),   out[4] = draws actually made per test.
 * The stage kernels call ddiv / drcp on ordinary numbers only and route every hyperviscosity ratio through
 * kappa_ratio (or its fast path, taken only when every M1 of the warp is >= 2^-923).  Runs on the current device. */
int smaug_selftest_division(int exp_lo, int exp_hi, unsigned long long seed, long long draws, unsigned long long out[5]);

/* fp64-pipe micro-benchmark on the current device (the measurement behind DESIGN.md section 5's "one fp64 warp instruction
 * per two cycles and SM sub-partition, dependent latency 9 cycles"): every warp of a grid of one CTA per SM with
 * 128 * warps_per_subpartition threads runs `iters` trips of `ilp` (1, 2, 4 or 8) independent dependent-DFMA chains.
 * out[0] = clock cycles per warp instruction and sub-partition, out[1] = cycles per trip (the chain latency while the
 * pipe is not saturated).  Errors: EINVAL, ECUDA.  tests/test_gpu_division.py prints and bounds both. */
int smaug_selftest_fp64_pipe(int ilp, int warps_per_subpartition, int iters, double out[2]);

/* ---- Wave-speed maxima without any device allocation --------------------------------------------------------------
 * out = { max(|vx|+c_fx), max(|vy|+c_fy), max a^2, max b^2 } (c-4; "maximum wave speed") of a state the
 * caller already holds on the device -- the numbers a CFL monitor or an output routine wants -- bit for bit what
 * smaug_set_state + smaug_get_wavespeeds return for the same arrays.
 *
 * Who this is for: a caller that cannot call cudaMalloc, directly or through this library.  The usual cases are a
 * process whose GPU memory belongs to somebody else's allocator (a framework's caching pool or a job-wide arena has
 * reserved the device, so a raw cudaMalloc fails or breaks the memory budget) and a time-critical loop that must not
 * take cudaMalloc / cudaFree's device-wide synchronisation.  The context route needs a workspace of some 24 padded
 * planes (over 12 GB at 8000 x 8000) just to own four reduction slots; this call needs none: its working memory is a
 * 524,544-byte array inside the library image, which every GPU that loads libsmaug.so holds until the process exits.
 * It calls neither cudaMalloc nor cudaFree nor any routine that allocates.
 *
 * Arguments: w [6][ny][nx] and bg [4][ny][nx] (NULL = zero background) are DEVICE pointers in the layout above,
 * out is a DEVICE pointer to 4 doubles; all three stay the caller's.  Host pointers are refused (SMAUG_EINVAL): there
 * is nowhere to stage them.  The work is enqueued on `stream` (a cudaStream_t, NULL = default stream) of the CURRENT
 * device and the call returns without waiting: out is valid once that stream reaches the end of the kernel.
 * Limit: nx * ny <= SMAUG_WAVESPEEDS_STATIC_MAX_CELLS (the array holds four partial maxima per block of 4096 cells);
 * larger grids are refused with SMAUG_EINVAL and a message that names the limit.
 * First call on each device: looks up the array's device address (cudaGetSymbolAddress), so make that first call
 * outside any stream capture; later calls on that device reuse the address.
 * Sharing: all calls in the process use the same array, which keeps the last call's contents.  The one word that
 * must start at zero is cleared on `stream` before each launch, so calls that are ordered on the GPU (one stream, or
 * streams joined by events) are independent of each other; calls that can OVERLAP on the GPU race on the array and
 * give undefined results -- serialise them.  Not for use from several host threads at once on one device either.
 * As in smaug_get_wavespeeds, NaN and negative candidates are skipped (maxima start at 0). */
#define SMAUG_WAVESPEEDS_STATIC_MAX_CELLS 67108864LL /* 16384 blocks x 4096 cells; 8000 x 8000 fits, 8192 x 8193 does not */
int smaug_wavespeeds_static(int nx, int ny, double gamma, const double* w, const double* bg, double* out, void* stream);

void smaug_destroy(smaug_ctx* ctx); /* NULL is a no-op */

/* ---- Domain decomposition (SURVEY.md 8(f) NEXT-1; PAPER.md:25 Fig. 1, :55-59 "the full domain is divided into
 * sub-regions", :61-73 exchange_halo) ----------------------------------------------------------------------------
 * A group splits the nx-by-ny grid into px x py near-equal blocks (block column a covers global columns
 * [a nx / px, (a+1) nx / px), rows likewise), one context per block, member b * px + a on device devices[b * px + a]
 * (devices == NULL: all on the current device; distinct devices need peer access to each other).  The paper's
 * exchange_halo (gather -> D2H -> MPI_Isend/Irecv -> H2D -> scatter per field) becomes one small kernel per member and
 * RK stage that PULLS the member's ghost cells (width 3, 6 fields, corners included) straight out of the owning
 * neighbours' planes (peer pointers: same-device pointers on one GPU, NVLink P2P mappings across GPUs); the global
 * boundary kinds `bc` (periodic / open / fixed, as in smaug_create) are applied on the global grid.  The four
 * wave-speed maxima (c-4) are reduced by every member's stage kernels into the leader's slots with atomicMax, so dt
 * and v_t are global (the paper's implied MAX all-reduce).  Members step in lockstep: per stage, all exchanges run
 * after all members' previous stage (events between the members' streams), then all stage kernels.
 * Contract: a decomposed run is BIT-IDENTICAL to the single-context run of the same global problem.
 * Status of the several-GPU form: EXPERIMENTAL.  With all members on one device the contract is tested (tests/
 * test_gpu_group.py).  With distinct devices the same kernels run over peer mappings and the reduction uses system-scope
 * atomics (atomicMax_system: a device-scope atomic is atomic among the threads of one GPU only), but that path has not
 * run on hardware yet; its test is collected only where two GPUs are visible.
 * State / background arrays are the GLOBAL ones, [6][ny][nx] / [4][ny][nx], host or device; the group scatters and
 * gathers the blocks.  All group calls synchronise before returning.  Errors as for the context calls. */
int smaug_group_create(int px, int py, int nx, int ny, double gamma, const int bc[4], const double* bg,
                       const int* devices, smaug_group** out);
int smaug_group_size(smaug_group* grp, int* px, int* py);
int smaug_group_set_param(smaug_group* grp, int key, double value);   /* forwarded to every member; LX, LY are global */
int smaug_group_set_state(smaug_group* grp, const double* w);
int smaug_group_step(smaug_group* grp, int n_steps, double cfl);
int smaug_group_get_state(smaug_group* grp, double* w);
int smaug_group_get_time(smaug_group* grp, double* t, double* last_dt);
int smaug_group_get_wavespeeds(smaug_group* grp, double out[4]);
/* kernels launched so far: stage / dt / reduction kernels of all members, and exchange (halo) kernels */
int smaug_group_get_launch_count(smaug_group* grp, long long* stage_and_aux, long long* exchange);
/* The paper's load-balance measure: T = T_comp + T_comm + T_idle and tau = ln(T_comp / (T_comm + T_idle)).
 * smaug_group_set_timing(grp, 1) starts recording CUDA events on every member's stream (and clears what was recorded);
 * smaug_group_get_tau returns out = { T_comp, T_comm, T_idle, tau }, times in milliseconds, mean over the members, of all
 * steps since then:  T_comm = the halo-pull kernels (the whole of the paper's exchange_halo),  T_comp = the stage kernels
 * (and the leader's dt kernel),  T_idle = what a member's stream spends in the inter-member barriers after its own work
 * is done.  With all members on ONE device they share its SMs, so a member's intervals contain the time its kernels
 * wait for, or share the device with, the other members' kernels: the three terms then sum to the wall time of the
 * steps, and tau describes the lockstep schedule, not a communication link.  Both calls synchronise.  0 = timing off. */
int smaug_group_set_timing(smaug_group* grp, int on);
int smaug_group_get_tau(smaug_group* grp, double out[4]);
void smaug_group_destroy(smaug_group* grp); /* destroys the members too; NULL is a no-op */
/* Host-only view of the decomposition logic (needs no GPU; used by the CPU tests): for ghost cell (i, j) -- local
 * indices outside [0, nx_m) x [0, ny_m) -- of member `member`, out = { x0, y0, nx_m, ny_m of the member,  source member
 * (-1: the cell is never rewritten: fixed global side, freeze == 0),  source local i,  source local j }. */
int smaug_group_map_cell(int px, int py, int nx, int ny, const int bc[4], int member, int i, int j, int freeze, int out[7]);

const char* smaug_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SMAUG_H_ */
