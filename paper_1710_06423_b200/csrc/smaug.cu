// smaug.cu -- host side of libsmaug.so: the C ABI of include/smaug.h, device memory layout, the launch sequence of
// one time step (plain launches, CUDA-graph replays, the one-launch path of 1-D problems) and the decomposition
// groups.  No torch types, no CPU fallback: every numerical step is a kernel from smaug_aux_kernels.cuh and the stage
// kernels smaug_split_kernel.cuh / smaug_flux_kernel.cuh / smaug_line_kernel.cuh (second implementations:
// smaug_stage_kernel.cuh, smaug_march_kernel.cuh).
#include "../../include/smaug.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "smaug_flux_kernel.cuh"
#ifndef SMAUG_PRODUCT_ONLY             // -DSMAUG_PRODUCT_ONLY: a library without the two second implementations
#include "smaug_march_kernel.cuh"      // (SMAUG_PARAM_KERNEL = 0 / 1 is then refused); the default build carries them:
#include "smaug_stage_kernel.cuh"      // the parity tests run every form against the oracle and against each other
#endif
#include "smaug_selftest.cuh"
#include "smaug_group.cuh"
#include "smaug_line_kernel.cuh"

using namespace smaug;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}

#define CU(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess)                                                                         \
      return fail(SMAUG_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));                \
  } while (0)

// Tile / launch configuration of the fused stage kernel.
#ifndef SMAUG_TW
#define SMAUG_TW 32
#endif
#ifndef SMAUG_TH
#define SMAUG_TH 8
#endif
#ifndef SMAUG_NT
#define SMAUG_NT 512
#endif
constexpr int TW = SMAUG_TW, TH = SMAUG_TH, NT = SMAUG_NT;

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Makes the context's device current for the duration of an ABI call and restores the caller's afterwards.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE attribute of a kernel: set it once per
// (kernel instantiation, device).  `mask` is the instantiation's own static bit set of configured devices.
template <typename K>
cudaError_t configure_smem(K kern, size_t smem, int device, unsigned long long& mask) {
  if (device >= 0 && device < 64 && (mask >> device & 1ULL)) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess && device >= 0 && device < 64) mask |= 1ULL << device;
  return e;
}

struct Layout {
  int pitch;
  long long plane;          // doubles
  size_t state_bytes;       // one buffer of 6 planes
  size_t bg_bytes;
  size_t scalars_off, bufs_off[4], bg_off, total;
};

Layout make_layout(int nx, int ny, bool has_bg) {
  Layout L;
  L.pitch = (int)align_up((size_t)XOFF + nx + NG, 16);
  L.plane = (long long)L.pitch * (ny + 2 * NG);
  const size_t plane_bytes = align_up((size_t)L.plane * sizeof(double), 256);
  L.state_bytes = NF * plane_bytes;
  L.bg_bytes = has_bg ? NBG * plane_bytes : 0;
  size_t off = 0;
  L.scalars_off = off; off += align_up(sizeof(DeviceScalars), 256);
  for (int b = 0; b < 4; ++b) { L.bufs_off[b] = off; off += L.state_bytes; }
  L.bg_off = off; off += L.bg_bytes;
  L.total = off;
  return L;
}

}  // namespace

struct smaug_ctx {
  Grid g;
  double gamma = 0;
  double Lx = 1, Ly = 1;
  int hd_on = 1;
  double c_rho = 0.02, c_mom = 0.4, c_e = 0.02, c_b = 0.02;
  int rk_order = 4;
  double fixed_dt = 0;
  double gx = 0, gy = 0;    // uniform gravity (c-10)
  bool has_bg = false;
  Layout L;
  char* base = nullptr;     // device workspace
  bool owns = false;
  cudaStream_t stream = nullptr;
  DeviceScalars* sc = nullptr;
  Planes6 buf[4];           // buf[0] holds the state between steps; 1, 2: stage buffers; 3: accumulator
  CPlanes4 bg;
  int state_set = 0;        // reduction set holding the maxima of the state (0 or 4)
  long long launches = 0;
  int last_ctas = 0;
  // stage-kernel timing (CUDA events on the stream)
  bool timing = false;
  std::vector<cudaEvent_t> ev;   // pairs
  size_t ev_used = 0;
  double stage_ms = 0;
  long long stage_launches = 0;
  bool pending_status = false;
  int kernel_mode = 2;      // SMAUG_PARAM_KERNEL: 2 role-split streaming kernel, 1 single-role streaming kernel
                            // (both only without background and with hyperdiffusion), 0 always the tile kernel
  int n_sm = 148;
  long long line_stage_equiv = 0;   // stages run inside line launches beyond the one the event pair counts (timing)
  bool line_ok = true;      // cleared if the device refuses the cluster launch of the small-grid path
  int device = 0;           // the device the workspace lives on; every ABI entry makes it current (DeviceGuard)
  // member of a decomposition group (smaug_group_*): the GLOBAL cell counts fix Delta and the n = 1 rule of c-7, the
  // reduction slots / dt / t / status are the group leader's, the ghost fill is the group's exchange kernel
  smaug_group* group = nullptr;
  int geo_nx = 0, geo_ny = 0;     // global interior size (= g.nx, g.ny outside a group)
  DeviceScalars* own_sc = nullptr;
  double* bg_owned = nullptr;     // background block allocated by the group (freed in smaug_destroy)
  // CUDA-graph replay of whole time steps (launch-bound small grids; SMAUG_PARAM_GRAPH).  One step is 9 launches
  // whose arguments are fixed except for the reduction-set parity (state_set 0 <-> 4), so three executables cover
  // every call: a step from set 0, a step from set 4, and the pair starting at set 0.  They are captured on a
  // library-owned stream (the caller's may be the legacy default stream, which cannot be captured) that is
  // chained to the caller's stream by events.
  int use_graph = 1;
  bool graph_valid = false;
  double graph_cfl = 0;
  cudaGraphExec_t gexec[3] = {nullptr, nullptr, nullptr};
  cudaStream_t gstream = nullptr;
  cudaEvent_t gev_in = nullptr, gev_out = nullptr;
  int launches_per_step = 0;
};

// A px x py decomposition of one global grid into member contexts.  The group owns its members.
struct smaug_group {
  int px = 1, py = 1, NX = 0, NY = 0;
  int gbc[4] = {0, 0, 0, 0};
  bool has_bg = false;
  std::vector<smaug_ctx*> m;            // member b * px + a
  std::vector<int> x0, y0;              // px + 1 / py + 1 prefix offsets
  std::vector<GroupTable*> table;       // device copy of the table on every member's device
  std::vector<cudaEvent_t> ev;          // one per member, for the inter-stream barrier
  bool one_stream = false;              // every member on the same device and stream: no events needed
  int state_set = 0;
  long long exchange_launches = 0;
  bool pending_status = false;
  // tau measurement (smaug_group_set_timing): per member a list of timestamps on its stream, each
  // tagged with what has just finished there -- 0: the member's own work (it now enters a barrier), 1: the barrier's
  // waits, 2: the halo pull.  The gaps 0->1, 1->2, 2->0 are T_idle, T_comm, T_comp of that member.
  bool tau_on = false, tau_broken = false;
  std::vector<std::vector<cudaEvent_t>> tev;
  std::vector<std::vector<unsigned char>> tkind;
  std::vector<size_t> tused;
};

namespace {

CPlanes6 cview(const Planes6& p) {
  CPlanes6 c;
  for (int f = 0; f < NF; ++f) c.p[f] = p.p[f];
  return c;
}

Params make_params(const smaug_ctx* c) {
  Params p;
  p.gamma = c->gamma;
  p.inv_dx = c->geo_nx / c->Lx;
  p.inv_dy = c->geo_ny / c->Ly;
  p.c_rho = c->c_rho; p.c_mom = c->c_mom; p.c_e = c->c_e; p.c_b = c->c_b;
  p.hd_on = c->hd_on;
  p.gx = c->gx; p.gy = c->gy;
  p.grav_on = (c->gx != 0.0 || c->gy != 0.0) ? 1 : 0;
  return p;
}

int launch_ghost(smaug_ctx* c, const Planes6& pl, int nplanes, int freeze) {
  const long long total = 2LL * NG * (c->g.nx + 2 * NG) + 2LL * NG * c->g.ny;
  const int blocks = (int)std::min<long long>((total + 255) / 256, 1024);
  ghost_fill_kernel<<<dim3(blocks, nplanes), 256, 0, c->stream>>>(c->g, pl, freeze);
  c->launches++;
  CU(cudaGetLastError());
  return SMAUG_OK;
}

int launch_wavespeeds(smaug_ctx* c, const Planes6& w, int set) {
  const long long n = (long long)c->g.nx * c->g.ny;
  const int blocks = (int)std::min<long long>((n + 255) / 256, (long long)c->n_sm * 8);
  unsigned long long* slots = c->sc->red[set];
  if (c->has_bg)
    wavespeed_kernel<true><<<blocks, 256, 0, c->stream>>>(c->g, cview(w), c->bg, c->gamma, slots);
  else
    wavespeed_kernel<false><<<blocks, 256, 0, c->stream>>>(c->g, cview(w), c->bg, c->gamma, slots);
  c->launches++;
  CU(cudaGetLastError());
  return SMAUG_OK;
}

#ifndef SMAUG_PRODUCT_ONLY
template <bool BG, bool HD>
int launch_stage_t(smaug_ctx* c, const StageArgs& a) {
  static unsigned long long configured = 0;     // devices on which this instantiation has its smem limit raised
  constexpr size_t smem = Tile<TW, TH, BG>::BYTES;
  auto kern = stage_kernel<TW, TH, NT, BG, HD>;
  CU(configure_smem(kern, smem, c->device, configured));
  dim3 grid((c->g.nx + TW - 1) / TW, (c->g.ny + TH - 1) / TH);
  c->last_ctas = (int)(grid.x * grid.y);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (c->timing && c->ev_used + 2 <= c->ev.size()) {
    e0 = c->ev[c->ev_used++];
    e1 = c->ev[c->ev_used++];
    CU(cudaEventRecord(e0, c->stream));
  }
  kern<<<grid, NT, smem, c->stream>>>(a);
  if (e1) CU(cudaEventRecord(e1, c->stream));
  c->launches++;
  CU(cudaGetLastError());
  return SMAUG_OK;
}

#ifndef SMAUG_MARCH_NT
#define SMAUG_MARCH_NT 256
#endif
constexpr int MARCH_NT = SMAUG_MARCH_NT;

// Streaming form (smaug_march_kernel.cuh): no background, hyperdiffusion on.
int launch_march(smaug_ctx* c, const StageArgs& a) {
  static unsigned long long configured = 0;     // devices on which this instantiation has its smem limit raised
  constexpr size_t smem = MarchSmem<MARCH_NT>::BYTES;
  auto kern = march_kernel<MARCH_NT>;
  CU(configure_smem(kern, smem, c->device, configured));
  const int W = MARCH_NT - 2 * NG;
  const int strips = (c->g.nx + W - 1) / W;
  const int target = c->n_sm * 8;
  int nchunks = std::max(1, (target + strips - 1) / strips);
  MarchGeom mg;
  mg.rows_per_cta = std::max(32, (c->g.ny + nchunks - 1) / nchunks);
  nchunks = (c->g.ny + mg.rows_per_cta - 1) / mg.rows_per_cta;
  dim3 grid(strips, nchunks);
  c->last_ctas = strips * nchunks;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (c->timing && c->ev_used + 2 <= c->ev.size()) {
    e0 = c->ev[c->ev_used++];
    e1 = c->ev[c->ev_used++];
    CU(cudaEventRecord(e0, c->stream));
  }
  kern<<<grid, MARCH_NT, smem, c->stream>>>(a, mg);
  if (e1) CU(cudaEventRecord(e1, c->stream));
  c->launches++;
  CU(cudaGetLastError());
  return SMAUG_OK;
}

#endif   // SMAUG_PRODUCT_ONLY

#ifndef SMAUG_SPLIT_NC
#define SMAUG_SPLIT_NC 128
#endif
constexpr int SPLIT_NC = SMAUG_SPLIT_NC;

// Chunk height of a streaming kernel: every CTA costs (rows + 6) row steps and CTAs run in waves of n_sm,
// so pick the chunk count that minimises waves * (rows + 6).
int pick_rows_per_cta(int ny, int strips, int n_sm, int warm_rows = 2 * NG) {
  int best_rows = ny;
  long long best_cost = -1;
  for (int k = 1; k <= 64; ++k) {
    int nch = std::max(1, n_sm * k / strips);
    int rows = std::max(std::min(ny, 16), (ny + nch - 1) / nch);
    nch = (ny + rows - 1) / rows;
    const long long waves = ((long long)strips * nch + n_sm - 1) / n_sm;
    const long long cost = waves * (rows + warm_rows);
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_rows = rows; }
  }
  return best_rows;
}

template <int COMBINE, int WS, bool BG = false, bool GRAV = false>
int launch_split_t(smaug_ctx* c, const StageArgs& a) {
  static unsigned long long configured = 0;     // devices on which this instantiation has its smem limit raised
  constexpr size_t smem = SplitSmem<SPLIT_NC, BG>::BYTES;
  auto kern = split_kernel<SPLIT_NC, COMBINE, WS, BG, GRAV>;
  CU(configure_smem(kern, smem, c->device, configured));
  const int W = SPLIT_NC - 8;
  const int strips = (c->g.nx + W - 1) / W;
  MarchGeom mg;
  mg.rows_per_cta = pick_rows_per_cta(c->g.ny, strips, c->n_sm * SplitSmem<SPLIT_NC, BG>::CTAS_PER_SM);
  const int nchunks = (c->g.ny + mg.rows_per_cta - 1) / mg.rows_per_cta;
  dim3 grid(strips, nchunks);
  c->last_ctas = strips * nchunks;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (c->timing && c->ev_used + 2 <= c->ev.size()) {
    e0 = c->ev[c->ev_used++];
    e1 = c->ev[c->ev_used++];
    CU(cudaEventRecord(e0, c->stream));
  }
  kern<<<grid, SPLIT_NC + SPLIT_NC / 2, smem, c->stream>>>(a, mg);
  if (e1) CU(cudaEventRecord(e1, c->stream));
  c->launches++;
  CU(cudaGetLastError());
  return SMAUG_OK;
}

// Role-split streaming form (smaug_split_kernel.cuh): hyperdiffusion on; BG instantiations for a background
// (with or without gravity).
int launch_split(smaug_ctx* c, const StageArgs& a) {
  if (c->has_bg) {
    if (a.combine == COMBINE_BASE && a.ws_mode == WS_VT) return launch_split_t<COMBINE_BASE, WS_VT, true>(c, a);
    if (a.combine == COMBINE_ACC && a.ws_mode == WS_VT) return launch_split_t<COMBINE_ACC, WS_VT, true>(c, a);
    if (a.combine == COMBINE_FINAL && a.ws_mode == WS_FULL) return launch_split_t<COMBINE_FINAL, WS_FULL, true>(c, a);
    if (a.combine == COMBINE_BASE && a.ws_mode == WS_FULL) return launch_split_t<COMBINE_BASE, WS_FULL, true>(c, a);
    return fail(SMAUG_EINVAL, "split kernel: unsupported combine / wave-speed mode");
  }
  if (a.prm.grav_on) {       // gravity on a zero background
    if (a.combine == COMBINE_BASE && a.ws_mode == WS_VT) return launch_split_t<COMBINE_BASE, WS_VT, false, true>(c, a);
    if (a.combine == COMBINE_ACC && a.ws_mode == WS_VT) return launch_split_t<COMBINE_ACC, WS_VT, false, true>(c, a);
    if (a.combine == COMBINE_FINAL && a.ws_mode == WS_FULL) return launch_split_t<COMBINE_FINAL, WS_FULL, false, true>(c, a);
    if (a.combine == COMBINE_BASE && a.ws_mode == WS_FULL) return launch_split_t<COMBINE_BASE, WS_FULL, false, true>(c, a);
    return fail(SMAUG_EINVAL, "split kernel: unsupported combine / wave-speed mode");
  }
  if (a.combine == COMBINE_BASE && a.ws_mode == WS_VT) return launch_split_t<COMBINE_BASE, WS_VT>(c, a);
  if (a.combine == COMBINE_ACC && a.ws_mode == WS_VT) return launch_split_t<COMBINE_ACC, WS_VT>(c, a);
  if (a.combine == COMBINE_FINAL && a.ws_mode == WS_FULL) return launch_split_t<COMBINE_FINAL, WS_FULL>(c, a);
  if (a.combine == COMBINE_BASE && a.ws_mode == WS_FULL) return launch_split_t<COMBINE_BASE, WS_FULL>(c, a);
  return fail(SMAUG_EINVAL, "split kernel: unsupported combine / wave-speed mode");
}

#ifndef SMAUG_FLUX_NT
#define SMAUG_FLUX_NT 0        // 0: strip width picked per grid (flux_strip_threads); 128 / 256: forced (tuning builds)
#endif

// Streaming form without hyperdiffusion (smaug_flux_kernel.cuh): HD off, with (BG) or without a background.
template <int NT, bool BG, bool GRAV>
int launch_flux_t(smaug_ctx* c, const StageArgs& a) {
  static unsigned long long configured = 0;     // devices on which this instantiation has its smem limit raised
  constexpr size_t smem = FluxSmem<NT, BG>::BYTES;
  auto kern = flux_kernel<NT, BG, GRAV>;
  CU(configure_smem(kern, smem, c->device, configured));
  const int W = NT - 4;
  const int strips = (c->g.nx + W - 1) / W;
  MarchGeom mg;
  mg.rows_per_cta = pick_rows_per_cta(c->g.ny, strips, c->n_sm * FluxSmem<NT, BG>::CTAS_PER_SM, 4);
  const int nchunks = (c->g.ny + mg.rows_per_cta - 1) / mg.rows_per_cta;
  dim3 grid(strips, nchunks);
  c->last_ctas = strips * nchunks;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (c->timing && c->ev_used + 2 <= c->ev.size()) {
    e0 = c->ev[c->ev_used++];
    e1 = c->ev[c->ev_used++];
    CU(cudaEventRecord(e0, c->stream));
  }
  kern<<<grid, NT, smem, c->stream>>>(a, mg);
  if (e1) CU(cudaEventRecord(e1, c->stream));
  c->launches++;
  CU(cudaGetLastError());
  return SMAUG_OK;
}

// Strip width of the streaming kernel without HD: 256 threads (two CTAs per SM) or 128 (four; three with a background).
// Modelled efficiency of a width = useful columns of its strips x useful rows of its chunks x filled CTA slots of its
// waves; the wide strip gets the 5 % it measures better at equal geometry (fewer halo columns, longer coalesced rows).
// Measured, HD off, ms per stage (128 / 256): 8000^2 1.70 / 1.66, 4000^2 0.451 / 0.435, 2044^2 0.126 / 0.175, 1000^2 0.0439 / 0.0396.
double flux_geometry_efficiency(const smaug_ctx* c, int nt, int ctas_per_sm) {
  const int W = nt - 4, strips = (c->g.nx + W - 1) / W, slots = c->n_sm * ctas_per_sm;
  const int rows = pick_rows_per_cta(c->g.ny, strips, slots, 4);
  const int nchunks = (c->g.ny + rows - 1) / rows;
  const long long ctas = (long long)strips * nchunks, waves = (ctas + slots - 1) / slots;
  return ((double)c->g.nx / ((double)strips * W)) * ((double)rows / (rows + 4)) * ((double)ctas / ((double)waves * slots));
}
int flux_strip_threads(const smaug_ctx* c) {
  if (SMAUG_FLUX_NT != 0) return SMAUG_FLUX_NT;
  const double e128 = flux_geometry_efficiency(c, 128, c->has_bg ? 3 : 4), e256 = 1.05 * flux_geometry_efficiency(c, 256, 2);
  return e256 >= e128 ? 256 : 128;
}

int launch_flux(smaug_ctx* c, const StageArgs& a) {
  if (flux_strip_threads(c) == 256) {
    if (c->has_bg) return launch_flux_t<256, true, false>(c, a);
    return a.prm.grav_on ? launch_flux_t<256, false, true>(c, a) : launch_flux_t<256, false, false>(c, a);
  }
  if (c->has_bg) return launch_flux_t<128, true, false>(c, a);
  return a.prm.grav_on ? launch_flux_t<128, false, true>(c, a) : launch_flux_t<128, false, false>(c, a);
}

// The streaming kernels cover every configuration; the tiled kernel runs when SMAUG_PARAM_KERNEL = 0 (tests), and
// hyperdiffusion-on cases when SMAUG_PARAM_KERNEL = 1 excludes the split kernel and march_kernel does not apply.
bool plain(const smaug_ctx* c) { return !c->has_bg && c->gx == 0.0 && c->gy == 0.0; }
// The small-grid path (smaug_line_kernel.cuh): a one-dimensional problem that one cluster of <= 8 CTAs covers, the
// y-boundary periodic or open (ghost rows are then copies of the row), no background, RK4 or RK2, not a member of a
// group, default kernel selection.
bool uses_line(const smaug_ctx* c) {
  return c->kernel_mode == 2 && !c->has_bg && !c->group && c->g.ny == 1 && c->g.nx <= LINE_MAX_NX &&
         c->g.bc[2] != BC_FIXED && c->g.bc[3] != BC_FIXED && (c->rk_order == 4 || c->rk_order == 2) && c->line_ok;
}
bool uses_flux(const smaug_ctx* c) { return !c->hd_on && c->kernel_mode != 0; }
bool uses_split(const smaug_ctx* c) { return c->hd_on && c->kernel_mode >= 2; }
bool uses_march(const smaug_ctx* c) { return plain(c) && c->hd_on && c->kernel_mode == 1; }

int launch_stage(smaug_ctx* c, const StageArgs& a) {
  if (uses_flux(c)) return launch_flux(c, a);
  if (uses_split(c)) return launch_split(c, a);
#ifndef SMAUG_PRODUCT_ONLY
  if (uses_march(c)) return launch_march(c, a);
  if (c->has_bg) return c->hd_on ? launch_stage_t<true, true>(c, a) : launch_stage_t<true, false>(c, a);
  return c->hd_on ? launch_stage_t<false, true>(c, a) : launch_stage_t<false, false>(c, a);
#else
  return fail(SMAUG_EINVAL, "this build carries no second implementations (SMAUG_PARAM_KERNEL = 0 / 1)");
#endif
}

// The fused kernel of one stage (the ghosts of buffer `in` must be filled).
int run_stage_kernel(smaug_ctx* c, int in, int base, int acc_in, int out, int acc_out, double coef, int combine,
                     int red_in, int red_out, int ws_mode) {
  StageArgs a;
  a.g = c->g;
  a.prm = make_params(c);
  a.in = cview(c->buf[in]);
  a.base = cview(c->buf[base]);
  a.acc_in = cview(c->buf[acc_in]);
  a.out = c->buf[out];
  a.acc_out = c->buf[acc_out];
  a.bg = c->bg;
  a.sc = c->sc;
  a.red_in = red_in;
  a.red_out = red_out;
  a.c = coef;
  a.combine = combine;
  a.ws_mode = ws_mode;
  return launch_stage(c, a);
}

// One stage: ghost fill of the input buffer, then the fused kernel.
int run_stage(smaug_ctx* c, int in, int base, int acc_in, int out, int acc_out, double coef, int combine,
              int red_in, int red_out, int ws_mode) {
  int rc = launch_ghost(c, c->buf[in], NF, 0);
  if (rc) return rc;
  return run_stage_kernel(c, in, base, acc_in, out, acc_out, coef, combine, red_in, red_out, ws_mode);
}

// The stages of one time step as a table (c-6), shared by the single-context path and the group path.
struct StageSpec { int in, base, acc_in, out, acc_out; double coef; int combine, red_in, red_out, ws; };
int stage_table(const smaug_ctx* c, int A, int B, StageSpec st[4]) {
  const int vt_mode = c->hd_on ? WS_VT : WS_NONE;
  if (c->rk_order == 4) {
    st[0] = {0, 0, 3, 1, 3, 0.5, COMBINE_BASE, A, 1, vt_mode};            // w1 = wn + dt/2 R(wn)
    st[1] = {1, 0, 3, 2, 3, 0.5, COMBINE_ACC, 1, 2, vt_mode};             // w2; acc = (w1 - wn) + 2 w2
    st[2] = {2, 0, 3, 1, 3, 1.0, COMBINE_BASE, 2, 3, vt_mode};            // w3 = wn + dt R(w2)
    st[3] = {1, 0, 3, 0, 3, 1.0 / 6.0, COMBINE_FINAL, 3, B, WS_FULL};     // w^{n+1}
    return 4;
  }
  if (c->rk_order == 2) {
    st[0] = {0, 0, 3, 1, 3, 0.5, COMBINE_BASE, A, 1, vt_mode};
    // in-place on buf[0] is safe: base is read and out written by the same thread at the same cell only
    st[1] = {1, 0, 3, 0, 3, 1.0, COMBINE_BASE, 1, B, WS_FULL};
    return 2;
  }
  st[0] = {0, 0, 3, 1, 3, 1.0, COMBINE_BASE, A, B, WS_FULL};             // Euler: the caller swaps buf[0], buf[1]
  return 1;
}

// One full time step (c-6, c-7).  The state lives in buf[0] before and after.
int enqueue_step(smaug_ctx* c, double cfl) {
  const int A = c->state_set, B = A == 0 ? 4 : 0;
  dt_kernel<<<1, 32, 0, c->stream>>>(c->sc, A, (1u << 1) | (1u << 2) | (1u << 3) | (1u << B), cfl,
                                     c->fixed_dt, c->Lx / c->geo_nx, c->Ly / c->geo_ny, c->geo_nx, c->geo_ny);
  c->launches++;
  CU(cudaGetLastError());
  StageSpec st[4];
  const int ns = stage_table(c, A, B, st);
  int rc = SMAUG_OK;
  for (int k = 0; k < ns && !rc; ++k)
    rc = run_stage(c, st[k].in, st[k].base, st[k].acc_in, st[k].out, st[k].acc_out, st[k].coef, st[k].combine,
                   st[k].red_in, st[k].red_out, st[k].ws);
  if (!rc && c->rk_order == 1) std::swap(c->buf[0], c->buf[1]);
  c->state_set = B;
  return rc;
}

// n whole time steps of a one-dimensional problem in one persistent cluster launch.
template <bool HD>
int launch_line_t(smaug_ctx* c, int n_steps, double cfl) {
  static unsigned long long configured = 0;
  constexpr size_t smem = LineSmem::BYTES;
  auto kern = line_step_kernel<HD>;
  CU(configure_smem(kern, smem, c->device, configured));
  LineArgs la;
  la.g = c->g;
  la.prm = make_params(c);
  for (int b = 0; b < 4; ++b) la.buf[b] = c->buf[b];
  la.sc = c->sc;
  la.state_set = c->state_set;
  la.n_steps = n_steps;
  la.rk_order = c->rk_order;
  la.cfl = cfl; la.fixed_dt = c->fixed_dt;
  la.dx = c->Lx / c->geo_nx; la.dy = c->Ly / c->geo_ny;
  const int ntiles = (c->g.nx + LINE_W - 1) / LINE_W;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(ntiles); cfg.blockDim = dim3(LINE_NT); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = ntiles; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (c->timing && c->ev_used + 2 <= c->ev.size()) {
    e0 = c->ev[c->ev_used++];
    e1 = c->ev[c->ev_used++];
    CU(cudaEventRecord(e0, c->stream));
  }
  const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, la);
  if (e != cudaSuccess) {
    cudaGetLastError();
    c->line_ok = false;                 // fall back to the ordinary launch sequence for this context
    if (e0) c->ev_used -= 2;
    return 1;
  }
  if (e1) CU(cudaEventRecord(e1, c->stream));
  c->last_ctas = ntiles;
  c->launches++;
  if (e1) c->line_stage_equiv += (long long)n_steps * (c->rk_order == 4 ? 4 : 2) - 1;   // the event pair counts as one launch
  if (n_steps & 1) c->state_set = c->state_set == 0 ? 4 : 0;
  return SMAUG_OK;
}

void invalidate_graphs(smaug_ctx* c) {
  for (auto& g : c->gexec) {
    if (g) cudaGraphExecDestroy(g);
    g = nullptr;
  }
  c->graph_valid = false;
}

// Capture the three step graphs for this cfl (parameters are baked into the kernel arguments: any
// smaug_set_param / smaug_set_stream invalidates them).  Leaves the context's state untouched.
int capture_graphs(smaug_ctx* c, double cfl) {
  invalidate_graphs(c);
  if (!c->gstream) {
    CU(cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&c->gev_in, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&c->gev_out, cudaEventDisableTiming));
  }
  const int saved_set = c->state_set;
  const long long saved_launches = c->launches;
  cudaStream_t user = c->stream;
  c->stream = c->gstream;
  int rc = SMAUG_OK;
  for (int k = 0; k < 3 && !rc; ++k) {
    c->state_set = k == 1 ? 4 : 0;
    const long long l0 = c->launches;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(c->gstream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
      rc = fail(SMAUG_ECUDA, "cudaStreamBeginCapture failed");
      break;
    }
    rc = enqueue_step(c, cfl);
    if (!rc && k == 2) rc = enqueue_step(c, cfl);
    const cudaError_t e = cudaStreamEndCapture(c->gstream, &graph);
    if (!rc && e != cudaSuccess) rc = fail(SMAUG_ECUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e));
    if (!rc && cudaGraphInstantiate(&c->gexec[k], graph, 0) != cudaSuccess)
      rc = fail(SMAUG_ECUDA, "cudaGraphInstantiate failed");
    if (graph) cudaGraphDestroy(graph);
    if (k == 0) c->launches_per_step = (int)(c->launches - l0);
  }
  c->stream = user;
  c->state_set = saved_set;
  c->launches = saved_launches;
  if (rc) {
    cudaGetLastError();
    invalidate_graphs(c);
    return rc;
  }
  c->graph_valid = true;
  c->graph_cfl = cfl;
  return SMAUG_OK;
}

// n steps as graph replays on the library's stream, ordered after / before the caller's stream by events.
int replay_steps(smaug_ctx* c, int n) {
  CU(cudaEventRecord(c->gev_in, c->stream));
  CU(cudaStreamWaitEvent(c->gstream, c->gev_in, 0));
  int left = n;
  if (left > 0 && c->state_set == 4) {
    CU(cudaGraphLaunch(c->gexec[1], c->gstream));
    c->state_set = 0;
    --left;
  }
  for (; left >= 2; left -= 2) CU(cudaGraphLaunch(c->gexec[2], c->gstream));
  if (left == 1) {
    CU(cudaGraphLaunch(c->gexec[0], c->gstream));
    c->state_set = 4;
  }
  c->launches += (long long)n * c->launches_per_step;
  CU(cudaEventRecord(c->gev_out, c->gstream));
  CU(cudaStreamWaitEvent(c->stream, c->gev_out, 0));
  return SMAUG_OK;
}

constexpr int GRAPH_MIN_STEPS = 8;   // fewer steps than this do not pay for a capture

int check_ctx(smaug_ctx* c) {
  if (!c) return fail(SMAUG_EINVAL, "NULL context");
  return SMAUG_OK;
}

// copy interior [6][ny][nx] (host or device) <-> padded planes
int copy_in(smaug_ctx* c, const double* src, double* const* planes, int nplanes) {
  const Grid& g = c->g;
  for (int f = 0; f < nplanes; ++f)
    CU(cudaMemcpy2DAsync(planes[f] + cell_addr(g, 0, 0), (size_t)g.pitch * sizeof(double),
                         src + (size_t)f * g.nx * g.ny, (size_t)g.nx * sizeof(double),
                         (size_t)g.nx * sizeof(double), g.ny, cudaMemcpyDefault, c->stream));
  return SMAUG_OK;
}

int collect_timing(smaug_ctx* c) {
  for (size_t k = 0; k + 1 < c->ev_used; k += 2) {
    float ms = 0;
    CU(cudaEventElapsedTime(&ms, c->ev[k], c->ev[k + 1]));
    c->stage_ms += ms;
    c->stage_launches++;
  }
  c->ev_used = 0;
  c->stage_launches += c->line_stage_equiv;
  c->line_stage_equiv = 0;
  return SMAUG_OK;
}

int sync_and_status(smaug_ctx* c) {
  CU(cudaStreamSynchronize(c->stream));
  if (c->timing) {
    int rc = collect_timing(c);
    if (rc) return rc;
  }
  if (c->pending_status) {
    int status = 0;
    CU(cudaMemcpy(&status, &c->sc->status, sizeof(int), cudaMemcpyDeviceToHost));
    c->pending_status = false;
    if (status) return fail(SMAUG_ENONFINITE, "a time step was non-finite or <= 0");
  }
  return SMAUG_OK;
}

}  // namespace

// For the library's other translation units (smaug_static.cu): leave a message where smaug_last_error() finds it.
namespace smaug {
__attribute__((visibility("hidden"))) int set_last_error(int code, const char* msg) { return fail(code, msg ? msg : ""); }
}  // namespace smaug

extern "C" {

const char* smaug_last_error(void) { return g_err.c_str(); }

size_t smaug_workspace_bytes(int nx, int ny, int has_bg) {
  if (nx < 1 || ny < 1) return 0;
  return make_layout(nx, ny, has_bg != 0).total;
}

int smaug_create_in_workspace(int nx, int ny, double gamma, const int bc[4], const double* bg,
                              void* workspace, size_t workspace_bytes, void* stream, smaug_ctx** out) {
  if (!out) return fail(SMAUG_EINVAL, "out is NULL");
  *out = nullptr;
  if (!bc) return fail(SMAUG_EINVAL, "bc is NULL");
  if (nx < 1 || ny < 1) return fail(SMAUG_EINVAL, "nx and ny must be >= 1");
  if (!(gamma > 1.0)) return fail(SMAUG_EINVAL, "gamma must be > 1");
  if (((long long)nx + XOFF + NG + 15) * ((long long)ny + 2 * NG) >= (1LL << 31))
    return fail(SMAUG_EINVAL, "grid too large: a padded plane must have fewer than 2^31 cells");
  for (int s = 0; s < 4; ++s)
    if (bc[s] < 0 || bc[s] > 2) return fail(SMAUG_EINVAL, "unknown boundary kind");
  for (int ax = 0; ax < 2; ++ax)
    if ((bc[2 * ax] == SMAUG_BC_PERIODIC) != (bc[2 * ax + 1] == SMAUG_BC_PERIODIC))
      return fail(SMAUG_EINVAL, "periodic must be set on both sides of an axis");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(SMAUG_ECUDA, "no CUDA device: libsmaug has no CPU fallback");
  }
  smaug_ctx* c = new (std::nothrow) smaug_ctx();
  if (!c) return fail(SMAUG_ENOMEM, "host allocation failed");
  // the context lives on the device of the caller's workspace, else on the current device; it is recorded and
  // made current by every later call (the caller's current device is restored on return)
  {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); dev = 0; }
    if (workspace) {
      cudaPointerAttributes at;
      if (cudaPointerGetAttributes(&at, workspace) == cudaSuccess && at.type == cudaMemoryTypeDevice) dev = at.device;
      else cudaGetLastError();
    }
    c->device = dev;
  }
  DeviceGuard guard_(c->device);
  {
    int n_sm = 0;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, c->device) == cudaSuccess && n_sm > 0)
      c->n_sm = n_sm;
  }
  c->has_bg = bg != nullptr;
  c->L = make_layout(nx, ny, c->has_bg);
  c->g.nx = nx; c->g.ny = ny; c->g.pitch = c->L.pitch; c->g.plane = c->L.plane;
  for (int s = 0; s < 4; ++s) c->g.bc[s] = bc[s];
  c->geo_nx = nx; c->geo_ny = ny;
  c->gamma = gamma;
  c->stream = (cudaStream_t)stream;
  if (workspace) {
    if (workspace_bytes < c->L.total || ((uintptr_t)workspace & 255)) {
      delete c;
      return fail(SMAUG_ENOMEM, "workspace too small or not 256-byte aligned");
    }
    c->base = (char*)workspace;
  } else {
    if (cudaMalloc((void**)&c->base, c->L.total) != cudaSuccess) {
      cudaGetLastError();
      delete c;
      return fail(SMAUG_ENOMEM, "cudaMalloc of the workspace failed");
    }
    c->owns = true;
  }
  auto cleanup = [&](int rc) { smaug_destroy(c); return rc; };
  if (cudaMemsetAsync(c->base, 0, c->L.total, c->stream) != cudaSuccess)
    return cleanup(fail(SMAUG_ECUDA, "cudaMemsetAsync failed"));
  c->sc = (DeviceScalars*)(c->base + c->L.scalars_off);
  c->own_sc = c->sc;
  const size_t plane_bytes = c->L.state_bytes / NF;
  for (int b = 0; b < 4; ++b)
    for (int f = 0; f < NF; ++f) c->buf[b].p[f] = (double*)(c->base + c->L.bufs_off[b] + f * plane_bytes);
  for (int k = 0; k < NBG; ++k)
    c->bg.p[k] = c->has_bg ? (const double*)(c->base + c->L.bg_off + k * plane_bytes) : nullptr;
  if (c->has_bg) {
    Planes6 bgp;
    for (int k = 0; k < NF; ++k) bgp.p[k] = k < NBG ? (double*)c->bg.p[k] : nullptr;
    int rc = copy_in(c, bg, bgp.p, NBG);
    if (!rc) rc = launch_ghost(c, bgp, NBG, 1);   // c-8: periodic -> wrap, else nearest interior, once
    if (rc) return cleanup(rc);
  }
  if (cudaStreamSynchronize(c->stream) != cudaSuccess)
    return cleanup(fail(SMAUG_ECUDA, "stream synchronise failed in create"));
  *out = c;
  return SMAUG_OK;
}

int smaug_create(int nx, int ny, double gamma, const int bc[4], const double* bg, smaug_ctx** out) {
  return smaug_create_in_workspace(nx, ny, gamma, bc, bg, nullptr, 0, nullptr, out);
}

void smaug_destroy(smaug_ctx* c) {
  if (!c) return;
  DeviceGuard guard_(c->device);
  cudaStreamSynchronize(c->stream);
  invalidate_graphs(c);
  if (c->gstream) {
    cudaStreamSynchronize(c->gstream);
    cudaStreamDestroy(c->gstream);
    cudaEventDestroy(c->gev_in);
    cudaEventDestroy(c->gev_out);
  }
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  if (c->bg_owned) cudaFree(c->bg_owned);
  if (c->owns && c->base) cudaFree(c->base);
  cudaGetLastError();
  delete c;
}

int smaug_set_stream(smaug_ctx* c, void* stream) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  CU(cudaStreamSynchronize(c->stream));
  c->stream = (cudaStream_t)stream;
  invalidate_graphs(c);
  return SMAUG_OK;
}

int smaug_set_param(smaug_ctx* c, int key, double v) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  invalidate_graphs(c);      // parameters are baked into captured kernel arguments
  switch (key) {
    case SMAUG_PARAM_LX: if (!(v > 0)) break; c->Lx = v; return SMAUG_OK;
    case SMAUG_PARAM_LY: if (!(v > 0)) break; c->Ly = v; return SMAUG_OK;
    case SMAUG_PARAM_HD_ON: c->hd_on = v != 0.0; return SMAUG_OK;
    case SMAUG_PARAM_C_RHO: if (!(v >= 0)) break; c->c_rho = v; return SMAUG_OK;
    case SMAUG_PARAM_C_MOM: if (!(v >= 0)) break; c->c_mom = v; return SMAUG_OK;
    case SMAUG_PARAM_C_E: if (!(v >= 0)) break; c->c_e = v; return SMAUG_OK;
    case SMAUG_PARAM_C_B: if (!(v >= 0)) break; c->c_b = v; return SMAUG_OK;
    case SMAUG_PARAM_RK_ORDER: if (v != 1 && v != 2 && v != 4) break; c->rk_order = (int)v; return SMAUG_OK;
    case SMAUG_PARAM_FIXED_DT: if (!(v >= 0)) break; c->fixed_dt = v; return SMAUG_OK;
    case SMAUG_PARAM_KERNEL: if (v != 0 && v != 1 && v != 2 && v != 3) break; c->kernel_mode = (int)v; return SMAUG_OK;
    case SMAUG_PARAM_GRAPH: c->use_graph = v != 0.0; return SMAUG_OK;
    case SMAUG_PARAM_GX: if (!std::isfinite(v)) break; c->gx = v; return SMAUG_OK;
    case SMAUG_PARAM_GY: if (!std::isfinite(v)) break; c->gy = v; return SMAUG_OK;
    default: return fail(SMAUG_EINVAL, "unknown parameter key");
  }
  return fail(SMAUG_EINVAL, "parameter value out of range");
}

int smaug_set_state(smaug_ctx* c, const double* w) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  if (!w) return fail(SMAUG_EINVAL, "w is NULL");
  int rc = copy_in(c, w, c->buf[0].p, NF);
  if (rc) return rc;
  // ghosts: fixed sides are frozen here, in every buffer that is ever read with its halo (0, 1, 2)
  if ((rc = launch_ghost(c, c->buf[0], NF, 1))) return rc;
  for (int b = 1; b <= 2; ++b)
    for (int f = 0; f < NF; ++f)
      CU(cudaMemcpyAsync(c->buf[b].p[f], c->buf[0].p[f], (size_t)c->g.plane * sizeof(double),
                         cudaMemcpyDeviceToDevice, c->stream));
  CU(cudaMemsetAsync(c->sc, 0, sizeof(DeviceScalars), c->stream));
  c->state_set = 0;
  if ((rc = launch_wavespeeds(c, c->buf[0], 0))) return rc;
  c->pending_status = false;
  CU(cudaStreamSynchronize(c->stream));
  return SMAUG_OK;
}

int smaug_step_async(smaug_ctx* c, int n_steps, double cfl) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  if (n_steps < 0) return fail(SMAUG_EINVAL, "n_steps must be >= 0");
  if (c->group) return fail(SMAUG_EINVAL, "this context is a member of a group: step it with smaug_group_step");
  if (!(c->fixed_dt > 0.0) && !(cfl > 0.0)) return fail(SMAUG_EINVAL, "cfl must be > 0");
  if (n_steps > 0 && uses_line(c)) {
    const int rc = c->hd_on ? launch_line_t<true>(c, n_steps, cfl) : launch_line_t<false>(c, n_steps, cfl);
    if (rc == SMAUG_OK) {
      c->pending_status = true;
      return SMAUG_OK;
    }
    if (rc < 0) return rc;              // rc == 1: the cluster launch was refused; use the ordinary sequence below
  }
  // Whole steps as CUDA-graph replays: worth it when launches are a visible share of the step (small grids);
  // harmless otherwise.  Not while per-kernel timing events are wanted, and not for Euler (its buffers swap).
  if (c->use_graph && !c->timing && c->rk_order != 1 && n_steps > 0 &&
      ((c->graph_valid && c->graph_cfl == cfl) || n_steps >= GRAPH_MIN_STEPS)) {
    int rc = SMAUG_OK;
    if (!(c->graph_valid && c->graph_cfl == cfl)) rc = capture_graphs(c, cfl);
    if (!rc) {
      rc = replay_steps(c, n_steps);
      if (rc) return rc;
      c->pending_status = true;
      return SMAUG_OK;
    }
    // capture unavailable (e.g. the stream is being captured by the caller): fall through to plain launches
  }
  for (int s = 0; s < n_steps; ++s) {
    int rc = enqueue_step(c, cfl);
    if (rc) return rc;
    // keep the event pool bounded: drain it when full (only when timing is on)
    if (c->timing && c->ev_used + 8 > c->ev.size()) {
      CU(cudaStreamSynchronize(c->stream));
      if ((rc = collect_timing(c))) return rc;
    }
  }
  if (n_steps > 0) c->pending_status = true;
  return SMAUG_OK;
}

int smaug_step(smaug_ctx* c, int n_steps, double cfl) {
  int rc = smaug_step_async(c, n_steps, cfl);
  if (rc) return rc;
  return sync_and_status(c);
}

int smaug_get_state(smaug_ctx* c, double* w) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  if (!w) return fail(SMAUG_EINVAL, "w is NULL");
  const Grid& g = c->g;
  for (int f = 0; f < NF; ++f)
    CU(cudaMemcpy2DAsync(w + (size_t)f * g.nx * g.ny, (size_t)g.nx * sizeof(double),
                         c->buf[0].p[f] + cell_addr(g, 0, 0), (size_t)g.pitch * sizeof(double),
                         (size_t)g.nx * sizeof(double), g.ny, cudaMemcpyDefault, c->stream));
  return sync_and_status(c);
}

int smaug_get_time(smaug_ctx* c, double* t, double* last_dt) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  int rc = sync_and_status(c);
  double v[2];
  CU(cudaMemcpy(v, &c->sc->dt, 2 * sizeof(double), cudaMemcpyDeviceToHost));
  if (last_dt) *last_dt = v[0];
  if (t) *t = v[1];
  return rc;
}

int smaug_get_wavespeeds(smaug_ctx* c, double out[4]) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  if (!out) return fail(SMAUG_EINVAL, "out is NULL");
  int rc = sync_and_status(c);
  CU(cudaMemcpy(out, c->sc->red[c->state_set], 4 * sizeof(double), cudaMemcpyDeviceToHost));
  return rc;
}

int smaug_get_launch_count(smaug_ctx* c, long long* n) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  if (!n) return fail(SMAUG_EINVAL, "n is NULL");
  *n = c->launches;
  return SMAUG_OK;
}

int smaug_get_kernel_info(smaug_ctx* c, int out[5]) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  if (!out) return fail(SMAUG_EINVAL, "out is NULL");
  if (uses_line(c)) {                                      // small-grid path: one cluster of tiles, whole steps per launch
    out[0] = LINE_W; out[1] = 1; out[2] = LINE_NT; out[3] = (int)LineSmem::BYTES;
  } else if (uses_flux(c)) {                               // streaming kernel without HD: a strip of NT-4 columns
    const int nt = flux_strip_threads(c);
    out[0] = nt - 4; out[1] = 1; out[2] = nt;
    out[3] = nt == 256 ? (int)(c->has_bg ? FluxSmem<256, true>::BYTES : FluxSmem<256>::BYTES)
                       : (int)(c->has_bg ? FluxSmem<128, true>::BYTES : FluxSmem<128>::BYTES);
  } else if (uses_split(c)) {   // role-split streaming kernel: a strip of NC-8 columns
    out[0] = SPLIT_NC - 8; out[1] = 1; out[2] = SPLIT_NC + SPLIT_NC / 2;
    out[3] = (int)(c->has_bg ? SplitSmem<SPLIT_NC, true>::BYTES : SplitSmem<SPLIT_NC>::BYTES);
  }
#ifndef SMAUG_PRODUCT_ONLY
  else if (uses_march(c)) {   // streaming kernel: a strip of NT-6 columns
    out[0] = MARCH_NT - 2 * NG; out[1] = 1; out[2] = MARCH_NT;
    out[3] = (int)MarchSmem<MARCH_NT>::BYTES;
  } else {
    out[0] = TW; out[1] = TH; out[2] = NT;
    out[3] = (int)(c->has_bg ? Tile<TW, TH, true>::BYTES : Tile<TW, TH, false>::BYTES);
  }
#endif
  out[4] = c->last_ctas;
  return SMAUG_OK;
}

const char* smaug_get_kernel_name(smaug_ctx* c) {
  if (!c) return "?";
  if (uses_line(c)) return "line_step_kernel<128>";
  if (uses_flux(c)) return flux_strip_threads(c) == 256 ? "flux_kernel<256>" : "flux_kernel<128>";
  if (uses_split(c)) return SPLIT_NC == 128 ? "split_kernel<128>" : "split_kernel";
  if (uses_march(c)) return "march_kernel<256>";
  return TW == 32 && TH == 8 && NT == 512 ? "stage_kernel<32,8,512>" : "stage_kernel";
}

int smaug_set_kernel_timing(smaug_ctx* c, int on) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  CU(cudaStreamSynchronize(c->stream));
  c->timing = on != 0;
  c->ev_used = 0;
  c->stage_ms = 0;
  c->stage_launches = 0;
  c->line_stage_equiv = 0;
  if (c->timing && c->ev.empty()) {
    c->ev.resize(2048);
    for (auto& e : c->ev) CU(cudaEventCreate(&e));
  }
  return SMAUG_OK;
}

int smaug_get_kernel_timing(smaug_ctx* c, double* stage_ms, long long* stage_launches) {
  if (int rc = check_ctx(c)) return rc;
  DeviceGuard guard_(c->device);
  CU(cudaStreamSynchronize(c->stream));
  if (int rc = collect_timing(c)) return rc;
  if (stage_ms) *stage_ms = c->stage_ms;
  if (stage_launches) *stage_launches = c->stage_launches;
  return SMAUG_OK;
}

int smaug_selftest_division(int exp_lo, int exp_hi, unsigned long long seed, long long draws, unsigned long long out[5]) {
  if (!out) return fail(SMAUG_EINVAL, "out is NULL");
  if (exp_lo > exp_hi || exp_lo < -1074 || exp_hi > 1000 || draws < 1) return fail(SMAUG_EINVAL, "bad exponent range or draw count");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(SMAUG_ECUDA, "no CUDA device: libsmaug has no CPU fallback");
  }
  const int blocks = 1184, threads = 256;
  const int per_thread = (int)std::min<long long>(std::max<long long>(1, draws / ((long long)blocks * threads)), 1 << 20);
  unsigned long long* d = nullptr;
  CU(cudaMalloc((void**)&d, 5 * sizeof(unsigned long long)));
  cudaError_t e = cudaMemset(d, 0, 5 * sizeof(unsigned long long));
  if (e == cudaSuccess) {
    division_selftest_kernel<<<blocks, threads>>>(exp_lo, exp_hi, seed, per_thread, d);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(out, d, 5 * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return fail(SMAUG_ECUDA, std::string("division self-test: ") + cudaGetErrorString(e));
  return SMAUG_OK;
}

int smaug_selftest_fp64_pipe(int ilp, int warps_per_subpartition, int iters, double out[2]) {
  if (!out) return fail(SMAUG_EINVAL, "out is NULL");
  if ((ilp != 1 && ilp != 2 && ilp != 4 && ilp != 8) || warps_per_subpartition < 1 || warps_per_subpartition > 8 || iters < 1)
    return fail(SMAUG_EINVAL, "ilp must be 1, 2, 4 or 8; warps per sub-partition 1..8; iters >= 1");
  int ndev = 0, dev = 0, n_sm = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(SMAUG_ECUDA, "no CUDA device: libsmaug has no CPU fallback");
  }
  CU(cudaGetDevice(&dev));
  CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  long long* d = nullptr;
  CU(cudaMalloc((void**)&d, 2 * sizeof(long long)));
  cudaError_t e = cudaMemset(d, 0, 2 * sizeof(long long));
  const int threads = 128 * warps_per_subpartition;
  for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {      // the second launch is the measurement
    switch (ilp) {
      case 1: fp64_pipe_selftest_kernel<1><<<n_sm, threads>>>(iters, 1.25, d); break;
      case 2: fp64_pipe_selftest_kernel<2><<<n_sm, threads>>>(iters, 1.25, d); break;
      case 4: fp64_pipe_selftest_kernel<4><<<n_sm, threads>>>(iters, 1.25, d); break;
      default: fp64_pipe_selftest_kernel<8><<<n_sm, threads>>>(iters, 1.25, d); break;
    }
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
  }
  long long h[2] = {0, 0};
  if (e == cudaSuccess) e = cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return fail(SMAUG_ECUDA, std::string("fp64 pipe self-test: ") + cudaGetErrorString(e));
  out[0] = (double)h[0] / ((double)iters * ilp * warps_per_subpartition);   // cycles per warp instruction and sub-partition
  out[1] = (double)h[0] / (double)iters;                                    // cycles per trip (= chain latency when not pipe-bound)
  return SMAUG_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// Decomposition group.  Host side: member creation, the exchange launches,
// the inter-stream barrier, the lockstep stage loop.
// ---------------------------------------------------------------------------------------------------------------
namespace {

// near-equal blocks ("equal sub-regions"): block column a covers global columns [a nx / px, (a+1) nx / px)
GroupGeom group_geom(int px, int py, int nx, int ny, const int bc[4]) {
  GroupGeom G;
  std::memset(&G, 0, sizeof(G));
  G.px = px; G.py = py; G.NX = nx; G.NY = ny;
  for (int s = 0; s < 4; ++s) G.gbc[s] = bc[s];
  for (int a = 0; a <= px; ++a) G.x0[a] = (int)((long long)a * nx / px);
  for (int b = 0; b <= py; ++b) G.y0[b] = (int)((long long)b * ny / py);
  return G;
}

int group_check(smaug_group* g) {
  if (!g) return fail(SMAUG_EINVAL, "NULL group");
  return SMAUG_OK;
}

// A timestamp on member k's stream for the tau measurement (the member's device is current).  Never throws and never
// fails the step: if the pool cannot grow or the event cannot be recorded the measurement is abandoned and
// smaug_group_get_tau says so.
void tau_mark(smaug_group* g, int k, unsigned char kind) {
  if (!g->tau_on) return;
  auto give_up = [&]() { cudaGetLastError(); g->tau_on = false; g->tau_broken = true; };
  if (g->tused[k] == g->tev[k].size()) {
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) return give_up();
    try {
      g->tkind[k].push_back(kind);
      g->tev[k].push_back(e);
    } catch (...) {
      cudaEventDestroy(e);
      return give_up();
    }
  }
  g->tkind[k][g->tused[k]] = kind;
  if (cudaEventRecord(g->tev[k][g->tused[k]], g->m[k]->stream) != cudaSuccess) return give_up();
  ++g->tused[k];
}

// Every member's stream waits for everything enqueued so far on every other member's stream.
int group_barrier(smaug_group* g) {
  if (g->one_stream) return SMAUG_OK;
  const int n = (int)g->m.size();
  for (int k = 0; k < n; ++k) {
    DeviceGuard dg(g->m[k]->device);
    tau_mark(g, k, 0);
    CU(cudaEventRecord(g->ev[k], g->m[k]->stream));
  }
  for (int k = 0; k < n; ++k) {
    DeviceGuard dg(g->m[k]->device);
    for (int o = 0; o < n; ++o)
      if (o != k) CU(cudaStreamWaitEvent(g->m[k]->stream, g->ev[o], 0));
    tau_mark(g, k, 1);
  }
  return SMAUG_OK;
}

int group_sync(smaug_group* g) {
  for (smaug_ctx* c : g->m) {
    DeviceGuard dg(c->device);
    CU(cudaStreamSynchronize(c->stream));
  }
  return SMAUG_OK;
}

// exchange fill of buffer `buf` (0..3, 4 = background) of every member; the members' interiors must be complete
int group_exchange(smaug_group* g, int buf, int nplanes, int freeze) {
  for (size_t k = 0; k < g->m.size(); ++k) {
    smaug_ctx* c = g->m[k];
    DeviceGuard dg(c->device);
    const long long total = 2LL * NG * (c->g.nx + 2 * NG) + 2LL * NG * c->g.ny;
    const int blocks = (int)std::min<long long>((total + 255) / 256, 1024);
    group_ghost_fill_kernel<<<dim3(blocks, nplanes), 256, 0, c->stream>>>(g->table[k], (int)k, buf, freeze);
    c->launches++;
    g->exchange_launches++;
    CU(cudaGetLastError());
    tau_mark(g, (int)k, 2);
  }
  return SMAUG_OK;
}

int group_upload_tables(smaug_group* g) {
  GroupTable T;
  std::memset(&T, 0, sizeof(T));
  T.geo = group_geom(g->px, g->py, g->NX, g->NY, g->gbc);
  for (size_t k = 0; k < g->m.size(); ++k) {
    const smaug_ctx* c = g->m[k];
    T.pitch[k] = c->g.pitch;
    for (int b = 0; b < 4; ++b)
      for (int f = 0; f < NF; ++f) T.planes[k][b][f] = c->buf[b].p[f];
    for (int f = 0; f < NF; ++f) T.planes[k][4][f] = f < NBG ? const_cast<double*>(c->bg.p[f]) : nullptr;
  }
  for (size_t k = 0; k < g->m.size(); ++k) {
    DeviceGuard dg(g->m[k]->device);
    CU(cudaMemcpy(g->table[k], &T, sizeof(T), cudaMemcpyHostToDevice));
  }
  return SMAUG_OK;
}

// one time step of the whole group: leader's dt, then per stage { exchange ; stage kernels } with barriers between
int group_enqueue_step(smaug_group* g, double cfl) {
  smaug_ctx* L = g->m[0];
  const int A = g->state_set, B = A == 0 ? 4 : 0;
  int rc = group_barrier(g);                      // every member's last stage has reduced into set A
  if (rc) return rc;
  {
    DeviceGuard dg(L->device);
    dt_kernel<<<1, 32, 0, L->stream>>>(L->sc, A, (1u << 1) | (1u << 2) | (1u << 3) | (1u << B), cfl, L->fixed_dt,
                                       L->Lx / g->NX, L->Ly / g->NY, g->NX, g->NY);
    L->launches++;
    CU(cudaGetLastError());
  }
  StageSpec st[4];
  const int ns = stage_table(L, A, B, st);
  for (int k = 0; k < ns; ++k) {
    if ((rc = group_barrier(g))) return rc;       // dt / the previous stage of EVERY member is complete
    if ((rc = group_exchange(g, st[k].in, NF, 0))) return rc;
    for (smaug_ctx* c : g->m) {
      DeviceGuard dg(c->device);
      if ((rc = run_stage_kernel(c, st[k].in, st[k].base, st[k].acc_in, st[k].out, st[k].acc_out, st[k].coef,
                                 st[k].combine, st[k].red_in, st[k].red_out, st[k].ws)))
        return rc;
    }
  }
  if (L->rk_order == 1) {                         // Euler: buffers swap -> the tables' plane pointers follow
    for (smaug_ctx* c : g->m) std::swap(c->buf[0], c->buf[1]);
    if ((rc = group_sync(g))) return rc;
    if ((rc = group_upload_tables(g))) return rc;
  }
  g->state_set = B;
  return SMAUG_OK;
}

int group_status(smaug_group* g) {
  int rc = group_sync(g);
  if (rc) return rc;
  if (g->pending_status) {
    smaug_ctx* L = g->m[0];
    DeviceGuard dg(L->device);
    int status = 0;
    CU(cudaMemcpy(&status, &L->sc->status, sizeof(int), cudaMemcpyDeviceToHost));
    g->pending_status = false;
    if (status) return fail(SMAUG_ENONFINITE, "a time step was non-finite or <= 0");
  }
  return SMAUG_OK;
}

}  // namespace

extern "C" {

void smaug_group_destroy(smaug_group* g) {
  if (!g) return;
  for (size_t k = 0; k < g->m.size(); ++k) {
    if (!g->m[k]) continue;
    DeviceGuard dg(g->m[k]->device);
    cudaStream_t st = g->m[k]->stream;
    cudaStreamSynchronize(st);
    if (k < g->table.size() && g->table[k]) cudaFree(g->table[k]);
    if (k < g->ev.size() && g->ev[k]) cudaEventDestroy(g->ev[k]);
    if (k < g->tev.size())
      for (cudaEvent_t e : g->tev[k]) cudaEventDestroy(e);
    g->m[k]->group = nullptr;
    smaug_destroy(g->m[k]);
    if (st) cudaStreamDestroy(st);
  }
  cudaGetLastError();
  delete g;
}

int smaug_group_create(int px, int py, int nx, int ny, double gamma, const int bc[4], const double* bg,
                       const int* devices, smaug_group** out) {
  if (!out) return fail(SMAUG_EINVAL, "out is NULL");
  *out = nullptr;
  if (!bc) return fail(SMAUG_EINVAL, "bc is NULL");
  if (px < 1 || py < 1 || px > GROUP_MAX_SIDE || py > GROUP_MAX_SIDE) return fail(SMAUG_EINVAL, "px, py must be in 1..8");
  if (nx < px || ny < py) return fail(SMAUG_EINVAL, "every sub-domain needs at least one cell along each axis");
  for (int s = 0; s < 4; ++s)
    if (bc[s] < 0 || bc[s] > 2) return fail(SMAUG_EINVAL, "unknown boundary kind");
  for (int ax = 0; ax < 2; ++ax)
    if ((bc[2 * ax] == SMAUG_BC_PERIODIC) != (bc[2 * ax + 1] == SMAUG_BC_PERIODIC))
      return fail(SMAUG_EINVAL, "periodic must be set on both sides of an axis");
  if (!(gamma > 1.0)) return fail(SMAUG_EINVAL, "gamma must be > 1");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail(SMAUG_ECUDA, "no CUDA device: libsmaug has no CPU fallback");
  }
  const int n = px * py;
  int cur = 0;
  if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); cur = 0; }
  std::vector<int> dev(n, cur);
  if (devices)
    for (int k = 0; k < n; ++k) {
      if (devices[k] < 0 || devices[k] >= ndev) return fail(SMAUG_EINVAL, "device index out of range");
      dev[k] = devices[k];
    }
  // the members read each other's planes and the leader's reduction slots: peer access between every device pair
  for (int k = 0; k < n; ++k)
    for (int o = 0; o < n; ++o) {
      if (dev[k] == dev[o]) continue;
      int can = 0;
      if (cudaDeviceCanAccessPeer(&can, dev[k], dev[o]) != cudaSuccess || !can) {
        cudaGetLastError();
        return fail(SMAUG_ECUDA, "the devices of a group need peer access to each other (NVLink / P2P)");
      }
      DeviceGuard dg(dev[k]);
      const cudaError_t e = cudaDeviceEnablePeerAccess(dev[o], 0);
      if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled)
        return fail(SMAUG_ECUDA, std::string("cudaDeviceEnablePeerAccess: ") + cudaGetErrorString(e));
      cudaGetLastError();
    }
  smaug_group* g = new (std::nothrow) smaug_group();
  if (!g) return fail(SMAUG_ENOMEM, "host allocation failed");
  g->px = px; g->py = py; g->NX = nx; g->NY = ny; g->has_bg = bg != nullptr;
  for (int s = 0; s < 4; ++s) g->gbc[s] = bc[s];
  g->x0.resize(px + 1); g->y0.resize(py + 1);
  {
    const GroupGeom G = group_geom(px, py, nx, ny, bc);
    for (int a = 0; a <= px; ++a) g->x0[a] = G.x0[a];
    for (int b = 0; b <= py; ++b) g->y0[b] = G.y0[b];
  }
  g->m.assign(n, nullptr); g->table.assign(n, nullptr); g->ev.assign(n, nullptr);
  auto cleanup = [&](int rc) { const std::string keep = g_err; smaug_group_destroy(g); g_err = keep; return rc; };
  const int member_bc[4] = {SMAUG_BC_OPEN, SMAUG_BC_OPEN, SMAUG_BC_OPEN, SMAUG_BC_OPEN};   // placeholder: the group fills
  std::vector<double> sub;              // host staging of a member's background block when bg is a host pointer
  for (int b = 0; b < py; ++b)
    for (int a = 0; a < px; ++a) {
      const int k = b * px + a;
      const int mnx = g->x0[a + 1] - g->x0[a], mny = g->y0[b + 1] - g->y0[b];
      DeviceGuard dg(dev[k]);
      cudaStream_t st = nullptr;
      if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess)
        return cleanup(fail(SMAUG_ECUDA, "cudaStreamCreate failed"));
      smaug_ctx* c = nullptr;
      // the background block is copied below (strided out of the global array); create with a dummy non-NULL marker
      int rc = smaug_create_in_workspace(mnx, mny, gamma, member_bc, nullptr, nullptr, 0, st, &c);
      if (rc) { cudaStreamDestroy(st); return cleanup(rc); }
      g->m[k] = c;
      c->group = g;
      c->geo_nx = nx; c->geo_ny = ny;
      c->use_graph = 0;
      if (cudaMalloc((void**)&g->table[k], sizeof(GroupTable)) != cudaSuccess) return cleanup(fail(SMAUG_ENOMEM, "cudaMalloc of the group table failed"));
      if (cudaEventCreateWithFlags(&g->ev[k], cudaEventDisableTiming) != cudaSuccess) return cleanup(fail(SMAUG_ECUDA, "cudaEventCreate failed"));
    }
  if (bg) {
    // members were created without a background: give each one its block of the four planes now
    for (int k = 0; k < n; ++k) {
      smaug_ctx* c = g->m[k];
      DeviceGuard dg(c->device);
      const int a = k % px, b = k / px;
      const size_t plane_bytes = c->L.state_bytes / NF;
      double* mem = nullptr;
      if (cudaMalloc((void**)&mem, NBG * plane_bytes) != cudaSuccess) return cleanup(fail(SMAUG_ENOMEM, "cudaMalloc of a background block failed"));
      c->bg_owned = mem;
      if (cudaMemsetAsync(mem, 0, NBG * plane_bytes, c->stream) != cudaSuccess) return cleanup(fail(SMAUG_ECUDA, "cudaMemsetAsync failed"));
      for (int f = 0; f < NBG; ++f) {
        c->bg.p[f] = (const double*)((char*)mem + f * plane_bytes);
        const double* src = bg + ((size_t)f * ny + g->y0[b]) * nx + g->x0[a];
        if (cudaMemcpy2DAsync((double*)c->bg.p[f] + cell_addr(c->g, 0, 0), (size_t)c->g.pitch * sizeof(double), src,
                              (size_t)nx * sizeof(double), (size_t)c->g.nx * sizeof(double), c->g.ny, cudaMemcpyDefault,
                              c->stream) != cudaSuccess)
          return cleanup(fail(SMAUG_ECUDA, "copy of a background block failed"));
      }
      c->has_bg = true;
    }
  }
  // shared scalars: the leader's
  for (int k = 1; k < n; ++k) g->m[k]->sc = g->m[0]->sc;
  g->one_stream = false;
  int rc = group_upload_tables(g);
  if (!rc && bg) {
    rc = group_sync(g);
    if (!rc) rc = group_exchange(g, 4, NBG, 1);       // c-8: background ghosts once (periodic -> wrap, else nearest interior)
  }
  if (!rc) rc = group_sync(g);
  if (rc) return cleanup(rc);
  *out = g;
  return SMAUG_OK;
}

int smaug_group_size(smaug_group* g, int* px, int* py) {
  if (int rc = group_check(g)) return rc;
  if (px) *px = g->px;
  if (py) *py = g->py;
  return SMAUG_OK;
}

int smaug_group_set_param(smaug_group* g, int key, double value) {
  if (int rc = group_check(g)) return rc;
  if (key == SMAUG_PARAM_GRAPH) return SMAUG_OK;      // groups always launch plainly
  for (smaug_ctx* c : g->m)
    if (int rc = smaug_set_param(c, key, value)) return rc;
  return SMAUG_OK;
}

int smaug_group_set_state(smaug_group* g, const double* w) {
  if (int rc = group_check(g)) return rc;
  if (!w) return fail(SMAUG_EINVAL, "w is NULL");
  int rc = group_sync(g);
  if (rc) return rc;
  for (size_t k = 0; k < g->m.size(); ++k) {
    smaug_ctx* c = g->m[k];
    DeviceGuard dg(c->device);
    const int a = (int)k % g->px, b = (int)k / g->px;
    for (int f = 0; f < NF; ++f) {
      const double* src = w + ((size_t)f * g->NY + g->y0[b]) * g->NX + g->x0[a];
      CU(cudaMemcpy2DAsync(c->buf[0].p[f] + cell_addr(c->g, 0, 0), (size_t)c->g.pitch * sizeof(double), src,
                           (size_t)g->NX * sizeof(double), (size_t)c->g.nx * sizeof(double), c->g.ny,
                           cudaMemcpyDefault, c->stream));
    }
  }
  {
    smaug_ctx* L = g->m[0];
    DeviceGuard dg(L->device);
    CU(cudaMemsetAsync(L->sc, 0, sizeof(DeviceScalars), L->stream));
  }
  if ((rc = group_barrier(g))) return rc;
  if ((rc = group_exchange(g, 0, NF, 1))) return rc;   // fixed sides are frozen here, as in smaug_set_state
  for (smaug_ctx* c : g->m) {
    DeviceGuard dg(c->device);
    for (int b = 1; b <= 2; ++b)
      for (int f = 0; f < NF; ++f)
        CU(cudaMemcpyAsync(c->buf[b].p[f], c->buf[0].p[f], (size_t)c->g.plane * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    c->state_set = 0;
    if ((rc = launch_wavespeeds(c, c->buf[0], 0))) return rc;
  }
  g->state_set = 0;
  g->pending_status = false;
  return group_sync(g);
}

int smaug_group_step(smaug_group* g, int n_steps, double cfl) {
  if (int rc = group_check(g)) return rc;
  if (n_steps < 0) return fail(SMAUG_EINVAL, "n_steps must be >= 0");
  if (!(g->m[0]->fixed_dt > 0.0) && !(cfl > 0.0)) return fail(SMAUG_EINVAL, "cfl must be > 0");
  for (int s = 0; s < n_steps; ++s)
    if (int rc = group_enqueue_step(g, cfl)) return rc;
  if (n_steps > 0) g->pending_status = true;
  if (g->tau_on)                                  // closes the last stage's compute interval of every member
    for (size_t k = 0; k < g->m.size(); ++k) {
      DeviceGuard dg(g->m[k]->device);
      tau_mark(g, (int)k, 0);
    }
  return group_status(g);
}

int smaug_group_set_timing(smaug_group* g, int on) {
  if (int rc = group_check(g)) return rc;
  if (int rc = group_sync(g)) return rc;          // recorded events may still be pending
  const size_t n = g->m.size();
  try {
    g->tev.resize(n);
    g->tkind.resize(n);
    g->tused.assign(n, 0);
  } catch (...) {
    return fail(SMAUG_ENOMEM, "host allocation failed");
  }
  g->tau_on = on != 0;
  g->tau_broken = false;
  return SMAUG_OK;
}

int smaug_group_get_tau(smaug_group* g, double out[4]) {
  if (int rc = group_check(g)) return rc;
  if (!out) return fail(SMAUG_EINVAL, "out is NULL");
  if (int rc = group_sync(g)) return rc;
  if (g->tau_broken) return fail(SMAUG_ECUDA, "the tau measurement was abandoned: a CUDA event could not be created or recorded");
  if (g->tused.size() != g->m.size()) return fail(SMAUG_EINVAL, "timing was never switched on (smaug_group_set_timing)");
  double sum[3] = {0.0, 0.0, 0.0};                // idle, comm, comp, summed over members
  for (size_t k = 0; k < g->m.size(); ++k) {
    DeviceGuard dg(g->m[k]->device);
    for (size_t e = 0; e + 1 < g->tused[k]; ++e) {
      const int a = g->tkind[k][e], b = g->tkind[k][e + 1];
      if (a == 0 && b == 0) continue;             // end of one call -> first barrier of the next: host time, not the step's
      float t = 0.f;
      CU(cudaEventElapsedTime(&t, g->tev[k][e], g->tev[k][e + 1]));
      sum[a == 0 ? 0 : (b == 2 ? 1 : 2)] += t;    // 0->1 idle; 1->2 comm; 2->0 and 1->0 (dt kernel / nothing) comp
    }
  }
  const double n = (double)g->m.size();
  out[0] = sum[2] / n;
  out[1] = sum[1] / n;
  out[2] = sum[0] / n;
  out[3] = std::log(out[0] / (out[1] + out[2]));
  return SMAUG_OK;
}

int smaug_group_get_state(smaug_group* g, double* w) {
  if (int rc = group_check(g)) return rc;
  if (!w) return fail(SMAUG_EINVAL, "w is NULL");
  for (size_t k = 0; k < g->m.size(); ++k) {
    smaug_ctx* c = g->m[k];
    DeviceGuard dg(c->device);
    const int a = (int)k % g->px, b = (int)k / g->px;
    for (int f = 0; f < NF; ++f) {
      double* dst = w + ((size_t)f * g->NY + g->y0[b]) * g->NX + g->x0[a];
      CU(cudaMemcpy2DAsync(dst, (size_t)g->NX * sizeof(double), c->buf[0].p[f] + cell_addr(c->g, 0, 0),
                           (size_t)c->g.pitch * sizeof(double), (size_t)c->g.nx * sizeof(double), c->g.ny,
                           cudaMemcpyDefault, c->stream));
    }
  }
  return group_status(g);
}

int smaug_group_get_time(smaug_group* g, double* t, double* last_dt) {
  if (int rc = group_check(g)) return rc;
  int rc = group_status(g);
  smaug_ctx* L = g->m[0];
  DeviceGuard dg(L->device);
  double v[2];
  CU(cudaMemcpy(v, &L->sc->dt, 2 * sizeof(double), cudaMemcpyDeviceToHost));
  if (last_dt) *last_dt = v[0];
  if (t) *t = v[1];
  return rc;
}

int smaug_group_get_wavespeeds(smaug_group* g, double out[4]) {
  if (int rc = group_check(g)) return rc;
  if (!out) return fail(SMAUG_EINVAL, "out is NULL");
  int rc = group_status(g);
  smaug_ctx* L = g->m[0];
  DeviceGuard dg(L->device);
  CU(cudaMemcpy(out, L->sc->red[g->state_set], 4 * sizeof(double), cudaMemcpyDeviceToHost));
  return rc;
}

int smaug_group_get_launch_count(smaug_group* g, long long* stage_and_aux, long long* exchange) {
  if (int rc = group_check(g)) return rc;
  long long n = 0;
  for (smaug_ctx* c : g->m) n += c->launches;
  if (stage_and_aux) *stage_and_aux = n - g->exchange_launches;
  if (exchange) *exchange = g->exchange_launches;
  return SMAUG_OK;
}

int smaug_group_map_cell(int px, int py, int nx, int ny, const int bc[4], int member, int i, int j, int freeze, int out[7]) {
  if (!bc || !out) return fail(SMAUG_EINVAL, "NULL argument");
  if (px < 1 || py < 1 || px > GROUP_MAX_SIDE || py > GROUP_MAX_SIDE || nx < px || ny < py || member < 0 || member >= px * py)
    return fail(SMAUG_EINVAL, "bad decomposition");
  const GroupGeom G = group_geom(px, py, nx, ny, bc);
  const int a = member % px, b = member / px;
  out[0] = G.x0[a]; out[1] = G.y0[b]; out[2] = G.x0[a + 1] - G.x0[a]; out[3] = G.y0[b + 1] - G.y0[b];
  int sm = -1, si = 0, sj = 0;
  const bool written = group_source_cell(G, member, i, j, freeze, &sm, &si, &sj);
  out[4] = written ? sm : -1; out[5] = si; out[6] = sj;
  return SMAUG_OK;
}

}  // extern "C"
