// smaug_group.cuh -- domain decomposition (SURVEY 8(f) NEXT-1; PAPER.md:25 Fig. 1, :55-59 section 3: "the full domain is
// divided into sub-regions, each GPU computes one"; :61-73 `exchange_halo`): the device side of a px x py group of
// contexts.  The paper's exchange is gather -> cudaMemcpy D2H -> MPI_Isend/Irecv -> H2D -> scatter per field; here the
// ghost cells of a sub-domain are PULLED straight out of the owning neighbour's planes by one small kernel per
// sub-domain and RK stage (peer pointers: plain device pointers on one GPU, NVLink P2P mappings across GPUs), and the
// four wave-speed maxima are reduced by the stage kernels' own atomicMax into ONE shared slot array.
//
// The fill reproduces the UNSPLIT ghost fill exactly (c-8: x over interior rows, then y over the padded width), so a
// decomposed run is bit-identical to the single-context run: a ghost cell (i, j) of member (a, b) is global cell
// (I, J) = (x0[a] + i, y0[b] + j); inside the global interior it is some member's interior cell, outside it the global
// boundary rule applies (periodic -> wrap, open -> clamp, fixed -> never rewritten) and gives a global source cell,
// which again some member owns (a corner next to a fixed x-side reads the owner's frozen ghost, as in the unsplit fill).
#pragma once
#include "smaug_device.cuh"

namespace smaug {

constexpr int GROUP_MAX_SIDE = 8;                       // px, py <= 8
constexpr int GROUP_MAX = GROUP_MAX_SIDE * GROUP_MAX_SIDE;
constexpr int GROUP_NBUF = 5;                           // buffers 0..3 of a context, 4 = its background planes

struct GroupGeom {
  int px, py, NX, NY;
  int gbc[4];                                           // GLOBAL boundary kinds x_lo, x_hi, y_lo, y_hi
  int x0[GROUP_MAX_SIDE + 1], y0[GROUP_MAX_SIDE + 1];   // first global column / row of every block column / row
};

struct GroupTable {                                     // lives in device memory (one copy per member device)
  GroupGeom geo;
  int pitch[GROUP_MAX];                                 // member m = b * px + a
  double* planes[GROUP_MAX][GROUP_NBUF][NF];            // peer-visible plane pointers
};

__host__ __device__ inline int group_wrap(int i, int n) {
  int r = i % n;
  return r < 0 ? r + n : r;
}
__host__ __device__ inline int group_owner(const int* first, int n, int g) {   // block holding global index g (clamped)
  int k = 0;
  while (k + 1 < n && g >= first[k + 1]) ++k;
  return k;
}

// Where ghost cell (i, j) (local indices, outside [0,nx) x [0,ny)) of member `me` takes its value from: member *sm,
// local cell (*si, *sj) of that member (an interior cell, or a frozen ghost next to a fixed x-side).  Returns false if
// the cell is never rewritten (a fixed global side, freeze == 0).  This is c-8 of the GLOBAL grid: x over interior
// rows, then y over the padded width, i.e. source = (mapx(I), mapy(J)) with map = wrap / clamp / identity.
__host__ __device__ inline bool group_source_cell(const GroupGeom& G, int me, int i, int j, int freeze, int* sm, int* si, int* sj) {
  const int a = me % G.px, b = me / G.px;
  const int I = G.x0[a] + i, J = G.y0[b] + j;
  const int kx = I < 0 ? G.gbc[0] : (I >= G.NX ? G.gbc[1] : -1);   // -1: inside the global grid along x
  const int ky = J < 0 ? G.gbc[2] : (J >= G.NY ? G.gbc[3] : -1);
  int SI = I, SJ = J;
  if (ky >= 0) {
    if (ky == BC_FIXED && !freeze) return false;
    SJ = ky == BC_PERIODIC ? group_wrap(J, G.NY) : (J < 0 ? 0 : G.NY - 1);
    if (kx >= 0 && !(kx == BC_FIXED && !freeze)) SI = kx == BC_PERIODIC ? group_wrap(I, G.NX) : (I < 0 ? 0 : G.NX - 1);
  } else if (kx >= 0) {
    if (kx == BC_FIXED && !freeze) return false;
    SI = kx == BC_PERIODIC ? group_wrap(I, G.NX) : (I < 0 ? 0 : G.NX - 1);
  }
  const int sa = group_owner(G.x0, G.px, SI), sb = group_owner(G.y0, G.py, SJ);
  *sm = sb * G.px + sa;
  *si = SI - G.x0[sa];
  *sj = SJ - G.y0[sb];
  return true;
}

// Ghost fill of member `me` for planes 0..gridDim.y-1 of buffer `buf`.  freeze = 1 (set_state, background): a fixed side
// acts like an open one.  Reads interior cells (or frozen fixed ghosts) of any member, writes only ghosts of `me`; all
// members' interiors of `buf` must be complete before the launch (the group's barrier).
__global__ void __launch_bounds__(256) group_ghost_fill_kernel(const GroupTable* __restrict__ T, int me, int buf, int freeze) {
  const GroupGeom& G = T->geo;
  const int a = me % G.px, b = me / G.px;
  const int nx = G.x0[a + 1] - G.x0[a], ny = G.y0[b + 1] - G.y0[b];
  const int f = blockIdx.y;
  double* const p = T->planes[me][buf][f];
  const int pitch = T->pitch[me];
  const int wpad = nx + 2 * NG;
  const long long n_y = 2LL * NG * wpad;
  const long long total = n_y + 2LL * NG * ny;
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
    int i, j;
    if (q < n_y) {
      const int row = (int)(q / wpad);
      i = (int)(q - (long long)row * wpad) - NG;
      j = row < NG ? row - NG : ny + (row - NG);
    } else {
      const long long r = q - n_y;
      j = (int)(r / (2 * NG));
      const int s = (int)(r - (long long)j * (2 * NG));
      i = s < NG ? s - NG : nx + (s - NG);
    }
    int sm, si, sj;
    if (!group_source_cell(G, me, i, j, freeze, &sm, &si, &sj)) continue;
    const double* const src = T->planes[sm][buf][f];
    p[(long long)(j + NG) * pitch + (i + XOFF)] = src[(long long)(sj + NG) * T->pitch[sm] + (si + XOFF)];
  }
}

}  // namespace smaug
