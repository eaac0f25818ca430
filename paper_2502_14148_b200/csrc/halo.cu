// halo.cu — a1: fill every halo element of every field in ONE launch (walls PAPER.md:349-353,
// DESIGN.md readings R5/R6).  Every halo element (or wall-face element) maps its three
// coordinates independently to the interior source, so edges and corners come out exactly as the sequential
// x -> y -> z fill of the oracle: Periodic wrap; Bounded + centre-located even mirror; Bounded + wall-normal
// face-located: zero on the wall face and beyond.  Pure copies: bitwise reproducible.
//
// Halo elements are enumerated as three slabs (z-slabs with full xy extent, y-slabs, x-strips), so only
// halo bytes are touched: traffic = 2 * sizeof * (padded - interior) per field.  Two kernels with the same map: fill_halos_kernel
// (one thread per element: the reference implementation) and fill_halos_rows_kernel (a warp per slab row, the default).
#include <algorithm>
#include <cstdlib>

#include "ocn_internal.h"

namespace {

struct HaloArgs {
  GridDev g;
  int nfields;
  int ext_y;                                     // y halos are supplied by the slab exchange: leave them alone
  void *q[3 + OCN_MAX_TRACERS];
  unsigned char loc[3 + OCN_MAX_TRACERS][3];   // 1 = face-located along that axis
};

// map coordinate c (1-based, halo range) to its source; returns false if the value is zero by construction
__device__ __forceinline__ bool map_coord(int c, int N, int topo, int face, int &src) {
  src = c;
  if (topo == OCN_PERIODIC) {
    if (c < 1) src = c + N;
    else if (c > N) src = c - N;
    return true;
  }
  if (topo == OCN_BOUNDED) {
    if (face) return !(c <= 1 || c > N);          // wall faces 1, N+1 and everything beyond: 0
    if (c < 1) src = 1 - c;
    else if (c > N) src = 2 * N + 1 - c;
  }
  return true;
}

template <class Real>
__global__ void __launch_bounds__(256) fill_halos_kernel(const HaloArgs a) {
  const GridDev &g = a.g;
  const int f = blockIdx.y;
  Real *q = (Real *)a.q[f];
  const int fx = a.loc[f][0], fy = a.loc[f][1], fz = a.loc[f][2];
  // a wall-normal face-located field also owns the wall face 1 (interior index) as a "halo" element
  const int ex = (g.topo[0] == OCN_BOUNDED && fx) ? 1 : 0;
  const int ey = (g.topo[1] == OCN_BOUNDED && fy) ? 1 : 0;
  const int ez = (g.topo[2] == OCN_BOUNDED && fz) ? 1 : 0;
  const long long nxp = g.Nx + 2 * g.Hx, nyp = g.Ny + 2 * g.Hy;
  const long long nzl = g.Hz + ez, nyl = g.Hy + ey, nxl = g.Hx + ex;       // low-side counts
  const long long nZ = (nzl + g.Hz) * nyp * nxp;                             // z-slabs, full xy
  const long long kin = g.Nz - ez, jin = g.Ny - ey;                          // remaining interior extents
  const long long nY = kin * (nyl + g.Hy) * nxp;
  const long long nX = kin * jin * (nxl + g.Hx);
  const long long total = nZ + nY + nX;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
    int i, j, k;
    if (t < nZ) {
      const long long kk = t / (nyp * nxp), r = t - kk * nyp * nxp;
      k = kk < nzl ? (int)(1 - g.Hz + kk) : (int)(g.Nz + 1 + (kk - nzl));
      j = (int)(r / nxp) + 1 - g.Hy;
      i = (int)(r % nxp) + 1 - g.Hx;
    } else if (t < nZ + nY) {
      const long long tt = t - nZ, per = (nyl + g.Hy) * nxp;
      const long long kk = tt / per, r = tt - kk * per, jj = r / nxp;
      k = (int)(1 + ez + kk);
      j = jj < nyl ? (int)(1 - g.Hy + jj) : (int)(g.Ny + 1 + (jj - nyl));
      i = (int)(r % nxp) + 1 - g.Hx;
    } else {
      const long long tt = t - nZ - nY, per = nxl + g.Hx;
      const long long row = tt / per, ii = tt - row * per;
      k = (int)(1 + ez + row / jin);
      j = (int)(1 + ey + row % jin);
      i = ii < nxl ? (int)(1 - g.Hx + ii) : (int)(g.Nx + 1 + (ii - nxl));
    }
    int si, sj, sk;
    const bool nzx = map_coord(i, g.Nx, g.topo[0], fx, si);
    const bool nzy = map_coord(j, g.Ny, g.topo[1], fy, sj);
    const bool nzz = map_coord(k, g.Nz, g.topo[2], fz, sk);
    if (a.ext_y && (j < 1 || j > g.Ny)) continue;            // multi-GPU y-slabs: rows (and corners) owned by the neighbour rank
    q[g.idx(i, j, k)] = (nzx && nzy && nzz) ? q[g.idx(si, sj, sk)] : Real(0);
  }
}

// Row-wise variant (the default): the same element -> source map, but a WARP owns a whole halo row of the z- and y-slabs (lanes stride
// along x: coalesced 256-byte accesses, the row's (j, k) decode and source row computed once per row in 32-bit arithmetic) and a
// LANE owns one interior row's two x-strips.  The per-element kernel above decodes three 64-bit quotients per element and reached
// 1.9 TB/s of algorithmic traffic at C2 (0.13 ms per substage); it stays as the reference implementation (OCN_HALO_ELEMENTWISE).
template <class Real>
__global__ void __launch_bounds__(256) fill_halos_rows_kernel(const HaloArgs a) {
  const GridDev &g = a.g;
  const int f = blockIdx.y;
  Real *q = (Real *)a.q[f];
  const int fx = a.loc[f][0], fy = a.loc[f][1], fz = a.loc[f][2];
  const int ex = (g.topo[0] == OCN_BOUNDED && fx) ? 1 : 0;
  const int ey = (g.topo[1] == OCN_BOUNDED && fy) ? 1 : 0;
  const int ez = (g.topo[2] == OCN_BOUNDED && fz) ? 1 : 0;
  const int nxp = g.Nx + 2 * g.Hx, nyp = g.Ny + 2 * g.Hy;
  const int nzl = g.Hz + ez, nyl = g.Hy + ey, nxl = g.Hx + ex;             // low-side counts
  const int kin = g.Nz - ez, jin = g.Ny - ey;                                // remaining interior extents
  const int nrowZ = (nzl + g.Hz) * nyp;                                      // z-slab rows (full xy extent)
  const int nrowY = kin * (nyl + g.Hy);                                      // y-slab rows
  const int nrowX = kin * jin;                                               // interior rows: two x-strips each
  const int per = nxl + g.Hx;                                                // x-strip elements per interior row (both sides)
  const int rpw = per > 0 ? max(1, 32 / per) : 1;                            // interior rows per warp: lane = (row, element)
  const long long W = (long long)nrowZ + nrowY + (per > 0 ? (nrowX + rpw - 1) / rpw : 0);   // warp-sized work items
  const int lane = threadIdx.x & 31;
  const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
  for (long long w = w0; w < W; w += nw) {
    if (w < nrowZ + nrowY) {
      int j, k;
      if (w < nrowZ) {
        const int kk = (int)w / nyp, jj = (int)w - kk * nyp;
        k = kk < nzl ? 1 - g.Hz + kk : g.Nz + 1 + (kk - nzl);
        j = jj + 1 - g.Hy;
      } else {
        const int t = (int)(w - nrowZ), per = nyl + g.Hy;
        const int kk = t / per, jj = t - kk * per;
        k = 1 + ez + kk;
        j = jj < nyl ? 1 - g.Hy + jj : g.Ny + 1 + (jj - nyl);
      }
      if (a.ext_y && (j < 1 || j > g.Ny)) continue;          // multi-GPU y-slabs: rows (and corners) owned by the neighbour rank
      int sj, sk;
      const bool nzy = map_coord(j, g.Ny, g.topo[1], fy, sj);
      const bool nzz = map_coord(k, g.Nz, g.topo[2], fz, sk);
      const bool nzr = nzy && nzz;
      Real *drow = q + g.idx(1, j, k) - 1;                     // element i of the row at drow[i]
      const Real *srow = q + g.idx(1, sj, sk) - 1;
      for (int ii = lane; ii < nxp; ii += 32) {
        const int i = ii + 1 - g.Hx;
        int si;
        const bool nzx = map_coord(i, g.Nx, g.topo[0], fx, si);
        drow[i] = (nzx && nzr) ? srow[si] : Real(0);
      }
    } else {
      // x-strips: lane = (row, element) so that one warp access touches 2 sectors per row instead of one row per lane
      // (32 rows a pitch apart = 32 wavefronts per access: the LSU, not DRAM, bounded the first version of this branch)
      const int r = lane / per, e0 = lane - r * per;
      const int row = (int)(w - nrowZ - nrowY) * rpw + r;
      if (r < rpw && row < nrowX) {
        const int kk = row / jin, jj = row - kk * jin;
        const int k = 1 + ez + kk, j = 1 + ey + jj;
        int sj, sk;
        const bool nzr = map_coord(j, g.Ny, g.topo[1], fy, sj) && map_coord(k, g.Nz, g.topo[2], fz, sk);
        Real *drow = q + g.idx(1, j, k) - 1;
        const Real *srow = q + g.idx(1, sj, sk) - 1;
        for (int ii = e0; ii < per; ii += 32) {               // one trip unless a row has more than 32 halo elements
          const int i = ii < nxl ? 1 - g.Hx + ii : g.Nx + 1 + (ii - nxl);
          int si;
          const bool nzx = map_coord(i, g.Nx, g.topo[0], fx, si);
          drow[i] = (nzx && nzr) ? srow[si] : Real(0);
        }
      }
    }
  }
}

// ---- y-slab exchange buffers (App. C "slab and pencil decomposition") ----------------------
// For every field and every padded level the H rows of one side are H * stride_y CONTIGUOUS elements of the layout, so
// packing is nfields * nz_pad straight 16-byte-vector copies; buffer element ((f * nz_pad + kk) * H * stride_y + e).
struct PackArgs {
  int nfields;
  void *q[3 + OCN_MAX_TRACERS];
  long long seg;          // 16-byte vectors per (field, level) segment
  long long sz_vec;       // stride_z in 16-byte vectors
  long long row0_vec;     // offset of the first row of the side, in 16-byte vectors
  int nzp;
};
__global__ void __launch_bounds__(256) halo_pack_y_kernel(const PackArgs a, uint4 *__restrict__ buf, const int unpack) {
  const int f = blockIdx.z, kk = blockIdx.y;
  uint4 *field = (uint4 *)a.q[f] + (long long)kk * a.sz_vec + a.row0_vec;
  uint4 *b = buf + ((long long)f * a.nzp + kk) * a.seg;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < a.seg; e += (long long)gridDim.x * blockDim.x) {
    if (unpack) field[e] = b[e];
    else b[e] = field[e];
  }
}

}  // namespace

int launch_halo_pack_y(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, int side, void *buf, bool unpack, cudaStream_t s) {
  PackArgs a;
  int n = 0;
  auto add = [&](void *p) { if (p) a.q[n++] = p; };
  add(st.u); add(st.v);
  if (!m.hydrostatic) add(st.w);
  for (int t = 0; t < m.n_tracers; ++t) add(st.c[t]);
  a.nfields = n;
  if (n == 0) return OCN_OK;
  const ocn_layout &L = g->lay;
  const int esz = g->dtype == OCN_F64 ? 8 : 4, vec = 16 / esz;
  a.seg = (long long)g->Hy * L.stride_y / vec;
  a.sz_vec = L.stride_z / vec;
  a.nzp = (int)L.nz_pad;
  // pack: the H outermost INTERIOR rows of the side (what the neighbour's halo needs); unpack: the side's HALO rows
  long long row = unpack ? (side == 0 ? 0 : g->Hy + g->Ny) : (side == 0 ? g->Hy : g->Hy + g->Ny - g->Hy);
  a.row0_vec = row * L.stride_y / vec;
  dim3 grid((unsigned)std::max(1LL, std::min(8LL, (a.seg + 255) / 256)), (unsigned)a.nzp, (unsigned)n);
  halo_pack_y_kernel<<<grid, 256, 0, s>>>(a, (uint4 *)buf, unpack ? 1 : 0);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "halo_pack_y_kernel launch");
}

int launch_fill_halos(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, cudaStream_t s) {
  HaloArgs a;
  a.g = g->dev;
  int n = 0;
  auto add = [&](void *p, int lx, int ly, int lz) {
    if (!p) return;
    a.q[n] = p; a.loc[n][0] = lx; a.loc[n][1] = ly; a.loc[n][2] = lz; ++n;
  };
  add(st.u, 1, 0, 0);
  add(st.v, 0, 1, 0);
  if (!m.hydrostatic) add(st.w, 0, 0, 1);
  for (int t = 0; t < m.n_tracers; ++t) add(st.c[t], 0, 0, 0);
  a.nfields = n;
  a.ext_y = g->ext_halo[1];
  if (n == 0) return OCN_OK;
  const long long nxp = g->Nx + 2 * g->Hx, nyp = g->Ny + 2 * g->Hy, nzp = g->Nz + 2 * g->Hz;
  long long total = nxp * nyp * nzp - (long long)g->Nx * g->Ny * g->Nz + nxp * nyp + nxp * nzp + nyp * nzp;  // upper bound
  if (total <= 0) return OCN_OK;
  if (g->diag & OCN_DIAG_HALO_ELEMENTWISE) {      // diagnostic switch: the per-element reference kernel
    long long blocks = (total + 255) / 256;
    if (blocks > 148LL * 32) blocks = 148LL * 32;
    dim3 grid((unsigned)blocks, (unsigned)n, 1);
    if (g->dtype == OCN_F64) fill_halos_kernel<double><<<grid, 256, 0, s>>>(a);
    else fill_halos_kernel<float><<<grid, 256, 0, s>>>(a);
  } else {
    const long long rows = 2LL * (g->Hz + 1) * nyp + (long long)g->Nz * 2 * (g->Hy + 1) + ((long long)g->Nz * g->Ny + 1) / 2;   // generous upper bound of warp items (the grid is capped below)
    long long blocks = (rows + 7) / 8;
    if (blocks > 148LL * 16) blocks = 148LL * 16;
    dim3 grid((unsigned)std::max(1LL, blocks), (unsigned)n, 1);
    if (g->dtype == OCN_F64) fill_halos_rows_kernel<double><<<grid, 256, 0, s>>>(a);
    else fill_halos_rows_kernel<float><<<grid, 256, 0, s>>>(a);
  }
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "fill_halos_kernel launch");
}
