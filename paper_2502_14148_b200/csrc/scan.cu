// scan.cu — the two column scans of the hydrostatic configuration.
//   a2  w from continuity, eq. (15):   w[1] = 0;  w[k+1] = w[k] - dz_c[k] (dx^-1 dx(u) + dy^-1 dy(v))
//   a3  hydrostatic pressure anomaly, eq. (14) PAPER.md:452-454 / (A6) PAPER.md:817-822:
//       p[Nz] = -b[Nz] dz_c[Nz]/2;  p[k-1] = p[k] - (b[k] + b[k-1])/2 * dz_f[k]
// One thread per (i,j) column, sequential in k (Nz is 50 in the hydrostatic config), coalesced in i:
// each level is one fully coalesced row read/write per warp; HBM-bound (3 fields x sizeof per cell each).
#include "ocn_internal.h"

namespace {

template <class Real>
__global__ void __launch_bounds__(128) compute_w_kernel(const GridDev g, const Real *__restrict__ u, const Real *__restrict__ v,
                                                        Real *__restrict__ w) {
  const bool hx = g.topo[0] != OCN_FLAT, hy = g.topo[1] != OCN_FLAT;
  const int ni = hx ? g.Nx + 2 * g.Hx - 1 : g.Nx, nj = hy ? g.Ny + 2 * g.Hy - 1 : g.Ny;
  const int ii = blockIdx.x * blockDim.x + threadIdx.x, jj = blockIdx.y * blockDim.y + threadIdx.y;
  if (ii >= ni || jj >= nj) return;
  const int i = ii + 1 - g.Hx, j = jj + 1 - g.Hy;
  long long o = g.idx(i, j, 1);
  Real wk = Real(0);
  w[o] = wk;
  const Real rdx = Real(g.rdx), rdy = Real(g.rdy);
  for (int k = 1; k <= g.Nz; ++k, o += g.sz) {
    // explicit roundings: the hydrostatic TMA-ring kernel diagnoses the same w itself (tend_fused.cu, a.diag_w), bit for bit
    Real d = Real(0);
    if (hx) d = ocn_fma(u[o + 1] - u[o], rdx, d);
    if (hy) d = ocn_fma(v[o + g.sy] - v[o], rdy, d);
    wk = ocn_fma(-Real(g.dzc[g.zi(k)]), d, wk);
    w[o + g.sz] = wk;
  }
}

template <class Real>
__global__ void __launch_bounds__(128) compute_phy_kernel(const GridDev g, const ModelDev m, const Real *__restrict__ T,
                                                          const Real *__restrict__ S, Real *__restrict__ p) {
  const int ni = g.Nx + 2 * g.Hx, nj = g.Ny + 2 * g.Hy;
  const int ii = blockIdx.x * blockDim.x + threadIdx.x, jj = blockIdx.y * blockDim.y + threadIdx.y;
  if (ii >= ni || jj >= nj) return;
  const int i = ii + 1 - g.Hx, j = jj + 1 - g.Hy;
  long long o = g.idx(i, j, g.Nz);
  auto buoy = [&](long long oo, int k) -> double {
    const double Ta = T ? (double)T[oo] - g.Tref[g.zi(k)] : 0.0;
    const double Sa = S ? (double)S[oo] - g.Sref[g.zi(k)] : 0.0;
    return m.g * (m.alpha_T * Ta - m.beta_S * Sa);
  };
  double bk = buoy(o, g.Nz);
  Real pk = Real(-bk * g.dzc[g.zi(g.Nz)] * 0.5);
  p[o] = pk;
  for (int k = g.Nz; k >= 2; --k) {
    const double bm = buoy(o - g.sz, k - 1);
    pk = Real((double)pk - 0.5 * (bk + bm) * g.dzf[g.zi(k)]);
    o -= g.sz;
    p[o] = pk;
    bk = bm;
  }
}

}  // namespace

int launch_compute_w(const ocn_grid *g, const FieldsDev &st, cudaStream_t s) {
  const int ni = g->Nx + 2 * g->Hx, nj = g->Ny + 2 * g->Hy;
  dim3 block(32, 4, 1), grid((ni + 31) / 32, (nj + 3) / 4, 1);
  if (g->dtype == OCN_F64) compute_w_kernel<double><<<grid, block, 0, s>>>(g->dev, (const double *)st.u, (const double *)st.v, (double *)st.w);
  else compute_w_kernel<float><<<grid, block, 0, s>>>(g->dev, (const float *)st.u, (const float *)st.v, (float *)st.w);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "compute_w_kernel launch");
}

int launch_compute_phy(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, void *phy, cudaStream_t s) {
  const int ni = g->Nx + 2 * g->Hx, nj = g->Ny + 2 * g->Hy;
  dim3 block(32, 4, 1), grid((ni + 31) / 32, (nj + 3) / 4, 1);
  const void *T = m.idx_T >= 0 ? st.c[m.idx_T] : nullptr;
  const void *S = m.idx_S >= 0 ? st.c[m.idx_S] : nullptr;
  if (g->dtype == OCN_F64) compute_phy_kernel<double><<<grid, block, 0, s>>>(g->dev, m, (const double *)T, (const double *)S, (double *)phy);
  else compute_phy_kernel<float><<<grid, block, 0, s>>>(g->dev, m, (const float *)T, (const float *)S, (float *)phy);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "compute_phy_kernel launch");
}
