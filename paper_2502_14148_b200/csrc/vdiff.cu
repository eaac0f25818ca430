// vdiff.cu — SURVEY 8(f) N3: vertically-implicit diffusion, (A2) PAPER.md:785-803 for tracers and (A8) PAPER.md:829-835 for
// momentum:      (1 - dt d_z kz d_z) q^{m+1} = q*        per column, second-order in space, "solved with a tridiagonal algorithm".
// q* is the field after the explicit substage (A4) (whose tendencies then exclude the vertical diffusion term:
// ocn_params.implicit_vertical_diffusion); kz is the model's constant nu (u, v, w) or kappa[n] (reading R24); walls: no flux
// for fields centred in z, w = 0 on the wall faces.
//
// The matrix depends on the level only (dt, kz and the z-metrics are horizontally uniform), so the Thomas pivots are computed
// ONCE per call by vdiff_pivots_kernel (one thread per distinct (kz, z-location) pair, Nz serial steps, a few microseconds) into a
// small scratch block owned by the grid, and the per-column work of implicit_vdiff_kernel is two multiply-add sweeps:
//     forward   d'_k = (q_k - lo_k d'_{k-1}) inv_k         (written in place)
//     backward  x_k  = d'_k - cp_k x_{k+1}
// one thread per (i,j) column, coalesced in i, all fields in one launch (blockIdx.z = field).  HBM-bound: 2 reads + 2 writes
// per field-cell.  Arithmetic in double for both storage types.
#include "ocn_internal.h"

namespace {

constexpr int MAXF = 3 + OCN_MAX_TRACERS;

struct VdiffArgs {
  int nf;
  void *q[MAXF];
  int combo[MAXF];   // which pivot set
  int face[MAXF];    // 1: located on z-faces (w): unknown faces 2..Nz
};
struct PivotArgs {
  int ncombo;
  double kz[2 + OCN_MAX_TRACERS];
  int face[2 + OCN_MAX_TRACERS];
};

// pivots of combo c live at piv + c*3*nzm: lo[k], inv[k], cp[k], k = 1..Nz at index k
__global__ void vdiff_pivots_kernel(const GridDev g, const PivotArgs a, const double dt, double *__restrict__ piv, const int nzm) {
  const int c = threadIdx.x;
  if (c >= a.ncombo) return;
  double *lo = piv + (size_t)c * 3 * nzm, *inv = lo + nzm, *cp = inv + nzm;
  const bool face = a.face[c] != 0;
  const int k0 = face ? 2 : 1, Nz = g.Nz;
  const double s = -dt * a.kz[c];
  double cprev = 0.0;
  for (int k = k0; k <= Nz; ++k) {
    // flux-form second difference at level k: [(q[k+1]-q[k])/d_up - (q[k]-q[k-1])/d_dn] / d_vol
    const double dvol = face ? g.dzf[g.zi(k)] : g.dzc[g.zi(k)];
    const double dup = face ? g.dzc[g.zi(k)] : g.dzf[g.zi(k + 1)];
    const double ddn = face ? g.dzc[g.zi(k - 1)] : g.dzf[g.zi(k)];
    double l = s / (ddn * dvol), u = s / (dup * dvol), diag;
    if (!face) {                       // no flux through the walls
      if (k == 1) l = 0.0;
      if (k == Nz) u = 0.0;
      diag = 1.0 - l - u;
    } else {                           // w = 0 on the walls: the neighbour term vanishes, the diagonal keeps both
      diag = 1.0 - l - u;
      if (k == 2) l = 0.0;
      if (k == Nz) u = 0.0;
    }
    const double iv = 1.0 / (diag - l * cprev);
    cprev = u * iv;
    lo[k] = l; inv[k] = iv; cp[k] = cprev;
  }
}

template <class Real>
__global__ void __launch_bounds__(128) implicit_vdiff_kernel(const GridDev g, const VdiffArgs a, const double *__restrict__ piv,
                                                             const int nzm) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1, j = blockIdx.y * blockDim.y + threadIdx.y + 1, f = blockIdx.z;
  if (i > g.Nx || j > g.Ny) return;
  Real *__restrict__ q = (Real *)a.q[f];
  const double *lo = piv + (size_t)a.combo[f] * 3 * nzm, *inv = lo + nzm, *cp = inv + nzm;
  const int k0 = a.face[f] ? 2 : 1, Nz = g.Nz;
  long long o = g.idx(i, j, k0);
  double d = 0.0;
#pragma unroll 4
  for (int k = k0; k <= Nz; ++k, o += g.sz) {
    d = ((double)q[o] - lo[k] * d) * inv[k];
    q[o] = Real(d);
  }
  o -= 2 * g.sz;
  double x = d;
#pragma unroll 4
  for (int k = Nz - 1; k >= k0; --k, o -= g.sz) {
    x = (double)q[o] - cp[k] * x;
    q[o] = Real(x);
  }
}

}  // namespace

int launch_implicit_vdiff(const ocn_grid *g, const ModelDev &m, double dt, const FieldsDev &st, cudaStream_t s) {
  VdiffArgs a;
  PivotArgs pa;
  a.nf = 0; pa.ncombo = 0;
  auto combo = [&](double kz, int face) {
    for (int c = 0; c < pa.ncombo; ++c)
      if (pa.kz[c] == kz && pa.face[c] == face) return c;
    pa.kz[pa.ncombo] = kz; pa.face[pa.ncombo] = face;
    return pa.ncombo++;
  };
  auto add = [&](void *q, double kz, int face) {
    if (!q || kz == 0.0) return;       // kz = 0: the operator is the identity
    a.q[a.nf] = q; a.combo[a.nf] = combo(kz, face); a.face[a.nf] = face; ++a.nf;
  };
  if (m.momentum) {
    add(st.u, m.nu, 0); add(st.v, m.nu, 0);
    if (!m.hydrostatic) add(st.w, m.nu, 1);
  }
  for (int n = 0; n < m.n_tracers; ++n) add(st.c[n], m.kappa[n], 0);
  if (a.nf == 0) return OCN_OK;
  vdiff_pivots_kernel<<<1, 32, 0, s>>>(g->dev, pa, dt, g->d_vdiff, g->nzm);
  OCN_CUDA(cudaGetLastError());
  dim3 block(64, 2, 1), grid((g->Nx + 63) / 64, (g->Ny + 1) / 2, a.nf);
  if (g->dtype == OCN_F64) implicit_vdiff_kernel<double><<<grid, block, 0, s>>>(g->dev, a, g->d_vdiff, g->nzm);
  else implicit_vdiff_kernel<float><<<grid, block, 0, s>>>(g->dev, a, g->d_vdiff, g->nzm);
  ocn_count_launch(2);
  return ocn_check_cuda(cudaGetLastError(), "implicit_vdiff_kernel launch");
}
