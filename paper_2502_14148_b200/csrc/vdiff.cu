// vdiff.cu — SURVEY 8(f) N3: vertically-implicit diffusion, (A2) PAPER.md:785-803 for tracers and (A8) PAPER.md:829-835 for
// momentum:      (1 - dt d_z kz d_z) q^{m+1} = q*        per column, second-order in space, "solved with a tridiagonal algorithm".
// q* is the field after the explicit substage (A4) (whose tendencies then exclude the vertical diffusion term:
// ocn_params.implicit_vertical_diffusion); kz is the model's constant nu (u, v, w) or kappa[n] (reading R24); walls: no flux
// for fields centred in z, w = 0 on the wall faces.
//
// The matrix depends on the level only (dt, kz and the z-metrics are horizontally uniform), so the Thomas pivots are computed
// ONCE per call by vdiff_pivots_kernel (one thread per distinct (kz, z-location) pair, Nz serial steps, a few microseconds) into a
// small scratch block owned by the grid, and the per-column work is two sweeps with ONE fused multiply-add on the dependent chain:
//     forward   d'_k = q_k inv_k - (lo_k inv_k) d'_{k-1}
//     backward  x_k  = d'_k - cp_k x_{k+1}
// implicit_vdiff_tile_kernel (the default): one warp streams a 32-column x Nz tile of one field through shared memory with cp.async
// (every level a coalesced row, a rolling window of ~100 levels in flight), sweeps forward as the levels land, keeps d' on chip and
// writes the backward sweep straight to global memory: 1 read + 1 write per field-cell, the compulsory traffic.  implicit_vdiff_kernel (columns too tall for shared
// memory): one thread per column sweeping global memory in place, 2 reads + 2 writes.  Same arithmetic, in double for both
// storage types; all fields in one launch (blockIdx.z = field).
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

// pivots of combo c live at piv + c*3*nzm: al[k] = lo_k inv_k, inv[k], cp[k], k = 1..Nz at index k
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
    lo[k] = l * iv; inv[k] = iv; cp[k] = cprev;
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
    d = fma(-lo[k], d, (double)q[o] * inv[k]);
    q[o] = Real(d);
  }
  o -= 2 * g.sz;
  double x = d;
#pragma unroll 4
  for (int k = Nz - 1; k >= k0; --k, o -= g.sz) {
    x = fma(-cp[k], x, (double)q[o]);
    q[o] = Real(x);
  }
}

constexpr int TILE_X = 32;

__device__ __forceinline__ void cp_async_elem(void *smem, const double *g) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_elem(void *smem, const float *g) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(g) : "memory");
}

// One WARP per 32-column x Nz tile (block = 32 threads): lane = column.  The warp streams the tile into shared memory with 16-byte
// cp.async (a lane copies 2 (fp64) / 4 (fp32) adjacent columns of one level; 8-byte copies reached only 1.8 TB/s with 3 warps per
// SM, measured) through a rolling window of WIN batches of UB levels (~24 KB in flight per warp), runs the forward sweep on
// batch b as soon as it has landed (cp.async.wait_group WIN + __syncwarp), keeps d' in shared
// memory, and the backward sweep writes x straight to global memory (a coalesced row per level).  No block barrier, no second
// pass over global memory: 1 read + 1 write per field-cell.
template <class Real>
__global__ void __launch_bounds__(32) implicit_vdiff_tile_kernel(const GridDev g, const VdiffArgs a, const double *__restrict__ piv,
                                                                 const int nzm) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int UB = 16, WIN = 6;
  const int Nz = g.Nz;
  double *spiv = (double *)smem_raw;                               // al[Nz], inv[Nz], cp[Nz] of this field (index k-1)
  Real *tile = (Real *)(spiv + ((3 * Nz + 1) & ~1));               // [Nz][TILE_X], 16-byte aligned
  const int f = blockIdx.z, j = blockIdx.y + 1, i0 = blockIdx.x * TILE_X + 1, lane = threadIdx.x;
  const bool active = i0 + lane <= g.Nx;
  Real *__restrict__ q = (Real *)a.q[f];
  const int k0 = a.face[f] ? 2 : 1;
  const long long base = g.idx(active ? i0 + lane : i0, j, 1);
  Real *col = tile + lane;
  {   // the pivots: the oldest cp.async group
    const double *gp = piv + (size_t)a.combo[f] * 3 * nzm;
    for (int t = lane; t < 3 * Nz; t += 32) cp_async_elem(&spiv[t], gp + (t / Nz) * nzm + (t % Nz) + 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  const int nb = (Nz - k0 + 1 + UB - 1) / UB;
  // 16-byte cp.async: a lane copies EPL adjacent columns of one level, the warp covers EPL levels per instruction
  constexpr int EPL = 16 / (int)sizeof(Real), LPR = TILE_X / EPL;
  const int c0 = (lane % LPR) * EPL, lsub = lane / LPR;
  const int nvalid = min(EPL, g.Nx - (i0 + c0) + 1);                // columns of this lane's chunk inside the grid (<= 0: none)
  const long long cbase = g.idx(i0 + c0, j, 1);
  auto issue = [&](int b) {
    if (b < nb && nvalid > 0) {
      const int ka = k0 + b * UB, kb = min(ka + UB - 1, Nz);
      for (int k = ka + lsub; k <= kb; k += EPL) {
        Real *dst = &tile[(k - 1) * TILE_X + c0];
        const Real *src = q + cbase + (long long)(k - 1) * g.sz;
        if (nvalid == EPL)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
        else
          for (int e = 0; e < nvalid; ++e) cp_async_elem(dst + e, src + e);
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  for (int b = 0; b < WIN; ++b) issue(b);
  const double *al = spiv - 1, *inv = al + Nz, *cp = inv + Nz;      // indexed by k
  double d = 0.0;
  for (int b = 0; b < nb; ++b) {
    issue(b + WIN);
    asm volatile("cp.async.wait_group %0;" ::"n"(WIN) : "memory");
    __syncwarp();                                                   // the pivots were copied by other lanes
    const int ka = k0 + b * UB;
    if (ka + UB - 1 <= Nz) {
      double qv[UB], av[UB];
#pragma unroll
      for (int u = 0; u < UB; ++u) { qv[u] = (double)col[(ka + u - 1) * TILE_X] * inv[ka + u]; av[u] = al[ka + u]; }
#pragma unroll
      for (int u = 0; u < UB; ++u) { d = fma(-av[u], d, qv[u]); col[(ka + u - 1) * TILE_X] = Real(d); }
    } else {
      for (int k = ka; k <= Nz; ++k) {
        d = fma(-al[k], d, (double)col[(k - 1) * TILE_X] * inv[k]);
        col[(k - 1) * TILE_X] = Real(d);
      }
    }
  }
  if (!active || Nz < k0) return;
  double x = d;                                                     // level Nz
  q[base + (long long)(Nz - 1) * g.sz] = Real(x);
  int k = Nz - 1;
  for (; k - UB + 1 >= k0; k -= UB) {
    double qv[UB], cv[UB];
#pragma unroll
    for (int u = 0; u < UB; ++u) { qv[u] = (double)col[(k - u - 1) * TILE_X]; cv[u] = cp[k - u]; }
#pragma unroll
    for (int u = 0; u < UB; ++u) { x = fma(-cv[u], x, qv[u]); q[base + (long long)(k - u - 1) * g.sz] = Real(x); }
  }
  for (; k >= k0; --k) {
    x = fma(-cp[k], x, (double)col[(k - 1) * TILE_X]);
    q[base + (long long)(k - 1) * g.sz] = Real(x);
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
  const size_t esz = g->dtype == OCN_F64 ? 8 : 4, tile_bytes = (size_t)g->Nz * (TILE_X * esz + 3 * sizeof(double)) + 8;
  if (tile_bytes <= 74 * 1024 && g->Ny <= 65535) {     // three 64-KB tiles per SM keep load, sweep and store phases of different blocks overlapped
    dim3 block(32, 1, 1), grid((g->Nx + TILE_X - 1) / TILE_X, g->Ny, a.nf);
    if (g->dtype == OCN_F64) {
      static OcnPerDeviceOnce once64;
      if (once64.first()) OCN_CUDA(cudaFuncSetAttribute(implicit_vdiff_tile_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, 74 * 1024));
      implicit_vdiff_tile_kernel<double><<<grid, block, tile_bytes, s>>>(g->dev, a, g->d_vdiff, g->nzm);
    } else {
      static OcnPerDeviceOnce once32;
      if (once32.first()) OCN_CUDA(cudaFuncSetAttribute(implicit_vdiff_tile_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 74 * 1024));
      implicit_vdiff_tile_kernel<float><<<grid, block, tile_bytes, s>>>(g->dev, a, g->d_vdiff, g->nzm);
    }
  } else {
    dim3 block(64, 2, 1), grid((g->Nx + 63) / 64, (g->Ny + 1) / 2, a.nf);
    if (g->dtype == OCN_F64) implicit_vdiff_kernel<double><<<grid, block, 0, s>>>(g->dev, a, g->d_vdiff, g->nzm);
    else implicit_vdiff_kernel<float><<<grid, block, 0, s>>>(g->dev, a, g->d_vdiff, g->nzm);
  }
  ocn_count_launch(2);
  return ocn_check_cuda(cudaGetLastError(), "implicit_vdiff_kernel launch");
}
