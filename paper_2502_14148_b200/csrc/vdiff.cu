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
// implicit_vdiff_tma_kernel (the default): a 32- (fp64) or 64-column (fp32) x Nz tile of one field is brought into shared memory by
// TMA, TWO warps eliminate from both ends of the column at once (two-sided / twisted factorisation), meet in the middle, substitute
// outwards in place and return the tile by TMA stores: 1 read + 1 write per field-cell, the compulsory traffic, and no global-memory
// instruction in the sweeps.  implicit_vdiff_tile_kernel (no TMA encoder / Ny > 65535): one warp per tile, cp.async in, plain stores
// out, one-sided.  implicit_vdiff_kernel (columns too tall for shared memory): one thread per column sweeping global memory in
// place, 2 reads + 2 writes.  Arithmetic in double for both storage types; all fields in one launch (blockIdx.z = field).
#include <cuda.h>
#include <cudaTypedefs.h>

#include <algorithm>
#include <cstring>

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

// pivots of combo c live at piv + c*6*nzm, k = 1..Nz at index k:
//   top-down elimination (the Thomas algorithm):  al[k] = lo_k inv_k, inv[k], cp[k] = up_k inv_k,        inv_k  = 1/(diag_k - lo_k cp_{k-1})
//   bottom-up elimination (its mirror image):     au[k] = up_k inv'_k, inv'[k], cl[k] = lo_k inv'_k,     inv'_k = 1/(diag_k - up_k cl_{k+1})
// The two-sided ("twisted") solve of implicit_vdiff_tma_kernel eliminates from both ends at once and needs both sets.
constexpr int NPIV = 6;
__global__ void vdiff_pivots_kernel(const GridDev g, const PivotArgs a, const double dt, double *__restrict__ piv, const int nzm) {
  const int c = threadIdx.x >> 1, up = threadIdx.x & 1;      // two threads per combo: top-down, bottom-up
  if (c >= a.ncombo) return;
  double *p0 = piv + (size_t)c * NPIV * nzm + (up ? 3 * nzm : 0), *p1 = p0 + nzm, *p2 = p1 + nzm;
  const bool face = a.face[c] != 0;
  const int k0 = face ? 2 : 1, Nz = g.Nz;
  const double s = -dt * a.kz[c];
  double cprev = 0.0;
  for (int t = 0; t <= Nz - k0; ++t) {
    const int k = up ? Nz - t : k0 + t;
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
    const double towards = up ? u : l, away = up ? l : u;   // coupling to the level already eliminated / to the next one
    const double iv = 1.0 / (diag - towards * cprev);
    cprev = away * iv;
    p0[k] = towards * iv; p1[k] = iv; p2[k] = cprev;
  }
}

// The same pivots, fast: one block per combo.  All threads first evaluate the matrix rows (lo_k, diag_k, up_k) of every level in
// parallel into shared memory (the metric loads and the two divisions per level leave the serial chain; the serial version above
// spent 95 us at Nz = 256, one L2 round trip per level), then one thread of warp 0 runs the top-down recurrence and one of warp 1 the
// bottom-up one from shared memory, with a Newton-refined MUFU reciprocal on the chain.
__device__ __forceinline__ double vd_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));   // ~20 good bits
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);                                     // three Newton steps: correctly rounded to within 1 ulp
}
__global__ void __launch_bounds__(256) vdiff_pivots_block_kernel(const GridDev g, const PivotArgs a, const double dt, double *__restrict__ piv,
                                                                 const int nzm) {
  extern __shared__ double rows[];                        // lo[Nz+1], diag[Nz+1], up[Nz+1] (index k)
  const int c = blockIdx.x, Nz = g.Nz;
  double *slo = rows, *sdg = rows + (Nz + 1), *sup = rows + 2 * (Nz + 1);
  const bool face = a.face[c] != 0;
  const int k0 = face ? 2 : 1;
  const double s = -dt * a.kz[c];
  for (int k = k0 + threadIdx.x; k <= Nz; k += blockDim.x) {
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
    slo[k] = l; sdg[k] = diag; sup[k] = u;
  }
  __syncthreads();
  if ((threadIdx.x & 31) != 0 || threadIdx.x >= 64) return;
  const int up = threadIdx.x >> 5;                        // warp 0: top-down set, warp 1: bottom-up set
  double *p0 = piv + (size_t)c * NPIV * nzm + (up ? 3 * nzm : 0), *p1 = p0 + nzm, *p2 = p1 + nzm;
  double cprev = 0.0;
  for (int t = 0; t <= Nz - k0; ++t) {
    const int k = up ? Nz - t : k0 + t;
    const double towards = up ? sup[k] : slo[k], away = up ? slo[k] : sup[k];   // coupling to the level already eliminated / to the next one
    const double iv = vd_rcp(fma(-towards, cprev, sdg[k]));
    cprev = away * iv;
    p0[k] = towards * iv; p1[k] = iv; p2[k] = cprev;
  }
}

template <class Real>
__global__ void __launch_bounds__(128) implicit_vdiff_kernel(const GridDev g, const VdiffArgs a, const double *__restrict__ piv,
                                                             const int nzm) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1, j = blockIdx.y * blockDim.y + threadIdx.y + 1, f = blockIdx.z;
  if (i > g.Nx || j > g.Ny) return;
  Real *__restrict__ q = (Real *)a.q[f];
  const double *lo = piv + (size_t)a.combo[f] * NPIV * nzm, *inv = lo + nzm, *cp = inv + nzm;
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
    const double *gp = piv + (size_t)a.combo[f] * NPIV * nzm;
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


// ---- TMA-fed tile kernel (the default) ----------------------------------------------------------------------------
// The tile moves by TMA in both directions: 3-D boxes of TX columns x 1 row x zb levels (cp.async.bulk.tensor, SASS UTMALDG /
// UTMASTG), each load completing on its own mbarrier.  History (C2 / C3 / C4 ms): one warp per tile with cp.async 1.33 / 0.51 / 1.33,
// one warp with TMA loads 1.32 / 0.495 / 1.48 (bound by the in-order issue rate of ONE warp per scheduler: three 64-KB tiles per
// SM), two warps + two-sided elimination 1.07 / 0.50 / -, + TMA stores and everything requested up front 1.04 / 0.47 / 1.32
// (79 % / 90 % / 74 % of the measured copy peak).
struct VdiffTmaArgs {
  CUtensorMap tmap[MAXF];
  VdiffArgs v;
  int zb;            // levels per TMA chunk
  int nchunk;
  int win;           // chunks kept in flight
  int xa_off, ya_off, za_off;   // array coordinates of logical (i, j, k) = (i + xa_off, j + ya_off, k + za_off)
};
constexpr int VD_MAXCHUNK = 16;

__device__ __forceinline__ unsigned vd_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// Two warps per tile, TWO-SIDED elimination: warp 0 eliminates downwards-coupled terms from the bottom level k0 up to the
// split level m, warp 1 the mirror image from the top level Nz down to m+1 (the "twisted" factorisation of a tridiagonal
// matrix: exact in exact arithmetic, as stable as the Thomas algorithm for these diagonally dominant matrices); the two meet in
// a 2 x 2 system for (x_m, x_{m+1}) and substitute outwards IN PLACE; every chunk returns to global memory by one TMA store as
// soon as its last level is final.  The dependent chain per warp is half as long, twice as many loads are in flight per tile and
// the warps issue no global-memory instruction at all (ncu r1/r2: one warp per 64-KB tile left the kernel bound by the in-order
// issue rate of a single warp per scheduler, 58 % of the copy peak at Nz = 256).  A lane owns CPL adjacent columns (fp64: 1,
// fp32: 2 = two independent chains per thread and 256-byte rows), TX = 32 CPL columns per tile.
template <class Real, int CPL> struct VdVec;
template <> struct VdVec<double, 1> { using T = double; };
template <> struct VdVec<float, 2> { using T = float2; };
template <> struct VdVec<float, 1> { using T = float; };
__device__ __forceinline__ void vd_unpack(double v, double (&o)[1]) { o[0] = v; }
__device__ __forceinline__ void vd_unpack(float v, double (&o)[1]) { o[0] = (double)v; }
__device__ __forceinline__ void vd_unpack(float2 v, double (&o)[2]) { o[0] = (double)v.x; o[1] = (double)v.y; }
__device__ __forceinline__ void vd_pack(const double (&i)[1], double &v) { v = i[0]; }
__device__ __forceinline__ void vd_pack(const double (&i)[1], float &v) { v = (float)i[0]; }
__device__ __forceinline__ void vd_pack(const double (&i)[2], float2 &v) { v = make_float2((float)i[0], (float)i[1]); }

template <class Real, int CPL>
__global__ void __launch_bounds__(64) implicit_vdiff_tma_kernel(const GridDev g, const __grid_constant__ VdiffTmaArgs a,
                                                                const double *__restrict__ piv, const int nzm) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  using V = typename VdVec<Real, CPL>::T;
  constexpr int UB = 16 / CPL, TX = 32 * CPL;
  const int Nz = g.Nz;
  Real *tile = (Real *)smem_raw;                                   // [nchunk * zb][TX], chunk c at c * zb * TX (128-byte aligned)
  double *spiv = (double *)(tile + (size_t)a.nchunk * a.zb * TX);  // three pivot arrays of this field (index k-1), see below
  unsigned long long *bar = (unsigned long long *)(spiv + ((3 * Nz + 1) & ~1));
  const int f = blockIdx.z, j = blockIdx.y + 1, i0 = blockIdx.x * TX + 1, lane = threadIdx.x, up = threadIdx.y;
  const int k0 = a.v.face[f] ? 2 : 1;
  V *col = reinterpret_cast<V *>(tile) + lane;                     // this lane's CPL columns; levels are 32 V apart
  const int cA = (a.nchunk + 1) / 2;                               // chunks 0 .. cA-1 belong to warp 0, cA .. nchunk-1 to warp 1
  const int m = min(cA * a.zb, Nz);                                // warp 0: levels k0 .. m; warp 1: levels Nz .. m+1
  const unsigned chunk_bytes = (unsigned)(a.zb * TX * sizeof(Real));
  auto issue_chunk = [&](int c) {      // lane 0 only
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(vd_smem_u32(&bar[c])), "r"(chunk_bytes) : "memory");
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     vd_smem_u32(tile + (size_t)c * a.zb * TX)),
                 "l"(&a.tmap[f]), "r"(i0 + a.xa_off), "r"(j + a.ya_off), "r"(1 + c * a.zb + a.za_off), "r"(vd_smem_u32(&bar[c]))
                 : "memory");
  };
  const int win = a.win;               // chunks in flight per warp
  if (lane == 0 && up == 0) {
    for (int c = 0; c < a.nchunk; ++c) asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(vd_smem_u32(&bar[c])), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (lane == 0) {
    if (!up) for (int c = 0; c < min(win, cA); ++c) issue_chunk(c);
    else for (int c = a.nchunk - 1; c >= max(a.nchunk - win, cA); --c) issue_chunk(c);
  }
  {   // the pivots of this field (a few KB, L2-resident): levels <= m take the top-down set, levels > m the bottom-up set
    const double *gp = piv + (size_t)a.v.combo[f] * NPIV * nzm;
    for (int t = lane + 32 * up; t < 3 * Nz; t += 64) {
      const int arr = t / Nz, k = t % Nz + 1;
      spiv[t] = gp[(arr + (k > m ? 3 : 0)) * nzm + k];
    }
  }
  __syncthreads();
  const double *al = spiv - 1, *inv = al + Nz, *cp = inv + Nz;      // indexed by k: coupling to the eliminated side, 1/pivot, coupling to the other side
  auto wait_chunk = [&](int c) {
    unsigned done;
    do {
      asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\nselp.u32 %0, 1, 0, p;\n}\n"
                   : "=r"(done) : "r"(vd_smem_u32(&bar[c])), "r"(0u), "r"(20000u) : "memory");
    } while (!done);
  };
  // ---- elimination sweeps: d_k = q_k inv_k - al_k d_{k -+ 1}, warp 0 upwards from k0, warp 1 downwards from Nz
  const int sgn = up ? -1 : 1;
  const int kfirst = up ? Nz : k0, klast = up ? m + 1 : m;          // this warp's levels, in sweep order
  const int nlev = (klast - kfirst) * sgn + 1;                      // <= 0: nothing (warp 1 of a one-chunk tile)
  double d[CPL];
#pragma unroll
  for (int c = 0; c < CPL; ++c) d[c] = 0.0;
  {
    int cnext = up ? a.nchunk - 1 : 0;                              // next chunk (in sweep order) that has not been waited for
    for (int t0 = 0; t0 < nlev; t0 += UB) {
      const int ka = kfirst + sgn * t0, nb = min(UB, nlev - t0), kend = ka + sgn * (nb - 1);
      const int cneed = (kend - 1) / a.zb;
      while (up ? cnext >= cneed : cnext <= cneed) {
        wait_chunk(cnext);
        const int cn = cnext + sgn * win;
        if (lane == 0 && (up ? cn >= cA : cn < cA)) issue_chunk(cn);
        cnext += sgn;
      }
      if (nb == UB) {
        double qv[UB][CPL], av[UB];
#pragma unroll
        for (int u = 0; u < UB; ++u) {
          vd_unpack(col[(ka + sgn * u - 1) * 32], qv[u]);
          const double iv = inv[ka + sgn * u];
#pragma unroll
          for (int c = 0; c < CPL; ++c) qv[u][c] *= iv;
          av[u] = al[ka + sgn * u];
        }
#pragma unroll
        for (int u = 0; u < UB; ++u) {
#pragma unroll
          for (int c = 0; c < CPL; ++c) d[c] = fma(-av[u], d[c], qv[u][c]);
          vd_pack(d, col[(ka + sgn * u - 1) * 32]);
        }
      } else {
        for (int u = 0; u < nb; ++u) {
          const int k = ka + sgn * u;
          double qk[CPL];
          vd_unpack(col[(k - 1) * 32], qk);
#pragma unroll
          for (int c = 0; c < CPL; ++c) d[c] = fma(-al[k], d[c], qk[c] * inv[k]);
          vd_pack(d, col[(k - 1) * 32]);
        }
      }
    }
  }
  __syncthreads();                                                  // d_m (warp 0) and d_{m+1} (warp 1) are in the tile
  if (Nz < k0) return;
  // ---- the 2 x 2 system where the sweeps meet:  x_m + cp_m x_{m+1} = d_m,   cl_{m+1} x_m + x_{m+1} = d_{m+1}
  double x[CPL];
  if (m < Nz) {
    double dm[CPL], dm1[CPL];
    vd_unpack(col[(m - 1) * 32], dm);
    vd_unpack(col[m * 32], dm1);
    __syncthreads();                                                // both warps have read both values before either overwrites its own
    const double rden = 1.0 / (1.0 - cp[m] * cp[m + 1]);
#pragma unroll
    for (int c = 0; c < CPL; ++c) {
      const double xm = (dm[c] - cp[m] * dm1[c]) * rden;
      x[c] = up ? fma(-cp[m + 1], xm, dm1[c]) : xm;
    }
  } else {
#pragma unroll
    for (int c = 0; c < CPL; ++c) x[c] = d[c];                      // single-sided (one chunk): the last level of the Thomas sweep
    if (up) return;
  }
  // ---- substitution outwards from the meeting point, x_k = d_k - cp_k x_{k +- 1}, IN PLACE in the tile; every chunk goes back to
  // global memory with one TMA store as soon as its last level is final (the tensor map ends at the last interior column and
  // level, so ragged tiles and the levels above Nz are clipped by the hardware; level 1 of a face field is stored back unchanged).
  int cst = up ? cA : cA - 1;                                       // next chunk (in substitution order) to store
  auto flush = [&](int knext, bool fin) {
    while (up ? (cst < a.nchunk && (fin || knext > (cst + 1) * a.zb)) : (cst >= 0 && (fin || knext <= cst * a.zb))) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) {
        asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(&a.tmap[f]), "r"(i0 + a.xa_off),
                     "r"(j + a.ya_off), "r"(1 + cst * a.zb + a.za_off), "r"(vd_smem_u32(tile + (size_t)cst * a.zb * TX))
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      }
      cst -= sgn;
    }
  };
  int k = klast;
  vd_pack(x, col[(k - 1) * 32]);
  k -= sgn;
  for (; (k - kfirst) * sgn >= UB - 1; k -= sgn * UB) {
    flush(k, false);
    double qv[UB][CPL], cv[UB];
#pragma unroll
    for (int u = 0; u < UB; ++u) { vd_unpack(col[(k - sgn * u - 1) * 32], qv[u]); cv[u] = cp[k - sgn * u]; }
#pragma unroll
    for (int u = 0; u < UB; ++u) {
#pragma unroll
      for (int c = 0; c < CPL; ++c) x[c] = fma(-cv[u], x[c], qv[u][c]);
      vd_pack(x, col[(k - sgn * u - 1) * 32]);
    }
  }
  flush(k, false);
  for (; (k - kfirst) * sgn >= 0; k -= sgn) {
    double qk[CPL];
    vd_unpack(col[(k - 1) * 32], qk);
#pragma unroll
    for (int c = 0; c < CPL; ++c) x[c] = fma(-cp[k], x[c], qk[c]);
    vd_pack(x, col[(k - 1) * 32]);
  }
  flush(k, true);
  if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the tile must outlive the bulk reads
}

template <class Real>
int launch_vdiff_tma(const ocn_grid *g, const VdiffArgs &va, cudaStream_t s, bool *done) {
  *done = false;
  constexpr int CPL = sizeof(Real) == 8 ? 1 : 2, TX = 32 * CPL;
  auto enc = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(ocn_tensormap_encoder());
  if (!enc || g->Ny > 65535) return OCN_OK;
  VdiffTmaArgs a;
  memset(&a, 0, sizeof(a));
  a.v = va;
  const int Nz = g->Nz;
  // chunk = >= 16 levels, about an eighth of the column, a multiple of 8 levels (chunk bytes a multiple of 128); everything is
  // requested up front: with TMA stores the tiles of an SM drift out of phase by themselves (measured at C2, chunk x window:
  // 16 x 4 1.13 ms, 32 x 2 1.09, 32 x 4 (all) 1.04, 64 x 2 (all) 1.04; C3: 8 x 4 0.51, 16 x 4 (all) 0.47)
  int zb = std::max(16, (((Nz + 7) / 8 + 7) / 8) * 8);
  if (zb > 256) return OCN_OK;                                   // TMA box limit: fall back for columns taller than 2048 levels
  a.zb = zb;
  a.nchunk = (Nz + zb - 1) / zb;
  if (a.nchunk > VD_MAXCHUNK) return OCN_OK;
  a.win = a.nchunk;
  const size_t tile_bytes = (size_t)a.nchunk * zb * TX * sizeof(Real) + ((3 * Nz + 1) & ~1) * sizeof(double) + VD_MAXCHUNK * sizeof(unsigned long long);
  if (tile_bytes > 75 * 1024) return OCN_OK;                     // three tiles per SM
  const ocn_layout &L = g->lay;
  const int xoff = (int)(L.offset0 - (long long)L.hz * L.stride_z - (long long)L.hy * L.stride_y);   // array x of logical i = 1
  for (int f = 0; f < va.nf; ++f) {
    // the tensor ends at the last interior column and level: loads beyond are zero-filled, stores beyond are dropped
    cuuint64_t dims[3] = {(cuuint64_t)(xoff + g->Nx), (cuuint64_t)L.ny_pad, (cuuint64_t)(L.hz + Nz)};
    cuuint64_t strides[2] = {(cuuint64_t)L.stride_y * sizeof(Real), (cuuint64_t)L.stride_z * sizeof(Real)};
    cuuint32_t box[3] = {(cuuint32_t)TX, 1, (cuuint32_t)zb};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(&a.tmap[f], sizeof(Real) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, va.q[f], dims, strides,
                     box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return ocn_fail(OCN_ERR_CUDA, "implicit_vdiff: cuTensorMapEncodeTiled failed (%d) for field %d", (int)r, f);
  }
  a.xa_off = xoff - 1; a.ya_off = L.hy - 1; a.za_off = L.hz - 1;
  static OcnPerDeviceOnce once;
  if (once.first()) OCN_CUDA(cudaFuncSetAttribute(implicit_vdiff_tma_kernel<Real, CPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, 75 * 1024));
  dim3 block(32, 2, 1), grid((g->Nx + TX - 1) / TX, g->Ny, va.nf);
  implicit_vdiff_tma_kernel<Real, CPL><<<grid, block, tile_bytes, s>>>(g->dev, a, g->d_vdiff, g->nzm);
  *done = true;
  return OCN_OK;
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
  if ((size_t)3 * (g->Nz + 1) * sizeof(double) <= 48 * 1024)
    vdiff_pivots_block_kernel<<<pa.ncombo, 256, 3 * (g->Nz + 1) * sizeof(double), s>>>(g->dev, pa, dt, g->d_vdiff, g->nzm);
  else
    vdiff_pivots_kernel<<<1, 64, 0, s>>>(g->dev, pa, dt, g->d_vdiff, g->nzm);
  OCN_CUDA(cudaGetLastError());
  {
    bool done = false;
    const int rc = g->dtype == OCN_F64 ? launch_vdiff_tma<double>(g, a, s, &done) : launch_vdiff_tma<float>(g, a, s, &done);
    if (rc) return rc;
    if (done) {
      ocn_count_launch(2);
      return ocn_check_cuda(cudaGetLastError(), "implicit_vdiff_tma_kernel launch");
    }
  }
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
