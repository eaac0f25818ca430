// tend_fused.cu — OCN_KERNEL_FUSED: the fused tendency kernel for 3-D grids with WENO5 in x,y.
//
// 2.5-D blocking.  A block of 32 x (TY+1) threads owns a 31 x TY tile of (i,j) columns and marches along z:
//   * plane k of every input field, with a 3-cell halo, is staged in shared memory by ONE TMA tiled load per field
//     (cp.async.bulk.tensor.3d + mbarrier complete_tx), three planes in flight (ring of 3 buffers);
//   * the z-stencil of every field lives in a register window q(k-3..k+2) that slides one plane per iteration
//     (own-column values come from coalesced global loads issued one plane ahead);
//   * EVERY FACE FLUX IS COMPUTED ONCE: a thread computes the fluxes through the LOW x-, y- and z-face of its
//     control volumes; the high-face values come from lane+1 (warp shuffle), from row+1 (shared memory) and from the
//     next plane (the z-march is lagged by one plane: iteration k completes and stores plane k-1).  Lane 31 and row TY
//     are "ghost" threads that only supply those fluxes (row TY skips everything but its y-fluxes).
//   * tracers use the cancellation-free form (H1): flux anomalies relative to the low-side cell plus
//     c * div(u) with div(u) accumulated in double-double.
// Operators and citations are those of tend_percell.cu: (B2),(B3),(B8),(B9),(B21), eq. 6/8/9/17.
#include <cuda.h>
#include <cudaTypedefs.h>

#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <cstring>

#include "ocn_internal.h"
#include "recon.cuh"

namespace {

using namespace ocn;

constexpr int NBUF = 3;          // TMA ring depth (planes in flight)
constexpr int MAXF = 3 + 3;      // u, v, w + up to 3 tracers in the fused instantiations

template <class Real>
struct FusedArgs {
  CUtensorMap tmap[MAXF];        // one 3-D tiled map per input field: dims (pitch, ny_pad, nz_pad), box (TW, TY+6, 1)
  GridDev g;
  ModelDev m;
  const Real *q[MAXF];           // u, v, w, c0..  (own-column loads)
  const Real *phy;
  Real *G[MAXF];
  int xa_off, ya_off, za_off;    // array coordinates of logical (i,j,k) = (i + xa_off, j + ya_off, k + za_off)
  int kchunk;                    // planes per block along z
};

// ---- mbarrier / TMA primitives (PTX; SASS: SYNCS.*, UTMALDG) ------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int x, int y, int z, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
      : "memory");
}

__device__ __forceinline__ double shfl_down1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_down1(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }

template <class Real> struct TileGeom {
  static constexpr int TW = sizeof(Real) == 8 ? 38 : 40;   // box row: 37 columns (i0-3 .. i0+33) + start alignment slack; bytes % 16 == 0
};

template <class Real, int NT, int TY>
struct SmemLayout {
  static constexpr int NF = 3 + NT;
  static constexpr int TW = TileGeom<Real>::TW;
  static constexpr int TH = TY + 6;
  static constexpr int FS = ((TW * TH * (int)sizeof(Real) + 127) / 128) * 128 / (int)sizeof(Real);   // field stride (elements)
  static constexpr int TILE_ELEMS = NBUF * NF * FS;
  static constexpr int FY_SLOT = NF * (TY + 1) * 32;                    // y-face fluxes of one plane
  static constexpr int FY_ELEMS = NBUF * FY_SLOT;
  static constexpr int NBAR = NBUF * (2 + 2 * (TY + 1));                // full, empty, fy-ready per role and row
  static constexpr size_t BYTES = (size_t)(TILE_ELEMS + FY_ELEMS) * sizeof(Real) + NBAR * sizeof(uint64_t);
  static constexpr uint32_t PLANE_BYTES = (uint32_t)(NF * TW * TH * sizeof(Real));
};

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void mbar_wait_backoff(uint64_t *bar, uint32_t parity) {
  // for warps that are expected to wait long (ghost rows, the producer): do not burn issue slots while spinning
  uint32_t done;
  for (;;) {
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    if (done) break;
    __nanosleep(200);
  }
}

// Upwind-selected five-point stencils of N fields by ADDRESS selection (no value selects): hi[n] points at the
// element on the high side of the face (index m), step is the element stride along the flux direction.
// Left-biased (vel > 0): (a..e) = q[m-3 .. m+1]; right-biased: the mirror image q[m+2 .. m-2]  (reading R3).
template <class Real, int N>
__device__ __forceinline__ void upwind_diffs(const Real *const (&hi)[N], int step, const Real (&vel)[N], Real (&d1)[N],
                                             Real (&d2)[N], Real (&d3)[N], Real (&d4)[N], Real (&cc)[N]) {
#pragma unroll
  for (int n = 0; n < N; ++n) {
    const bool pos = vel[n] > Real(0);
    const int s = pos ? step : -step;
    const Real *c = pos ? hi[n] - step : hi[n];
    const Real qa = c[-2 * s], qb = c[-s], qc = c[0], qd = c[s], qe = c[2 * s];
    d1[n] = qb - qa; d2[n] = qc - qb; d3[n] = qd - qc; d4[n] = qe - qd;
    cc[n] = qc;
  }
}
// the same for N fields advected by ONE velocity (tracers): fields are `fs` elements apart
template <class Real, int N>
__device__ __forceinline__ void upwind_diffs_shared(const Real *hi0, int fs, int step, Real vel, Real (&d1)[N], Real (&d2)[N],
                                                    Real (&d3)[N], Real (&d4)[N], Real (&cc)[N]) {
  const bool pos = vel > Real(0);
  const int s = pos ? step : -step;
  const Real *c = pos ? hi0 - step : hi0;
#pragma unroll
  for (int n = 0; n < N; ++n) {
    const Real *cn = c + n * fs;
    const Real qa = cn[-2 * s], qb = cn[-s], qc = cn[0], qd = cn[s], qe = cn[2 * s];
    d1[n] = qb - qa; d2[n] = qc - qb; d3[n] = qd - qc; d4[n] = qe - qd;
    cc[n] = qc;
  }
}
// from a register window w[0..5] = q[m-3 .. m+2] (value selects)
template <class Real>
__device__ __forceinline__ void window_diffs(const Real (&w)[6], Real vel, Real &d1, Real &d2, Real &d3, Real &d4, Real &cc) {
  const bool pos = vel > Real(0);
  const Real qa = pos ? w[0] : w[5], qb = pos ? w[1] : w[4], qc = pos ? w[2] : w[3], qd = pos ? w[3] : w[2], qe = pos ? w[4] : w[1];
  d1 = qb - qa; d2 = qc - qb; d3 = qd - qc; d4 = qe - qd;
  cc = qc;
}

// Block = two warps per tile row, specialised by FIELD GROUP (role 0: tracers, role 1: momentum), each with its own
// ghost-row warp, + 1 producer warp (TMA).  A thread keeps the z-windows of its own group only, which is what lets
// 15-19 warps fit the register file (the FP64 pipe needs >= 4 independent DFMAs in flight per scheduler: measured
// dependent-issue latency 8.6 cycles, issue interval 2.18).  No __syncthreads in the plane loop:
//   TMA -> full[slot];  every consumer warp -> empty[slot];  row r of a role -> fyr[slot][role][r].
template <class Real, int NT, int SZ, bool HYDRO, int TY>
__global__ void __launch_bounds__(32 * (2 * TY + 3), 1) tend_fused_kernel(const __grid_constant__ FusedArgs<Real> a) {
  using SL = SmemLayout<Real, NT, TY>;
  constexpr int NF = SL::NF, TW = SL::TW, FS = SL::FS;
  constexpr int ZL = SZ == 5 ? 3 : 1, ZH = SZ == 5 ? 2 : 1, WD = ZL + ZH + 1;
  constexpr int FU = 0, FV = 1, FW = 2, FC = 3;
  constexpr int NM = HYDRO ? 2 : 3;                      // momentum components that carry a tendency
  constexpr int IA = SZ == 5 ? S_WENO5 : S_CENTERED2;   // interpolation order of the velocity advecting through z-faces (R4)
  constexpr int NR = TY + 1;                             // rows per role (incl. the ghost row)

  extern __shared__ __align__(1024) unsigned char smem_raw[];
  Real *tile = reinterpret_cast<Real *>(smem_raw);
  Real *fyb = tile + SL::TILE_ELEMS;
  uint64_t *full = reinterpret_cast<uint64_t *>(fyb + SL::FY_ELEMS);
  uint64_t *empty = full + NBUF;
  uint64_t *fyr = empty + NBUF;                          // [NBUF][2][NR]

  const GridDev &g = a.g;
  const ModelDev &m = a.m;
  const int lane = threadIdx.x, wid = threadIdx.y;
  const int i0 = blockIdx.x * 31 + 1, j0 = blockIdx.y * TY + 1;
  const int kc0 = 1 + blockIdx.z * a.kchunk;
  const int kc1 = min(kc0 + a.kchunk, g.Nz + 1);          // completion-only iteration

  if (lane == 0 && wid == 0) {
    for (int b = 0; b < NBUF; ++b) {
      mbar_init(&full[b], 1);
      mbar_init(&empty[b], 2 * NR);
      for (int r = 0; r < 2 * NR; ++r) mbar_init(&fyr[b * 2 * NR + r], 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  constexpr int XA = 16 / (int)sizeof(Real);
  if (wid == 2 * NR) {
    // ------------------------------------------------ producer warp: one lane feeds the TMA ring
    if (lane == 0) {
      // TMA needs the innermost start coordinate on a 16-byte boundary (measured: an odd fp64 x raises "illegal
      // instruction" on sm_100a): start the box at the aligned column at or left of i0-3; the readers shift by xs.
      const int tx0 = ((i0 - 3 + a.xa_off) / XA) * XA, ty0 = j0 - 3 + a.ya_off;
      for (int k = kc0, it = 0; k <= kc1; ++k, ++it) {
        const int b = it % NBUF;
        if (it >= NBUF) mbar_wait_backoff(&empty[b], (uint32_t)(((it / NBUF) - 1) & 1));
        mbar_expect_tx(&full[b], SL::PLANE_BYTES);
#pragma unroll
        for (int f = 0; f < NF; ++f) tma_load_3d(tile + (b * NF + f) * FS, &a.tmap[f], tx0, ty0, k + a.za_off, &full[b]);
      }
    }
    return;
  }

  const int role = wid / NR, row = wid - role * NR;
  const int xs = (i0 - 3 + a.xa_off) % XA;
  const int i = i0 + lane, j = j0 + row;
  const bool ghost_row = row == TY;
  const bool can_store = lane < 31 && !ghost_row && i <= g.Nx && j <= g.Ny;
  // own-column address (clamped inside the padded array for threads beyond the ragged edge; never stored)
  const int il = min(i, g.Nx + g.Hx), jl = min(j, g.Ny + g.Hy);
  const long long sz = g.sz;
  long long o = g.idx(il, jl, kc0);                        // offset of (i,j,k) for the current k
  const Real eps4 = Real(4.0 * m.weno_eps);
  const Real rdx = Real(g.rdx), rdy = Real(g.rdy);
  const Real rdx2 = Real(g.rdx * g.rdx), rdy2 = Real(g.rdy * g.rdy);
  uint64_t *my_fyr = fyr + role * NR + row;               // + b * 2 * NR

#define ZMETRICS                                                                                          \
  const int zk = g.zi(k);                                                                                 \
  Real rdzc_k, rdzc_km, rdzf_k, rdzf_kp, rdzf_km;                                                         \
  if (g.uniform_z) {                                                                                      \
    rdzc_k = rdzc_km = rdzf_k = rdzf_kp = rdzf_km = Real(g.rdz);                                          \
  } else {                                                                                                \
    rdzc_k = Real(g.rdzc[zk]); rdzc_km = Real(g.rdzc[zk - 1]);                                            \
    rdzf_k = Real(g.rdzf[zk]); rdzf_kp = Real(g.rdzf[zk + 1]); rdzf_km = Real(g.rdzf[zk - 1]);            \
  }                                                                                                       \
  (void)rdzf_km; (void)rdzf_k; (void)rdzf_kp; (void)rdzc_km;
#define S(f, di, dj) T[(f) * FS + (dj) * TW + (di)]

  if (role == 0) {
    // =========================================================================================== TRACERS
    constexpr int N = NT > 0 ? NT : 1;
    Real win[N][WD], pf[N], part[N];
#pragma unroll
    for (int n = 0; n < NT; ++n) {
#pragma unroll
      for (int t = 0; t < WD; ++t) win[n][t] = __ldg(a.q[FC + n] + o + (long long)(t - ZL) * sz);
      part[n] = Real(0);
    }
    Real wk1 = __ldg(a.q[FW] + o + sz), wpf = Real(0);      // w(k+1), needed by div(u)
    for (int k = kc0, it = 0; k <= kc1; ++k, ++it, o += sz) {
      const int b = it % NBUF;
      const uint32_t ph = (uint32_t)((it / NBUF) & 1);
      const bool more = k < kc1;
      if (more) {
#pragma unroll
        for (int n = 0; n < NT; ++n) pf[n] = __ldg(a.q[FC + n] + o + (long long)(ZH + 1) * sz);
        wpf = __ldg(a.q[FW] + o + 2 * sz);
      }
      ZMETRICS
      if (ghost_row) mbar_wait_backoff(&full[b], ph); else mbar_wait(&full[b], ph);
      const Real *T = tile + b * NF * FS + (row + 3) * TW + lane + 3 + xs;
      Real *fy = fyb + b * SL::FY_SLOT + row * 32 + lane;
      const Real ui = S(FU, 0, 0), vj = S(FV, 0, 0), wk = S(FW, 0, 0);
      Real acc[N];
      // ---- (A) low y-face (face j): F~ = v (recon - c(j-1)); published first
      if (more) {
        Real d1[N], d2[N], d3[N], d4[N], cc[N], r[N];
        upwind_diffs_shared<Real, N>(&S(FC, 0, 0), FS, TW, vj, d1, d2, d3, d4, cc);
        weno5z_anom_v<N>(d1, d2, d3, d4, eps4, r);
#pragma unroll
        for (int n = 0; n < NT; ++n) {
          const Real cm = S(FC + n, 0, -1);
          const Real F = vj * (r[n] + (cc[n] - cm));
          fy[(FC + n) * NR * 32] = F;
          acc[n] = (F + vj * (cm - win[n][ZL])) * rdy;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(my_fyr + b * 2 * NR);
      }
      if (!ghost_row) {
        // ---- (B) low z-face (face k); completes plane k-1
        Real Fz[N];
        if constexpr (SZ == 5) {
          Real d1[N], d2[N], d3[N], d4[N], cc[N], r[N];
#pragma unroll
          for (int n = 0; n < NT; ++n) window_diffs<Real>(win[n], wk, d1[n], d2[n], d3[n], d4[n], cc[n]);
          weno5z_anom_v<N>(d1, d2, d3, d4, eps4, r);
#pragma unroll
          for (int n = 0; n < NT; ++n) Fz[n] = wk * (r[n] + (cc[n] - win[n][ZL - 1]));
        } else {
#pragma unroll
          for (int n = 0; n < NT; ++n) Fz[n] = wk * (Real(0.5) * (win[n][1] - win[n][0]));     // Centered(2) minus c(k-1)
        }
        if (it > 0 && can_store) {
#pragma unroll
          for (int n = 0; n < NT; ++n) a.G[FC + n][o - sz] = part[n] - Fz[n] * rdzc_km;
        }
        if (more) {
#pragma unroll
          for (int n = 0; n < NT; ++n) acc[n] += (Fz[n] + wk * (win[n][ZL - 1] - win[n][ZL])) * rdzc_k;
        }
      }
      if (!more) break;
      if (!ghost_row) {
        // ---- (C) low x-face (face i); high face from lane+1
        {
          Real d1[N], d2[N], d3[N], d4[N], cc[N], r[N];
          upwind_diffs_shared<Real, N>(&S(FC, 0, 0), FS, 1, ui, d1, d2, d3, d4, cc);
          weno5z_anom_v<N>(d1, d2, d3, d4, eps4, r);
#pragma unroll
          for (int n = 0; n < NT; ++n) {
            const Real cm = S(FC + n, -1, 0);
            const Real F = ui * (r[n] + (cc[n] - cm));
            const Real Fh = shfl_down1(F);
            acc[n] -= (Fh - F - ui * (cm - win[n][ZL])) * rdx;
          }
        }
        // ---- c * div(u) with div(u) in double-double (H1), diffusion
        {
          double rdzc_kd, rdzc_klo;
          if (g.uniform_z) { rdzc_kd = g.rdz; rdzc_klo = g.rdz_lo; } else { rdzc_kd = g.rdzc[zk]; rdzc_klo = g.rdzc_lo[zk]; }
          double D = 0.0, Dlo = 0.0;
          dd_add_diff_scaled((double)S(FU, 1, 0), (double)ui, g.rdx, g.rdx_lo, D, Dlo);
          dd_add_diff_scaled((double)S(FV, 0, 1), (double)vj, g.rdy, g.rdy_lo, D, Dlo);
          dd_add_diff_scaled((double)wk1, (double)wk, rdzc_kd, rdzc_klo, D, Dlo);
          const double Dsum = D + Dlo;
#pragma unroll
          for (int n = 0; n < NT; ++n) {
            const int f = FC + n;
            const Real c0 = win[n][ZL];
            Real lap = ((S(f, 1, 0) - c0) - (c0 - S(f, -1, 0))) * rdx2 + ((S(f, 0, 1) - c0) - (c0 - S(f, 0, -1))) * rdy2;
            lap += ((win[n][ZL + 1] - c0) * rdzf_kp - (c0 - win[n][ZL - 1]) * rdzf_k) * rdzc_k;
            acc[n] += Real(m.kappa[n]) * lap - Real((double)c0 * Dsum);
          }
        }
        // ---- high y-face fluxes from row+1
        mbar_wait(my_fyr + b * 2 * NR + 1, ph);
#pragma unroll
        for (int n = 0; n < NT; ++n) acc[n] -= fy[(FC + n) * NR * 32 + 32] * rdy;
      }
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        part[n] = acc[n];
#pragma unroll
        for (int t = 0; t < WD - 1; ++t) win[n][t] = win[n][t + 1];
        win[n][WD - 1] = pf[n];
      }
      wk1 = wpf;
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[b]);
    }
  } else {
    // =========================================================================================== MOMENTUM
    Real win[NM][WD], pf[NM], part[NM];
#pragma unroll
    for (int n = 0; n < NM; ++n) {
#pragma unroll
      for (int t = 0; t < WD; ++t) win[n][t] = __ldg(a.q[n] + o + (long long)(t - ZL) * sz);
      part[n] = Real(0);
    }
    // buoyancy of the level below (b = g[alpha (T - Tref) - beta (S - Sref)], reading R9), carried along the march
    auto buoy = [&](Real Tv, Real Sv, int zz) -> double {
      const double Ta = m.idx_T >= 0 ? (double)Tv - g.Tref[zz] : 0.0;
      const double Sa = m.idx_S >= 0 ? (double)Sv - g.Sref[zz] : 0.0;
      return m.g * (m.alpha_T * Ta - m.beta_S * Sa);
    };
    double b_km = 0.0;
    if (!HYDRO && m.buoyancy)
      b_km = buoy(__ldg(a.q[FC] + o - sz), NT > 1 ? __ldg(a.q[FC + (NT > 1 ? 1 : 0)] + o - sz) : Real(0), g.zi(kc0) - 1);
    const Real fu = Real(m.f0 + m.beta * ((j - 0.5) * g.dy - m.y0));      // f at the u point (y_c[j]), R8
    const Real fv = Real(m.f0 + m.beta * ((j - 1.0) * g.dy - m.y0));      // f at the v point (y_f[j])
    const Real nu = Real(m.nu);
    const bool wall_u = g.topo[0] == OCN_BOUNDED && i == 1;
    const bool wall_v = g.topo[1] == OCN_BOUNDED && j == 1;
    for (int k = kc0, it = 0; k <= kc1; ++k, ++it, o += sz) {
      const int b = it % NBUF;
      const uint32_t ph = (uint32_t)((it / NBUF) & 1);
      const bool more = k < kc1;
      if (more) {
#pragma unroll
        for (int n = 0; n < NM; ++n) pf[n] = __ldg(a.q[n] + o + (long long)(ZH + 1) * sz);
      }
      ZMETRICS
      if (ghost_row) mbar_wait_backoff(&full[b], ph); else mbar_wait(&full[b], ph);
      const Real *T = tile + b * NF * FS + (row + 3) * TW + lane + 3 + xs;
      Real *fy = fyb + b * SL::FY_SLOT + row * 32 + lane;
      const Real ui = win[FU][ZL], vj = win[FV][ZL], wk = S(FW, 0, 0);
      Real acc[NM];
      // ---- (A) low y-face fluxes, published first
      if (more) {
        const Real *hi[NM];
        Real vl[NM], d1[NM], d2[NM], d3[NM], d4[NM], cc[NM], r[NM];
        hi[FU] = &S(FU, 0, 0);                                                                      // u along y at (i-1/2, j-1/2)
        vl[FU] = interp_adv<Real>(S_WENO5, S(FV, -2, 0), S(FV, -1, 0), vj, S(FV, 1, 0));            // v~: Centered(4) along x (B21)
        hi[FV] = &S(FV, 0, 0);                                                                      // v at the centre j-1 (m = j)
        vl[FV] = interp_adv<Real>(S_WENO5, S(FV, 0, -2), S(FV, 0, -1), vj, S(FV, 0, 1));
        if constexpr (!HYDRO) {
          hi[FW] = &S(FW, 0, 0);                                                                    // w along y at (j-1/2, k-1/2)
          vl[FW] = interp_adv<Real>(S_WENO5, win[FV][ZL - 2], win[FV][ZL - 1], vj, win[FV][ZL + 1]);   // v~ along z
        }
        upwind_diffs<Real, NM>(hi, TW, vl, d1, d2, d3, d4, cc);
        weno5z_anom_v<NM>(d1, d2, d3, d4, eps4, r);
#pragma unroll
        for (int n = 0; n < NM; ++n) {
          const Real F = vl[n] * (r[n] + cc[n]);
          fy[n * NR * 32] = F;
          acc[n] = F * rdy;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(my_fyr + b * 2 * NR);
      }
      if (!ghost_row) {
        // ---- (B) low z-face (face k); completes plane k-1
        Real Fz[NM], vl[NM];
        vl[FU] = interp_adv<Real>(IA, S(FW, -2, 0), S(FW, -1, 0), wk, S(FW, 1, 0));      // w~ along x at (i-1/2, k-1/2)
        vl[FV] = interp_adv<Real>(IA, S(FW, 0, -2), S(FW, 0, -1), wk, S(FW, 0, 1));      // w~ along y at (j-1/2, k-1/2)
        if constexpr (SZ == 5) {
          if constexpr (!HYDRO) vl[FW] = interp_adv<Real>(IA, win[FW][ZL - 2], win[FW][ZL - 1], win[FW][ZL], win[FW][ZL + 1]);   // centre k-1
          Real d1[NM], d2[NM], d3[NM], d4[NM], cc[NM], r[NM];
#pragma unroll
          for (int n = 0; n < NM; ++n) window_diffs<Real>(win[n], vl[n], d1[n], d2[n], d3[n], d4[n], cc[n]);
          weno5z_anom_v<NM>(d1, d2, d3, d4, eps4, r);
#pragma unroll
          for (int n = 0; n < NM; ++n) Fz[n] = vl[n] * (r[n] + cc[n]);
        } else {
          // Centered(2) along z (B4): window = q(k-1), q(k), q(k+1)
          Fz[FU] = vl[FU] * (Real(0.5) * (win[FU][0] + win[FU][1]));
          Fz[FV] = vl[FV] * (Real(0.5) * (win[FV][0] + win[FV][1]));
          if constexpr (!HYDRO) { const Real wz = Real(0.5) * (win[FW][0] + win[FW][1]); Fz[FW] = wz * wz; }
        }
        if (it > 0 && can_store) {
          a.G[FU][o - sz] = wall_u ? Real(0) : part[FU] - Fz[FU] * rdzc_km;
          a.G[FV][o - sz] = wall_v ? Real(0) : part[FV] - Fz[FV] * rdzc_km;
          if constexpr (!HYDRO)      // control volume k-1 has thickness dz_f[k-1]; the bottom wall face gets 0
            a.G[FW][o - sz] = (g.topo[2] == OCN_BOUNDED && k == 2) ? Real(0) : part[FW] - Fz[FW] * rdzf_km;
        }
        if (more) {
          acc[FU] += Fz[FU] * rdzc_k;
          acc[FV] += Fz[FV] * rdzc_k;
          if constexpr (!HYDRO) acc[FW] += Fz[FW] * rdzf_k;
        }
      }
      if (!more) break;
      double b_k = 0.0;
      if (!HYDRO && m.buoyancy) b_k = buoy(S(FC, 0, 0), NT > 1 ? S(FC + (NT > 1 ? 1 : 0), 0, 0) : Real(0), zk);
      if (!ghost_row) {
        // ---- (C) low x-face fluxes; high face from lane+1
        {
          const Real *hi[NM];
          Real vl[NM], d1[NM], d2[NM], d3[NM], d4[NM], cc[NM], r[NM];
          hi[FU] = &S(FU, 0, 0);                                                                    // u at the centre i-1 (m = i)
          vl[FU] = interp_adv<Real>(S_WENO5, S(FU, -2, 0), S(FU, -1, 0), ui, S(FU, 1, 0));
          hi[FV] = &S(FV, 0, 0);                                                                    // v along x at (i-1/2, j-1/2)
          vl[FV] = interp_adv<Real>(S_WENO5, S(FU, 0, -2), S(FU, 0, -1), ui, S(FU, 0, 1));          // u~ along y
          if constexpr (!HYDRO) {
            hi[FW] = &S(FW, 0, 0);                                                                  // w along x at (i-1/2, k-1/2)
            vl[FW] = interp_adv<Real>(S_WENO5, win[FU][ZL - 2], win[FU][ZL - 1], ui, win[FU][ZL + 1]);   // u~ along z
          }
          upwind_diffs<Real, NM>(hi, 1, vl, d1, d2, d3, d4, cc);
          weno5z_anom_v<NM>(d1, d2, d3, d4, eps4, r);
#pragma unroll
          for (int n = 0; n < NM; ++n) {
            const Real F = vl[n] * (r[n] + cc[n]);
            acc[n] -= (shfl_down1(F) - F) * rdx;
          }
        }
        // ---- Coriolis, viscosity, buoyancy / hydrostatic pressure gradient
        {
          Real lap = ((S(FU, 1, 0) - ui) - (ui - S(FU, -1, 0))) * rdx2 + ((S(FU, 0, 1) - ui) - (ui - S(FU, 0, -1))) * rdy2;
          lap += ((win[FU][ZL + 1] - ui) * rdzf_kp - (ui - win[FU][ZL - 1]) * rdzf_k) * rdzc_k;
          Real G = acc[FU] + nu * lap;
          if (m.coriolis) G += fu * (Real(0.25) * ((S(FV, -1, 0) + vj) + (S(FV, -1, 1) + S(FV, 0, 1))));
          if (HYDRO && a.phy != nullptr) G -= (__ldg(a.phy + o) - __ldg(a.phy + o - 1)) * rdx;
          acc[FU] = G;
        }
        {
          Real lap = ((S(FV, 1, 0) - vj) - (vj - S(FV, -1, 0))) * rdx2 + ((S(FV, 0, 1) - vj) - (vj - S(FV, 0, -1))) * rdy2;
          lap += ((win[FV][ZL + 1] - vj) * rdzf_kp - (vj - win[FV][ZL - 1]) * rdzf_k) * rdzc_k;
          Real G = acc[FV] + nu * lap;
          if (m.coriolis) G -= fv * (Real(0.25) * ((S(FU, 0, -1) + S(FU, 1, -1)) + (ui + S(FU, 1, 0))));
          if (HYDRO && a.phy != nullptr) G -= (__ldg(a.phy + o) - __ldg(a.phy + o - g.sy)) * rdy;
          acc[FV] = G;
        }
        if constexpr (!HYDRO) {
          const Real w0 = win[FW][ZL];
          Real lap = ((S(FW, 1, 0) - w0) - (w0 - S(FW, -1, 0))) * rdx2 + ((S(FW, 0, 1) - w0) - (w0 - S(FW, 0, -1))) * rdy2;
          lap += ((win[FW][ZL + 1] - w0) * rdzc_k - (w0 - win[FW][ZL - 1]) * rdzc_km) * rdzf_k;
          acc[FW] += nu * lap + Real(0.5 * (b_km + b_k));
        }
        // ---- high y-face fluxes from row+1
        mbar_wait(my_fyr + b * 2 * NR + 1, ph);
#pragma unroll
        for (int n = 0; n < NM; ++n) acc[n] -= fy[n * NR * 32 + 32] * rdy;
      }
      b_km = b_k;
#pragma unroll
      for (int n = 0; n < NM; ++n) {
        part[n] = acc[n];
#pragma unroll
        for (int t = 0; t < WD - 1; ++t) win[n][t] = win[n][t + 1];
        win[n][WD - 1] = pf[n];
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[b]);
    }
  }
#undef S
#undef ZMETRICS
}

// ---- host side --------------------------------------------------------------------------------------------
PFN_cuTensorMapEncodeTiled_v12000 get_encode() {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(p);
  }
  return fn;
}

template <class Real, int NT, int SZ, bool HYDRO, int TY>
int launch_fused_t(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G, cudaStream_t s) {
  using SL = SmemLayout<Real, NT, TY>;
  auto enc = get_encode();
  if (!enc) return ocn_fail(OCN_ERR_CUDA, "tend_fused: cuTensorMapEncodeTiled entry point not available");
  FusedArgs<Real> a;
  memset(&a, 0, sizeof(a));
  a.g = g->dev;
  a.m = m;
  const void *in[MAXF] = {st.u, st.v, st.w, st.c[0], st.c[1], st.c[2]};
  void *out[MAXF] = {G.u, G.v, G.w, G.c[0], G.c[1], G.c[2]};
  const ocn_layout &L = g->lay;
  for (int f = 0; f < 3 + NT; ++f) {
    a.q[f] = (const Real *)in[f];
    a.G[f] = (Real *)out[f];
    cuuint64_t dims[3] = {(cuuint64_t)L.stride_y, (cuuint64_t)L.ny_pad, (cuuint64_t)L.nz_pad};
    cuuint64_t strides[2] = {(cuuint64_t)L.stride_y * sizeof(Real), (cuuint64_t)L.stride_z * sizeof(Real)};
    cuuint32_t box[3] = {(cuuint32_t)SL::TW, (cuuint32_t)SL::TH, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(&a.tmap[f], sizeof(Real) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3,
                     const_cast<void *>(in[f]), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return ocn_fail(OCN_ERR_CUDA, "tend_fused: cuTensorMapEncodeTiled failed (%d) for field %d", (int)r, f);
  }
  a.phy = (const Real *)phy;
  const int xoff = (int)(L.offset0 - (long long)L.hz * L.stride_z - (long long)L.hy * L.stride_y);   // array x of logical i = 1
  a.xa_off = xoff - 1;
  a.ya_off = L.hy - 1;
  a.za_off = L.hz - 1;
  const int nbx = (g->Nx + 30) / 31, nby = (g->Ny + TY - 1) / TY;
  // z-chunks: enough blocks for >= 2 waves of 148 SMs, but chunks of at least 8 planes (each chunk re-primes one plane)
  int nch = (2 * 148 + nbx * nby - 1) / (nbx * nby);
  nch = std::max(1, std::min(nch, (g->Nz + 7) / 8));
  a.kchunk = (g->Nz + nch - 1) / nch;
  nch = (g->Nz + a.kchunk - 1) / a.kchunk;
  auto kern = tend_fused_kernel<Real, NT, SZ, HYDRO, TY>;
  static bool attr_done = false;
  if (!attr_done) {
    OCN_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SL::BYTES));
    attr_done = true;
  }
  dim3 block(32, 2 * TY + 3, 1), grid(nbx, nby, nch);
  kern<<<grid, block, SL::BYTES, s>>>(a);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "tend_fused_kernel launch");
}

constexpr int TYD = 8;   // rows per tile

}  // namespace

bool fused_applicable(const ocn_grid *g, const ModelDev &m, std::string *why) {
  auto no = [&](const char *w) { if (why) *why = w; return false; };
  if (g->topo[0] == OCN_FLAT || g->topo[1] == OCN_FLAT || g->topo[2] == OCN_FLAT) return no("needs a 3-D grid");
  if (g->H < 3) return no("needs halo >= 3");
  if (m.adv[0] != OCN_ADV_WENO5 || m.adv[1] != OCN_ADV_WENO5) return no("needs WENO5 in x and y");
  if (!m.momentum) return no("needs prognostic momentum");
  const bool les = !m.hydrostatic && m.adv[2] == OCN_ADV_WENO5 && g->uniform_z;
  const bool hyd = m.hydrostatic && m.adv[2] == OCN_ADV_CENTERED2;
  if (!les && !hyd) return no("needs (nonhydrostatic, WENO5 in z, uniform dz) or (hydrostatic, Centered2 in z)");
  if (les && m.buoyancy && !((m.idx_T == 0 || m.idx_T < 0) && (m.idx_S == 1 || m.idx_S < 0))) return no("needs T, S as tracers 0, 1");
  if (g->dtype == OCN_F64 && m.n_tracers == 2) return true;
  if (g->dtype == OCN_F32 && les && (m.n_tracers == 2 || m.n_tracers == 3)) return true;
  return no("tracer count / precision combination not instantiated");
}

int launch_tendencies_fused(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G,
                            cudaStream_t s) {
  std::string why;
  if (!fused_applicable(g, m, &why)) return ocn_fail(OCN_ERR_UNSUPPORTED, "fused kernels not applicable: %s", why.c_str());
  const bool hyd = m.hydrostatic != 0;
  if (g->dtype == OCN_F64) {
    if (hyd) return launch_fused_t<double, 2, 2, true, TYD>(g, m, st, phy, G, s);
    static int ty = -1;
    if (ty < 0) { const char *e = getenv("OCN_FUSED_TY"); ty = e ? atoi(e) : TYD; }
    if (ty == 6) return launch_fused_t<double, 2, 5, false, 6>(g, m, st, phy, G, s);
    if (ty == 7) return launch_fused_t<double, 2, 5, false, 7>(g, m, st, phy, G, s);
    if (ty == 5) return launch_fused_t<double, 2, 5, false, 5>(g, m, st, phy, G, s);
    return launch_fused_t<double, 2, 5, false, TYD>(g, m, st, phy, G, s);
  }
  if (m.n_tracers == 3) return launch_fused_t<float, 3, 5, false, TYD>(g, m, st, phy, G, s);
  return launch_fused_t<float, 2, 5, false, TYD>(g, m, st, phy, G, s);
}
