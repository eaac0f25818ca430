// tend_hiorder.cu — WENO7-Z / WENO9-Z advection ("WENO reconstructions of orders up to 11", 79,
// 409, 429: every showcase run uses order 9), halo >= 4 / 5.  Axes that do not use WENO run Centered(2) (hydrostatic vertical) or
// nothing (Flat).  Same discrete operators as tend_percell.cu with
//   [.]   = WENO(2R-1)-Z, R = 4, 5, in undivided-difference form (weno_hi.cuh, generated), upwind by the sign of the
//           advecting velocity (mirror image for flow in the negative direction, reading R3),
//   a~    = Centered(2R-2) interpolation of the advecting velocity across the flux direction ((B21), reading R4),
// tracers in the cancellation-free form (H1): sum_faces u_f ([c]_f - c_ijk) + c_ijk div(u), div(u) in double-double.
// Three kernels:
//   tend_hiorder_kernel        one thread per interior cell, operands from global memory, any topology (Flat axes, 1-D, 2-D);
//   tend_hiorder_march_kernel  3-D grids: a block owns 31 x 7 columns and marches along z, every face flux once, operands from
//                              global memory (the fallback of the next one: more than 3 tracers, tiles that do not fit);
//   tend_hiorder_tma_kernel    the default on 3-D grids: the same march with the x-y operands of every plane staged in shared memory
//                              by TMA, no ghost warp, and optionally the (A4) substage fused in (ocn_tendencies_rk3).
#include <cuda.h>
#include <cudaTypedefs.h>

#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <string>

#include "ocn_internal.h"
#include "weno_hi.cuh"

namespace {

using namespace ocn;

template <class Real>
struct HArgs {
  GridDev g;
  ModelDev m;
  const Real *u, *v, *w, *phy;
  const Real *c[OCN_MAX_TRACERS];
  Real *Gu, *Gv, *Gw;
  Real *Gc[OCN_MAX_TRACERS];
  // fused substage (A4) of the per-cell and the global-load marching kernels (RK != 0): q_new = q + (rk_a G - rk_b G_prev)
  const Real *Pu, *Pv, *Pw;
  const Real *Pc[OCN_MAX_TRACERS];
  Real *Qu, *Qv, *Qw;
  Real *Qc[OCN_MAX_TRACERS];
  Real rk_a, rk_b;
};

// store G and, with the substage fused in, the new state (same arithmetic as rk3.cu: rk3_update); wall: G is 0 and q stays
template <int RK, class Real>
__device__ __forceinline__ void hi_store_GQ(Real *Gf, const Real *Pf, Real *Qf, long long o, Real G, Real q, bool wall, Real rk_a, Real rk_b) {
  Gf[o] = G;
  if constexpr (RK != 0) {
    const Real qn = RK == 2 ? rk3_update(q, G, Pf[o], rk_a, rk_b) : rk3_update(q, G, rk_a);
    Qf[o] = wall ? q : qn;
  }
}

template <class Real, int R>
__device__ __forceinline__ Real weno_hi_anom(const Real *v, Real eps) {
  if constexpr (R == 4) return weno7z_anom<Real>(v, eps);
  else return weno9z_anom<Real>(v, eps);
}

// advecting velocity at the point between q[-s] and q[0]: Centered(2R-2) where the flux direction uses WENO(2R-1),
// Centered(2) otherwise (reading R4)
template <class Real, int R>
__device__ __forceinline__ Real centered_hi(const Real *q, long long s) {
  if constexpr (R == 4) return centered6<Real>(q, s);
  else return centered8<Real>(q, s);
}
template <class Real, int R>
__device__ __forceinline__ Real interp_hi(bool weno, const Real *q, long long s) {
  if (!weno) return Real(0.5) * (q[-s] + q[0]);
  if constexpr (R == 4) return centered6<Real>(q, s);
  else return centered8<Real>(q, s);
}

// F_hi - F_lo of the advected sequence q (element stride s) through the two faces of the control volume centred on
// q[0]: the low face lies between q[-s] and q[0], the high face between q[0] and q[s]; F = a~ ([q] - base).
//   weno: [q] from q[m-R .. m+R-2] (a~ > 0) or its mirror image q[m+R-1 .. m-R+1];  else Centered(2) (B4).
template <class Real, int R>
__device__ __forceinline__ Real flux_diff(bool weno, const Real *q, long long s, Real alo, Real ahi, Real base, Real eps) {
  if (!weno) {
    const Real q0 = q[0] - base;
    const Real Flo = alo * (Real(0.5) * ((q[-s] - base) + q0));
    const Real Fhi = ahi * (Real(0.5) * (q0 + (q[s] - base)));
    return Fhi - Flo;
  }
  Real w[2 * R + 1];                                    // q[-R .. R]
#pragma unroll
  for (int t = 0; t <= 2 * R; ++t) w[t] = q[(t - R) * s];
  Real F[2];
#pragma unroll
  for (int f = 0; f < 2; ++f) {                         // f = 0: low face (window w[0 .. 2R-1]), f = 1: high face (w[1 .. 2R])
    const Real a = f ? ahi : alo;
    const bool pos = a > Real(0);
    Real v[2 * R - 1];
#pragma unroll
    for (int t = 0; t < 2 * R - 1; ++t) v[t] = pos ? w[f + t] : w[f + 2 * R - 1 - t];
    F[f] = a * (weno_hi_anom<Real, R>(v, eps) + (v[R - 1] - base));
  }
  return F[1] - F[0];
}

// 7-point Laplacian of a field centred in z (c, u, v): flux-divergence form (B2), eq. 8
template <class Real>
__device__ __forceinline__ Real lap_c(const GridDev &g, const Real *q, int k, bool hx, bool hy, bool hz) {
  const Real q0 = q[0];
  Real s = Real(0);
  if (hx) s += ((q[1] - q0) - (q0 - q[-1])) * Real(g.rdx * g.rdx);
  if (hy) s += ((q[g.sy] - q0) - (q0 - q[-g.sy])) * Real(g.rdy * g.rdy);
  if (hz) {
    const int z = g.zi(k);
    s += ((q[g.sz] - q0) * Real(g.rdzf[z + 1]) - (q0 - q[-g.sz]) * Real(g.rdzf[z])) * Real(g.rdzc[z]);
  }
  return s;
}

template <class Real, int R, int RK>
__global__ void __launch_bounds__(128) tend_hiorder_kernel(const HArgs<Real> a) {
  const GridDev &g = a.g;
  const ModelDev &m = a.m;
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1;
  const int j = blockIdx.y * blockDim.y + threadIdx.y + 1;
  const int k = blockIdx.z + 1;
  if (i > g.Nx || j > g.Ny) return;
  const long long o = g.idx(i, j, k), SX = 1, SY = g.sy, SZ = g.sz;
  const bool hx = g.topo[0] != OCN_FLAT, hy = g.topo[1] != OCN_FLAT, hz = g.topo[2] != OCN_FLAT;
  constexpr int HI = 2 * R - 1;
  const bool wx = m.adv[0] == HI, wy = m.adv[1] == HI, wz = m.adv[2] == HI;
  const bool ax = hx && a.u != nullptr && m.adv[0] != OCN_ADV_NONE;
  const bool ay = hy && a.v != nullptr && m.adv[1] != OCN_ADV_NONE;
  const bool az = hz && a.w != nullptr && m.adv[2] != OCN_ADV_NONE;
  const Real eps = Real(m.weno_eps);
  const int zk = g.zi(k);
  const Real rdx = Real(g.rdx), rdy = Real(g.rdy);
  const Real rdzc = hz ? Real(g.rdzc[zk]) : Real(0);
  const Real *U = a.u + o, *V = a.v + o, *W = a.w + o;   // only dereferenced when the field exists

  // ------------------------------------------------------------------ tracers at ccc: (B2),(B3) PAPER.md:990-1003
  if (m.n_tracers > 0) {
    const Real ul = ax ? U[0] : Real(0), uh = ax ? U[SX] : Real(0);
    const Real vl = ay ? V[0] : Real(0), vh = ay ? V[SY] : Real(0);
    const Real wl = az ? W[0] : Real(0), wh = az ? W[SZ] : Real(0);
    double D = 0.0, Dlo = 0.0;
    if (ax) dd_add_diff_scaled((double)uh, (double)ul, g.rdx, g.rdx_lo, D, Dlo);
    if (ay) dd_add_diff_scaled((double)vh, (double)vl, g.rdy, g.rdy_lo, D, Dlo);
    if (az) dd_add_diff_scaled((double)wh, (double)wl, g.rdzc[zk], g.rdzc_lo[zk], D, Dlo);
    const double Dsum = D + Dlo;
    for (int n = 0; n < m.n_tracers; ++n) {
      const Real *C = a.c[n] + o;
      const Real c0 = C[0];
      Real adv = Real(0);
      if (ax) adv += flux_diff<Real, R>(wx, C, SX, ul, uh, c0, eps) * rdx;      // face velocity used directly (B3)
      if (ay) adv += flux_diff<Real, R>(wy, C, SY, vl, vh, c0, eps) * rdy;
      if (az) adv += flux_diff<Real, R>(wz, C, SZ, wl, wh, c0, eps) * rdzc;
      Real G = -adv - Real((double)c0 * Dsum);
      if (m.kappa[n] != 0.0) G += Real(m.kappa[n]) * lap_c<Real>(g, C, k, hx, hy, hz && !m.vimplicit);
      hi_store_GQ<RK, Real>(a.Gc[n], a.Pc[n], a.Qc[n], o, G, c0, false, a.rk_a, a.rk_b);
    }
  }
  if (!m.momentum) return;

  // ------------------------------------------------------------------ u at fcc: eq. 6/17, flux form (7)/(18), (B21)
  if (a.Gu != nullptr) {
    Real G = Real(0);
    if (i >= first_face(g.topo[0])) {
      Real div = Real(0);
      if (ax) {   // x-faces of the u control volume are the cell centres i-1 (m = i) and i (m = i+1)
        const Real al = interp_hi<Real, R>(wx, U, SX), ah = interp_hi<Real, R>(wx, U + SX, SX);
        div += flux_diff<Real, R>(wx, U, SX, al, ah, Real(0), eps) * rdx;
      }
      if (ay) {   // v interpolated along x to x-face i, at the y-faces j and j+1
        const Real al = interp_hi<Real, R>(wy, V, SX), ah = interp_hi<Real, R>(wy, V + SY, SX);
        div += flux_diff<Real, R>(wy, U, SY, al, ah, Real(0), eps) * rdy;
      }
      if (az) {
        const Real al = interp_hi<Real, R>(wz, W, SX), ah = interp_hi<Real, R>(wz, W + SZ, SX);
        div += flux_diff<Real, R>(wz, U, SZ, al, ah, Real(0), eps) * rdzc;
      }
      G = -div;
      if (m.coriolis && a.v != nullptr) {                 // reading R8: 4-point average, f at y_c[j]
        const double f = m.f0 + m.beta * ((j - 0.5) * g.dy - m.y0);
        G += Real(f) * (Real(0.25) * ((V[-SX] + V[0]) + (V[SY - SX] + V[SY])));
      }
      if (m.nu != 0.0) G += Real(m.nu) * lap_c<Real>(g, U, k, hx, hy, hz && !m.vimplicit);
      if (m.hydrostatic && a.phy != nullptr) G -= (a.phy[o] - a.phy[o - 1]) * rdx;
    }
    hi_store_GQ<RK, Real>(a.Gu, a.Pu, a.Qu, o, G, U[0], i < first_face(g.topo[0]), a.rk_a, a.rk_b);
  }

  // ------------------------------------------------------------------ v at cfc (mirror of u with x <-> y)
  if (a.Gv != nullptr) {
    Real G = Real(0);
    if (j >= first_face(g.topo[1])) {
      Real div = Real(0);
      if (ax) {   // u interpolated along y to y-face j, at the x-faces i and i+1
        const Real al = interp_hi<Real, R>(wx, U, SY), ah = interp_hi<Real, R>(wx, U + SX, SY);
        div += flux_diff<Real, R>(wx, V, SX, al, ah, Real(0), eps) * rdx;
      }
      if (ay) {
        const Real al = interp_hi<Real, R>(wy, V, SY), ah = interp_hi<Real, R>(wy, V + SY, SY);
        div += flux_diff<Real, R>(wy, V, SY, al, ah, Real(0), eps) * rdy;
      }
      if (az) {
        const Real al = interp_hi<Real, R>(wz, W, SY), ah = interp_hi<Real, R>(wz, W + SZ, SY);
        div += flux_diff<Real, R>(wz, V, SZ, al, ah, Real(0), eps) * rdzc;
      }
      G = -div;
      if (m.coriolis && a.u != nullptr) {                 // f at y_f[j]
        const double f = m.f0 + m.beta * ((j - 1.0) * g.dy - m.y0);
        G -= Real(f) * (Real(0.25) * ((U[-SY] + U[SX - SY]) + (U[0] + U[SX])));
      }
      if (m.nu != 0.0) G += Real(m.nu) * lap_c<Real>(g, V, k, hx, hy, hz && !m.vimplicit);
      if (m.hydrostatic && a.phy != nullptr) G -= (a.phy[o] - a.phy[o - g.sy]) * rdy;
    }
    hi_store_GQ<RK, Real>(a.Gv, a.Pv, a.Qv, o, G, V[0], j < first_face(g.topo[1]), a.rk_a, a.rk_b);
  }

  // ------------------------------------------------------------------ w at ccf (nonhydrostatic; uniform dz: launcher)
  if (a.Gw != nullptr && !m.hydrostatic && hz) {
    Real G = Real(0);
    if (k >= first_face(g.topo[2])) {
      const Real rdzf = Real(g.rdzf[zk]);
      Real div = Real(0);
      if (ax) {   // u interpolated along z to z-face k, at the x-faces i and i+1
        const Real al = interp_hi<Real, R>(wx, U, SZ), ah = interp_hi<Real, R>(wx, U + SX, SZ);
        div += flux_diff<Real, R>(wx, W, SX, al, ah, Real(0), eps) * rdx;
      }
      if (ay) {
        const Real al = interp_hi<Real, R>(wy, V, SZ), ah = interp_hi<Real, R>(wy, V + SY, SZ);
        div += flux_diff<Real, R>(wy, W, SY, al, ah, Real(0), eps) * rdy;
      }
      if (az) {   // z-faces of the w control volume are the cell centres k-1 and k
        const Real al = interp_hi<Real, R>(wz, W, SZ), ah = interp_hi<Real, R>(wz, W + SZ, SZ);
        div += flux_diff<Real, R>(wz, W, SZ, al, ah, Real(0), eps) * rdzf;
      }
      G = -div;
      if (m.buoyancy) {   // b = g [alpha (T - Tref) - beta (S - Sref)] at k-1 and k (reading R9, R10)
        double bsum = 0.0;
        for (int dk = -1; dk <= 0; ++dk) {
          double T = 0.0, S = 0.0;
          if (m.idx_T >= 0) T = (double)a.c[m.idx_T][o + dk * g.sz] - g.Tref[zk + dk];
          if (m.idx_S >= 0) S = (double)a.c[m.idx_S][o + dk * g.sz] - g.Sref[zk + dk];
          bsum += m.g * (m.alpha_T * T - m.beta_S * S);
        }
        G += Real(0.5 * bsum);
      }
      if (m.nu != 0.0) {
        const Real q0 = W[0];
        Real s = Real(0);
        if (hx) s += ((W[SX] - q0) - (q0 - W[-SX])) * Real(g.rdx * g.rdx);
        if (hy) s += ((W[SY] - q0) - (q0 - W[-SY])) * Real(g.rdy * g.rdy);
        if (!m.vimplicit) s += ((W[SZ] - q0) * Real(g.rdzc[zk]) - (q0 - W[-SZ]) * Real(g.rdzc[zk - 1])) * rdzf;
        G += Real(m.nu) * s;
      }
    }
    hi_store_GQ<RK, Real>(a.Gw, a.Pw, a.Qw, o, G, W[0], k < first_face(g.topo[2]), a.rk_a, a.rk_b);
  }
}

// =====================================================================================================================
// Marching variant for 3-D grids: EVERY FACE FLUX IS COMPUTED ONCE.  A block owns a 31 x TY tile of columns and marches
// along z.  Each thread computes, for every prognostic field, the flux through the LOW x-face and the LOW y-face of its
// control volume and through the HIGH z-face; the high x-face comes from lane+1 (shuffle; lane 31 only serves lane 30),
// the high y-face from row+1 (shared memory; row TY is a ghost row that computes y-fluxes only) and the low z-face is
// the previous plane's high face (a per-thread shared-memory slot).  Tracer fluxes are carried as anomalies and re-based
// to the receiving cell's own value (H1).  Operands come from global memory through L1/L2 (the upwind stencil is
// selected by ADDRESS, 2R-1 loads per reconstruction).  One __syncthreads per plane (double-buffered y exchange).
// =====================================================================================================================

// value of the reconstruction at the face between qm[-s] and qm[0], MINUS the returned upwind cell value `cup`
template <class Real, int R>
__device__ __forceinline__ Real face_anom(bool weno, const Real *qm, long long s, Real a, Real eps, Real &cup) {
  if (!weno) {                                           // Centered(2) (B4)
    cup = qm[-s];
    return Real(0.5) * (qm[0] - cup);
  }
  // All 2R cells m-R .. m+R-1 are loaded with STATIC offsets — independent of the velocity, so every load of a (field, direction)
  // unit is in flight before the advecting velocity has been interpolated — and the upwind stencil (q[m-R .. m+R-2] or the mirror
  // image q[m+R-1 .. m-R+1]) is picked by value selects.  (Address selection put the velocity's load latency in front of the
  // stencil's and cost ~60 integer instructions per reconstruction in 64-bit address arithmetic.)
  const bool pos = a > Real(0);
  Real q[2 * R];
#pragma unroll
  for (int t = 0; t < 2 * R; ++t) q[t] = qm[(t - R) * s];
  Real v[2 * R - 1];
#pragma unroll
  for (int t = 0; t < 2 * R - 1; ++t) v[t] = pos ? q[t] : q[2 * R - 1 - t];
  cup = v[R - 1];
  return weno_hi_anom<Real, R>(v, eps);
}

// the same from the 2R cell values q[0 .. 2R-1] = cells m-R .. m+R-1 of the face between q[R-1] and q[R]
template <class Real, int R>
__device__ __forceinline__ Real face_anom_vals(const Real (&q)[2 * R], Real a, Real eps, Real &cup) {
  const bool pos = a > Real(0);
  Real v[2 * R - 1];
#pragma unroll
  for (int t = 0; t < 2 * R - 1; ++t) v[t] = pos ? q[t] : q[2 * R - 1 - t];
  cup = v[R - 1];
  return weno_hi_anom<Real, R>(v, eps);
}

__device__ __forceinline__ void hi_cp_async(double *dst, const double *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void hi_cp_async(float *dst, const float *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}

template <class Real>
struct MArgs {
  HArgs<Real> h;
  int kchunk, nf;
};

template <class Real, int R, int TY, int RK>
__global__ void __launch_bounds__(32 * (TY + 1), 2) tend_hiorder_march_kernel(const MArgs<Real> ma) {
  const HArgs<Real> &a = ma.h;
  const GridDev &g = a.g;
  const ModelDev &m = a.m;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int nf = ma.nf;                                  // u, v, (w), tracers: fields that carry a tendency
  Real *fyb = reinterpret_cast<Real *>(smem_raw);        // [2][nf][TY+1][32]  low y-face fluxes, based for the row below
  Real *fzb = fyb + 2 * nf * (TY + 1) * 32;              // [nf][TY][32]       carried high z-face fluxes, based for the cell above
  Real *pb = fzb + nf * TY * 32;                         // [nf][TY][32]       everything but the high y-face
  const int lane = threadIdx.x, row = threadIdx.y;
  const bool ghost = row == TY;
  const int i = blockIdx.x * 31 + 1 + lane, j = blockIdx.y * TY + 1 + row;
  const int ic = min(i, g.Nx + 1), jc = min(j, g.Ny + 1);   // clamped columns compute finite duplicates that nobody stores
  const int kc0 = 1 + blockIdx.z * ma.kchunk, kc1 = min(kc0 + ma.kchunk, g.Nz + 1);
  const bool store = lane < 31 && !ghost && i <= g.Nx && j <= g.Ny;
  auto Sax = [&](int ax_) -> long long { return ax_ == 0 ? 1 : (ax_ == 1 ? g.sy : g.sz); };   // element stride of an axis
  constexpr int HI = 2 * R - 1;
  const Real eps = Real(m.weno_eps);
  const Real rdx = Real(g.rdx), rdy = Real(g.rdy);
  const bool mom = m.momentum != 0, hasGw = mom && !m.hydrostatic;
  const int fc0 = mom ? (hasGw ? 3 : 2) : 0;            // index of the first tracer among the tendency fields
  const int slot = row * 32 + lane;
  auto velp = [&](int c_) -> const Real * { return c_ == 0 ? a.u : (c_ == 1 ? a.v : a.w); };
  auto FY = [&](int buf, int f, int r) -> Real & { return fyb[((buf * nf + f) * (TY + 1) + r) * 32 + lane]; };
  auto FZ = [&](int f) -> Real & { return fzb[f * TY * 32 + slot]; };
  auto PB = [&](int f) -> Real & { return pb[f * TY * 32 + slot]; };

  long long o = g.idx(ic, jc, kc0);
  for (int k = kc0, n = 0; k < kc1; ++k, ++n, o += g.sz) {
    const int buf = n & 1;
    const int zk = g.zi(k);
    const Real rdzc = Real(g.rdzc[zk]), rdzf = Real(g.rdzf[zk]);
    const bool first = n == 0;
    // velocity divergence of the cell in double-double (tracers, H1)
    double Dsum = 0.0;
    if (m.n_tracers > 0 && !ghost) {
      double D = 0.0, Dlo = 0.0;
      if (m.adv[0] != OCN_ADV_NONE) dd_add_diff_scaled((double)a.u[o + 1], (double)a.u[o], g.rdx, g.rdx_lo, D, Dlo);
      if (m.adv[1] != OCN_ADV_NONE) dd_add_diff_scaled((double)a.v[o + g.sy], (double)a.v[o], g.rdy, g.rdy_lo, D, Dlo);
      if (m.adv[2] != OCN_ADV_NONE) dd_add_diff_scaled((double)a.w[o + g.sz], (double)a.w[o], g.rdzc[zk], g.rdzc_lo[zk], D, Dlo);
      Dsum = D + Dlo;
    }
    // ONE instance of the reconstruction code serves every (field, direction) pair: runtime loops, not unrolled
    // (15-18 inlined copies of WENO9 overflow the instruction cache: ncu "no_instruction" was the top stall)
#pragma unroll 1
    for (int f = 0; f < nf; ++f) {
      const bool tr = f >= fc0;
      const Real *Q = (tr ? a.c[f - fc0] : velp(f)) + o;
      const long long Sf = tr ? 0 : Sax(f);               // the axis along which a velocity component is face-located
      const Real c0 = tr ? Q[0] : Real(0);
      Real part = Real(0);
#pragma unroll
      for (int d = 0; d < 3; ++d) {        // unrolled: three instances of the reconstruction code (x, y, z), fields looped
        if (m.adv[d] == OCN_ADV_NONE) {
          if (d == 1) FY(buf, f, row) = Real(0);
          continue;
        }
        if (ghost && d != 1) continue;
        const bool weno = m.adv[d] == HI;
        const long long Sd = Sax(d);
        const Real *vd = velp(d) + o;
        Real Flo_prime = Real(0);
        // x, y: the LOW face of the control volume; z: the HIGH face (plus, on the first plane of a chunk, the low one)
#pragma unroll 1
        for (int pass = (d == 2 && first) ? 0 : 1; pass < 2; ++pass) {
          const long long fo = (d == 2 && pass == 1) ? Sd : 0;              // offset of the element on the high side of the face
          const Real *qm = Q + fo;
          // advecting velocity at the face: tracers use the face velocity directly (B3); momentum interpolates
          // component d across the flux direction, along the advected component's own axis ((B21), reading R4)
          const Real av = tr ? vd[fo] : interp_hi<Real, R>(weno, vd + fo, Sf);
          Real cup;
          const Real val = face_anom<Real, R>(weno, qm, Sd, av, eps, cup);
          const bool hiface = fo != 0;
          const Real own = tr ? (hiface ? qm[-Sd] : qm[0]) : Real(0);       // the cell this thread owns
          const Real nbr = tr ? (hiface ? qm[0] : qm[-Sd]) : Real(0);       // the cell on the other side of the face
          const Real Fown = av * (val + (cup - own)), Fnbr = av * (val + (cup - nbr));
          if (d == 0) {
            part -= (__shfl_down_sync(0xffffffffu, Fnbr, 1) - Fown) * rdx;
          } else if (d == 1) {
            FY(buf, f, row) = Fnbr;
            part += Fown * rdy;
          } else if (pass == 0) {
            Flo_prime = Fown;
          } else {
            const Real Flo = first ? Flo_prime : FZ(f);
            FZ(f) = Fnbr;
            part -= (Fown - Flo) * ((!tr && f == 2) ? rdzf : rdzc);
          }
        }
      }
      if (ghost) continue;
      // ---- pointwise terms
      if (tr) {
        part -= Real((double)c0 * Dsum);
        if (m.kappa[f - fc0] != 0.0) part += Real(m.kappa[f - fc0]) * lap_c<Real>(g, Q, k, true, true, !m.vimplicit);
      } else if (f == 0) {
        if (m.coriolis) {                                  // reading R8: f at y_c[j]
          const Real *V = a.v + o;
          const double fc = m.f0 + m.beta * ((j - 0.5) * g.dy - m.y0);
          part += Real(fc) * (Real(0.25) * ((V[-1] + V[0]) + (V[g.sy - 1] + V[g.sy])));
        }
        if (m.nu != 0.0) part += Real(m.nu) * lap_c<Real>(g, Q, k, true, true, !m.vimplicit);
        if (m.hydrostatic && a.phy != nullptr) part -= (a.phy[o] - a.phy[o - 1]) * rdx;
      } else if (f == 1) {
        if (m.coriolis) {                                  // f at y_f[j]
          const Real *U = a.u + o;
          const double fc = m.f0 + m.beta * ((j - 1.0) * g.dy - m.y0);
          part -= Real(fc) * (Real(0.25) * ((U[-g.sy] + U[1 - g.sy]) + (U[0] + U[1])));
        }
        if (m.nu != 0.0) part += Real(m.nu) * lap_c<Real>(g, Q, k, true, true, !m.vimplicit);
        if (m.hydrostatic && a.phy != nullptr) part -= (a.phy[o] - a.phy[o - g.sy]) * rdy;
      } else {
        if (m.buoyancy) {                                  // readings R9, R10
          double bsum = 0.0;
          for (int dk = -1; dk <= 0; ++dk) {
            double T = 0.0, Sa = 0.0;
            if (m.idx_T >= 0) T = (double)a.c[m.idx_T][o + dk * g.sz] - g.Tref[zk + dk];
            if (m.idx_S >= 0) Sa = (double)a.c[m.idx_S][o + dk * g.sz] - g.Sref[zk + dk];
            bsum += m.g * (m.alpha_T * T - m.beta_S * Sa);
          }
          part += Real(0.5 * bsum);
        }
        if (m.nu != 0.0) {
          const Real q0 = Q[0];
          Real s = ((Q[1] - q0) - (q0 - Q[-1])) * Real(g.rdx * g.rdx) + ((Q[g.sy] - q0) - (q0 - Q[-g.sy])) * Real(g.rdy * g.rdy);
          if (!m.vimplicit) s += ((Q[g.sz] - q0) * Real(g.rdzc[zk]) - (q0 - Q[-g.sz]) * Real(g.rdzc[zk - 1])) * rdzf;
          part += Real(m.nu) * s;
        }
      }
      PB(f) = part;
    }
    __syncthreads();
    if (store) {
      for (int f = 0; f < nf; ++f) {
        const Real Gf = PB(f) - FY(buf, f, row + 1) * rdy;
        if (f < fc0) {                                      // wall faces of wall-normal velocities: G = 0
          const bool wall = g.topo[f] == OCN_BOUNDED && (f == 0 ? i : (f == 1 ? j : k)) == 1;
          Real *Gm = f == 0 ? a.Gu : (f == 1 ? a.Gv : a.Gw);
          const Real *Pm = f == 0 ? a.Pu : (f == 1 ? a.Pv : a.Pw);
          Real *Qm = f == 0 ? a.Qu : (f == 1 ? a.Qv : a.Qw);
          hi_store_GQ<RK, Real>(Gm, Pm, Qm, o, wall ? Real(0) : Gf, RK != 0 ? velp(f)[o] : Real(0), wall, a.rk_a, a.rk_b);
        } else {
          hi_store_GQ<RK, Real>(a.Gc[f - fc0], a.Pc[f - fc0], a.Qc[f - fc0], o, Gf, RK != 0 ? a.c[f - fc0][o] : Real(0), false, a.rk_a, a.rk_b);
        }
      }
    }
  }
}

// =====================================================================================================================
// TMA-staged marching kernel (the default for 3-D grids with <= 3 tracers).  Same decomposition as tend_hiorder_march_kernel
// (31 x TY columns per block, z-march, every face flux once), but the x-y operands no longer come through L1/L2: thread 0
// streams, plane after plane, a (32 + 2R - 1) x (TY + 2R) box of EVERY input field (R-cell halo included) into a two-slot
// shared-memory ring by TMA (cp.async.bulk.tensor.3d + mbarrier complete_tx; SASS UTMALDG): slot n & 1 holds plane k, the other
// slot plane k+1 (the high z-face's advecting w, w(k+1) of div(u), the upper neighbour of the vertical Laplacians).  The x- and
// y-stencils, the advecting velocities interpolated along x or y, div(u), Coriolis and the horizontal Laplacians are shared-memory
// loads at compile-time offsets (no address arithmetic, ~30-cycle latency); only the z-stencils (2R loads per field, coalesced
// rows that the previous plane already pulled into L1/L2) and the two z-interpolated advecting velocities still come from global
// memory.  ncu of the global-load version at C2 / WENO9: long-scoreboard stalls 2.1 per issue, issue active 48 %, FP64 pipe 52 %.
// =====================================================================================================================
#ifndef OCN_HI_PAIR
#define OCN_HI_PAIR(R) ((R) == 4)
#endif
constexpr int TMA_MAXIN = 6;                              // u, v, w + up to 3 tracers staged per plane

template <class Real>
struct TArgs {
  CUtensorMap tmap[TMA_MAXIN];                          // one 3-D tiled map per input field: box (TW, TY + 2R, 1)
  HArgs<Real> h;
  int kchunk, nf, nin;
  int zwin;                                             // 1: the z-windows are prefetched into per-thread shared-memory slots (when they fit)
  int xa_off, ya_off, za_off;                           // array coordinates of logical (i,j,k) = (i + xa_off, j + ya_off, k + za_off)
  // fused substage (A4) (RK != 0): q_new = q + (rk_a G - rk_b G_prev) written to the OTHER state buffer of the ping-pong pair;
  // indexed like the staged input fields (u, v, w, tracers)
  const Real *Gp[TMA_MAXIN];
  Real *Qn[TMA_MAXIN];
  Real rk_a, rk_b;
};

template <class Real, int R, int TY>
struct StagedGeom {
  static constexpr int XA = 16 / (int)sizeof(Real);                         // elements per 16 bytes (TMA start alignment)
  static constexpr int TW = ((32 + 2 * R - 1 + XA - 1 + XA - 1) / XA) * XA; // lanes 0..31 + stencil reach + alignment slack
  static constexpr int TH = TY + 2 * R;                                     // rows 0..TY (ghost) + stencil reach
  static constexpr int FS = ((TW * TH * (int)sizeof(Real) + 127) / 128) * 128 / (int)sizeof(Real);
  static size_t bytes(int nin, int nf, bool zwin) {
    return (size_t)2 * nin * FS * sizeof(Real) + (size_t)nf * (2 * (TY + 1) + 2 * TY) * 32 * sizeof(Real) +
           (zwin ? (size_t)(2 * R - 2) * TY * 32 * sizeof(Real) : 0) + 2 * sizeof(unsigned long long);
  }
};

__device__ __forceinline__ unsigned hi_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// RK: 0 tendencies only, 1 fused substage without G_prev (zeta = 0), 2 with G_prev (same arithmetic as rk3.cu: rk3_update)
template <class Real, int R, int TY, int RK>
__global__ void __launch_bounds__(32 * TY, 2) tend_hiorder_tma_kernel(const __grid_constant__ TArgs<Real> ta) {
  constexpr bool PAIR = OCN_HI_PAIR(R);
  using SG = StagedGeom<Real, R, TY>;
  constexpr int TW = SG::TW, FS = SG::FS, XA = SG::XA;
  const HArgs<Real> &a = ta.h;
  const GridDev &g = a.g;
  const ModelDev &m = a.m;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int nf = ta.nf, nin = ta.nin;                    // fields that carry a tendency; staged input fields (u, v, w, tracers)
  Real *tile = reinterpret_cast<Real *>(smem_raw);       // [2][nin][FS]
  Real *fyb = tile + 2 * nin * FS;                       // [2][nf][TY+1][32]  low y-face fluxes, based for the row below
  Real *fzb = fyb + 2 * nf * (TY + 1) * 32;              // [nf][TY][32]       carried high z-face fluxes, based for the cell above
  Real *pb = fzb + nf * TY * 32;                         // [nf][TY][32]       everything but the high y-face
  Real *zwb = pb + nf * TY * 32;                         // [2R-2][TY][32]     this thread's z-window of the current field (cp.async), if zwin
  unsigned long long *full = reinterpret_cast<unsigned long long *>(zwb + (ta.zwin ? (2 * R - 2) * TY * 32 : 0));
  const int lane = threadIdx.x, row = threadIdx.y;
  // No ghost warp: the y-fluxes through the top edge of the tile (row TY, the high face of row TY-1) are computed by the warp whose
  // row index equals the field index, as a second trip through its y-pass (a warp that only did those fluxes idled two thirds
  // of every plane at the barrier and cost an eighth of the block's warp slots; ncu r2: barrier 1.2 of 4 warps per scheduler).
  const int i0 = blockIdx.x * 31 + 1, j0 = blockIdx.y * TY + 1;
  const int i = i0 + lane, j = j0 + row;
  const int ic = min(i, g.Nx + 1), jc = min(j, g.Ny + 1);   // clamped columns compute finite duplicates that nobody stores
  const int kc0 = 1 + blockIdx.z * ta.kchunk, kc1 = min(kc0 + ta.kchunk, g.Nz + 1);
  const bool store = lane < 31 && i <= g.Nx && j <= g.Ny;
  constexpr int HI = 2 * R - 1;
  const Real eps = Real(m.weno_eps);
  const Real rdx = Real(g.rdx), rdy = Real(g.rdy);
  const bool mom = m.momentum != 0, hasGw = mom && !m.hydrostatic;
  const int fc0 = mom ? (hasGw ? 3 : 2) : 0;            // index of the first tracer among the tendency fields
  const int slot_ = row * 32 + lane;
  const long long SZ = g.sz;
  const long long og = (long long)(min(j0 + TY, g.Ny + 1) - jc) * g.sy;   // element offset from this thread's (clamped) column to the top-edge row
  auto gin = [&](int fi) -> const Real * { return fi == 0 ? a.u : (fi == 1 ? a.v : (fi == 2 ? a.w : a.c[fi - 3])); };
  auto FY = [&](int buf, int f, int r) -> Real & { return fyb[((buf * nf + f) * (TY + 1) + r) * 32 + lane]; };
  auto FZ = [&](int f) -> Real & { return fzb[f * TY * 32 + slot_]; };
  auto PB = [&](int f) -> Real & { return pb[f * TY * 32 + slot_]; };

  // ---- the plane ring: thread 0 is the producer
  const int tx0 = ((i0 - R + ta.xa_off) / XA) * XA, ty0 = j0 - R + ta.ya_off;   // the box starts on a 16-byte boundary at or left of i0-R
  const int xs = (i0 - R + ta.xa_off) - tx0;
  const int pos0 = (row + R) * TW + lane + R + xs;      // this thread's cell inside a staged field
  const bool producer = lane == 0 && row == 0;
  const unsigned plane_bytes = (unsigned)(nin * TW * SG::TH * sizeof(Real));
  auto issue = [&](int plane, int sl) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(hi_smem_u32(&full[sl])), "r"(plane_bytes) : "memory");
    for (int fi = 0; fi < nin; ++fi)
      asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                       hi_smem_u32(tile + (sl * nin + fi) * FS)),
                   "l"(&ta.tmap[fi]), "r"(tx0), "r"(ty0), "r"(plane + ta.za_off), "r"(hi_smem_u32(&full[sl]))
                   : "memory");
  };
  auto wait_full = [&](int sl, unsigned parity) {
    unsigned done;
    do {
      asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\nselp.u32 %0, 1, 0, p;\n}\n"
                   : "=r"(done) : "r"(hi_smem_u32(&full[sl])), "r"(parity), "r"(20000u) : "memory");
    } while (!done);
  };
  if (producer) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(hi_smem_u32(&full[0])), "r"(1));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(hi_smem_u32(&full[1])), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (producer && kc1 > kc0) { issue(kc0, 0); issue(kc0 + 1, 1); }

  long long o = g.idx(ic, jc, kc0);
  for (int k = kc0, n = 0; k < kc1; ++k, ++n, o += g.sz) {
    const int buf = n & 1;
    const int zk = g.zi(k);
    const Real rdzc = Real(g.rdzc[zk]), rdzf = Real(g.rdzf[zk]);
    const bool first = n == 0;
    wait_full(buf, (unsigned)((n >> 1) & 1));             // plane k
    wait_full(buf ^ 1, (unsigned)(((n + 1) >> 1) & 1));   // plane k+1 (requested a whole plane-time ago)
    const Real *P0 = tile + buf * nin * FS + pos0;        // plane k, this thread's cell, field 0
    const Real *P1 = tile + (buf ^ 1) * nin * FS + pos0;  // plane k+1
    // velocity divergence of the cell in double-double (tracers, H1)
    double Dsum = 0.0;
    if (m.n_tracers > 0) {
      double D = 0.0, Dlo = 0.0;
      if (m.adv[0] != OCN_ADV_NONE) dd_add_diff_scaled((double)P0[1], (double)P0[0], g.rdx, g.rdx_lo, D, Dlo);
      if (m.adv[1] != OCN_ADV_NONE) dd_add_diff_scaled((double)P0[FS + TW], (double)P0[FS], g.rdy, g.rdy_lo, D, Dlo);
      if (m.adv[2] != OCN_ADV_NONE) dd_add_diff_scaled((double)P1[2 * FS], (double)P0[2 * FS], g.rdzc[zk], g.rdzc_lo[zk], D, Dlo);
      Dsum = D + Dlo;
    }
    // ONE instance of the reconstruction code per direction serves every field: runtime loop over the fields
#pragma unroll 1
    for (int f = 0; f < nf; ++f) {
      const bool tr = f >= fc0;
      const int fi = tr ? 3 + (f - fc0) : f;              // index among the staged input fields
      const Real *Qk = P0 + fi * FS;                      // shared memory: plane k
      const Real *Qg = gin(fi) + o;                       // global memory: the z-stencils
      const Real c0 = tr ? Qk[0] : Real(0);
      Real part = Real(0);
      // the z-stencil of the high face: planes k-R+1 .. k+R; k and k+1 are staged, the other 2R-2 values of this thread's column
      // start their way into the thread's own shared-memory slots now and are read after the x- and y-work (no registers held,
      // no load latency on the in-order path: ncu showed the z-stencil's first use at 8 % of all stall samples)
      const bool zweno = m.adv[2] == HI && ta.zwin != 0;
      if (zweno) {
#pragma unroll
        for (int t = 0; t < 2 * R - 2; ++t) hi_cp_async(zwb + t * TY * 32 + slot_, Qg + (long long)(t < R - 1 ? t - R + 1 : t - R + 3) * SZ);
        asm volatile("cp.async.commit_group;" ::: "memory");
      }
      // ---------------- x and y together where both use WENO (PAIR instantiations): the two reconstructions sit in ONE basic block, so
      // the instruction scheduler interleaves their dependent chains (ncu r2: "wait" — fixed-latency dependency — was the top stall
      // with four warps per scheduler and one reconstruction in flight per warp)
      bool pair_done = false;
      if (PAIR && m.adv[0] == HI && m.adv[1] == HI) {
        Real avx, avy;
        if (tr) { avx = P0[0]; avy = P0[FS]; }
        else if (f == 0) { avx = centered_hi<Real, R>(P0, 1); avy = centered_hi<Real, R>(P0 + FS, 1); }
        else if (f == 1) { avx = centered_hi<Real, R>(P0, TW); avy = centered_hi<Real, R>(P0 + FS, TW); }
        else { avx = centered_hi<Real, R>(a.u + o, SZ); avy = centered_hi<Real, R>(a.v + o, SZ); }
        const bool px = avx > Real(0), py = avy > Real(0);
        Real vx[2 * R - 1], vy[2 * R - 1];
        {
          Real qx[2 * R], qy[2 * R];
#pragma unroll
          for (int t = 0; t < 2 * R; ++t) { qx[t] = Qk[t - R]; qy[t] = Qk[(t - R) * TW]; }
#pragma unroll
          for (int t = 0; t < 2 * R - 1; ++t) { vx[t] = px ? qx[t] : qx[2 * R - 1 - t]; vy[t] = py ? qy[t] : qy[2 * R - 1 - t]; }
        }
        const Real cupx = vx[R - 1], cupy = vy[R - 1];
        const Real valx = weno_hi_anom<Real, R>(vx, eps), valy = weno_hi_anom<Real, R>(vy, eps);
        const Real nbx_ = tr ? Qk[-1] : Real(0), nby_ = tr ? Qk[-TW] : Real(0);
        const Real Fxo = avx * (valx + (cupx - c0)), Fxn = avx * (valx + (cupx - nbx_));
        const Real Fyo = avy * (valy + (cupy - c0)), Fyn = avy * (valy + (cupy - nby_));
        part -= (__shfl_down_sync(0xffffffffu, Fxn, 1) - Fxo) * rdx;
        FY(buf, f, row) = Fyn;
        part += Fyo * rdy;
        pair_done = true;
      }
      // ---------------- x: LOW face of the control volume, operands from the staged plane
      if (m.adv[0] != OCN_ADV_NONE && !pair_done) {
        const bool weno = m.adv[0] == HI;
        Real av;
        if (tr) av = P0[0];
        else if (f == 0) av = interp_hi<Real, R>(weno, P0, 1);                     // u~ along x
        else if (f == 1) av = interp_hi<Real, R>(weno, P0, TW);                    // u~ along y  (B21)
        else av = interp_hi<Real, R>(weno, a.u + o, SZ);                           // u~ along z
        Real cup;
        const Real val = face_anom<Real, R>(weno, Qk, 1, av, eps, cup);
        const Real nbr = tr ? Qk[-1] : Real(0);
        const Real Fown = av * (val + (cup - c0)), Fnbr = av * (val + (cup - nbr));
        part -= (__shfl_down_sync(0xffffffffu, Fnbr, 1) - Fown) * rdx;
      }
      // ---------------- y: LOW face; the high face comes from row+1 through shared memory.  The warp whose row equals the field
      // index takes a second trip for the top edge of the tile (row TY): same code instance, operands TY - row rows up
      if (m.adv[1] != OCN_ADV_NONE) {
        const bool weno = m.adv[1] == HI;
        const int trips = row == f ? 2 : 1;
#pragma unroll 1
        for (int yr = pair_done ? 1 : 0; yr < trips; ++yr) {
          const int dr = yr ? (TY - row) * TW : 0;
          const Real *Py = P0 + dr, *Qy = Qk + dr;
          Real av;
          if (tr) av = Py[FS];
          else if (f == 0) av = interp_hi<Real, R>(weno, Py + FS, 1);                // v~ along x
          else if (f == 1) av = interp_hi<Real, R>(weno, Py + FS, TW);               // v~ along y
          else av = interp_hi<Real, R>(weno, a.v + o + (yr ? og : 0), SZ);           // v~ along z
          Real cup;
          const Real val = face_anom<Real, R>(weno, Qy, TW, av, eps, cup);
          const Real own = tr ? Qy[0] : Real(0), nbr = tr ? Qy[-TW] : Real(0);
          const Real Fown = av * (val + (cup - own)), Fnbr = av * (val + (cup - nbr));
          FY(buf, f, yr ? TY : row) = Fnbr;
          if (!yr) part += Fown * rdy;
        }
      } else {
        FY(buf, f, row) = Real(0);
        if (row == f) FY(buf, f, TY) = Real(0);
      }
      // ---------------- z: HIGH face (plus, on the first plane of a chunk, the low one); stencils from global memory
      if (m.adv[2] != OCN_ADV_NONE) {
        const bool weno = m.adv[2] == HI;
        Real Flo_prime = Real(0);
#pragma unroll 1
        for (int pass = first ? 0 : 1; pass < 2; ++pass) {
          const bool hiface = pass == 1;
          const Real *Pw = (hiface ? P1 : P0) + 2 * FS;                            // w on the plane of the face
          const long long fo = hiface ? SZ : 0;
          Real av;
          if (tr) av = Pw[0];
          else if (f == 0) av = interp_hi<Real, R>(weno, Pw, 1);                   // w~ along x
          else if (f == 1) av = interp_hi<Real, R>(weno, Pw, TW);                  // w~ along y
          else av = interp_hi<Real, R>(weno, a.w + o + fo, SZ);                    // w~ along z
          Real cup, val;
          if (zweno && hiface) {
            Real q[2 * R];
            asm volatile("cp.async.wait_all;" ::: "memory");
#pragma unroll
            for (int t = 0; t < R - 1; ++t) { q[t] = zwb[t * TY * 32 + slot_]; q[R + 1 + t] = zwb[(R - 1 + t) * TY * 32 + slot_]; }
            q[R - 1] = Qk[0]; q[R] = P1[fi * FS];
            val = face_anom_vals<Real, R>(q, av, eps, cup);
          } else {
            val = face_anom<Real, R>(weno, Qg + fo, SZ, av, eps, cup);
          }
          const Real nbr = tr ? (hiface ? P1[fi * FS] : Qg[-SZ]) : Real(0);        // the cell on the other side of the face
          const Real Fown = av * (val + (cup - c0)), Fnbr = av * (val + (cup - nbr));
          if (!hiface) {
            Flo_prime = Fown;
          } else {
            const Real Flo = first ? Flo_prime : FZ(f);
            FZ(f) = Fnbr;
            part -= (Fown - Flo) * ((!tr && f == 2) ? rdzf : rdzc);
          }
        }
      }
      // ---- pointwise terms: horizontal neighbours and level k+1 from the staged planes, level k-1 from global memory
      auto lap_xy = [&](const Real *q) -> Real {
        const Real q0 = q[0];
        return ((q[1] - q0) - (q0 - q[-1])) * Real(g.rdx * g.rdx) + ((q[TW] - q0) - (q0 - q[-TW])) * Real(g.rdy * g.rdy);
      };
      auto lap_zc = [&](const Real *q) -> Real {          // fields centred in z
        const Real q0 = q[0];
        return ((P1[fi * FS] - q0) * Real(g.rdzf[zk + 1]) - (q0 - Qg[-SZ]) * Real(g.rdzf[zk])) * Real(g.rdzc[zk]);
      };
      if (tr) {
        part -= Real((double)c0 * Dsum);
        if (m.kappa[f - fc0] != 0.0) {
          Real sxy = lap_xy(Qk);
          if (!m.vimplicit) sxy += lap_zc(Qk);
          part += Real(m.kappa[f - fc0]) * sxy;
        }
      } else if (f == 0) {
        if (m.coriolis) {                                  // reading R8: f at y_c[j]
          const Real *V = P0 + FS;
          const double fc = m.f0 + m.beta * ((j - 0.5) * g.dy - m.y0);
          part += Real(fc) * (Real(0.25) * ((V[-1] + V[0]) + (V[TW - 1] + V[TW])));
        }
        if (m.nu != 0.0) {
          Real sxy = lap_xy(Qk);
          if (!m.vimplicit) sxy += lap_zc(Qk);
          part += Real(m.nu) * sxy;
        }
        if (m.hydrostatic && a.phy != nullptr) part -= (a.phy[o] - a.phy[o - 1]) * rdx;
      } else if (f == 1) {
        if (m.coriolis) {                                  // f at y_f[j]
          const Real *U = P0;
          const double fc = m.f0 + m.beta * ((j - 1.0) * g.dy - m.y0);
          part -= Real(fc) * (Real(0.25) * ((U[-TW] + U[1 - TW]) + (U[0] + U[1])));
        }
        if (m.nu != 0.0) {
          Real sxy = lap_xy(Qk);
          if (!m.vimplicit) sxy += lap_zc(Qk);
          part += Real(m.nu) * sxy;
        }
        if (m.hydrostatic && a.phy != nullptr) part -= (a.phy[o] - a.phy[o - g.sy]) * rdy;
      } else {
        if (m.buoyancy) {                                  // readings R9, R10
          double bsum = 0.0;
          for (int dk = -1; dk <= 0; ++dk) {
            double T = 0.0, Sa = 0.0;
            if (m.idx_T >= 0) T = (double)(dk ? a.c[m.idx_T][o - g.sz] : P0[(3 + m.idx_T) * FS]) - g.Tref[zk + dk];
            if (m.idx_S >= 0) Sa = (double)(dk ? a.c[m.idx_S][o - g.sz] : P0[(3 + m.idx_S) * FS]) - g.Sref[zk + dk];
            bsum += m.g * (m.alpha_T * T - m.beta_S * Sa);
          }
          part += Real(0.5 * bsum);
        }
        if (m.nu != 0.0) {
          const Real q0 = Qk[0];
          Real sxy = lap_xy(Qk);
          if (!m.vimplicit) sxy += ((P1[fi * FS] - q0) * Real(g.rdzc[zk]) - (q0 - Qg[-SZ]) * Real(g.rdzc[zk - 1])) * rdzf;
          part += Real(m.nu) * sxy;
        }
      }
      PB(f) = part;
    }
    __syncthreads();
    if (producer && k + 2 <= kc1) issue(k + 2, buf);       // every thread is done with plane k: its slot takes plane k+2
    if (store) {
      if constexpr (RK != 0) {
        // the state value comes from global memory (L2: the plane was just staged; its shared-memory slot is being refilled) and
        // every load of the substage is issued before the first store
        Real qv[TMA_MAXIN], gp[TMA_MAXIN];
#pragma unroll
        for (int f = 0; f < TMA_MAXIN; ++f) {
          if (f < nf) {
            const int fi = f >= fc0 ? 3 + (f - fc0) : f;
            qv[f] = gin(fi)[o];
            gp[f] = RK == 2 ? ta.Gp[fi][o] : Real(0);
          }
        }
#pragma unroll
        for (int f = 0; f < TMA_MAXIN; ++f) {
          if (f < nf) {
            const int fi = f >= fc0 ? 3 + (f - fc0) : f;
            const bool wall = f < fc0 && g.topo[f] == OCN_BOUNDED && (f == 0 ? i : (f == 1 ? j : k)) == 1;
            const Real Gf = wall ? Real(0) : PB(f) - FY(buf, f, row + 1) * rdy;   // wall faces of wall-normal velocities: G = 0, q untouched
            Real *Gm = f >= fc0 ? a.Gc[f - fc0] : (f == 0 ? a.Gu : (f == 1 ? a.Gv : a.Gw));
            Gm[o] = Gf;
            const Real qn = RK == 2 ? rk3_update(qv[f], Gf, gp[f], ta.rk_a, ta.rk_b) : rk3_update(qv[f], Gf, ta.rk_a);
            ta.Qn[fi][o] = wall ? qv[f] : qn;
          }
        }
      } else {
        for (int f = 0; f < nf; ++f) {
          const Real Gf = PB(f) - FY(buf, f, row + 1) * rdy;
          if (f < fc0) {                                      // wall faces of wall-normal velocities: G = 0
            const bool wall = g.topo[f] == OCN_BOUNDED && (f == 0 ? i : (f == 1 ? j : k)) == 1;
            Real *Gm = f == 0 ? a.Gu : (f == 1 ? a.Gv : a.Gw);
            Gm[o] = wall ? Real(0) : Gf;
          } else {
            a.Gc[f - fc0][o] = Gf;
          }
        }
      }
    }
  }
}

template <class Real>
void fill_hargs(HArgs<Real> &a, const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G, const Rk3Fuse *rk) {
  memset(&a, 0, sizeof(a));
  a.g = g->dev;
  a.m = m;
  a.u = (const Real *)st.u; a.v = (const Real *)st.v; a.w = (const Real *)st.w; a.phy = (const Real *)phy;
  a.Gu = (Real *)G.u; a.Gv = (Real *)G.v; a.Gw = (Real *)G.w;
  for (int n = 0; n < OCN_MAX_TRACERS; ++n) { a.c[n] = (const Real *)st.c[n]; a.Gc[n] = (Real *)G.c[n]; }
  if (rk) {
    a.Pu = (const Real *)rk->Gp.u; a.Pv = (const Real *)rk->Gp.v; a.Pw = (const Real *)rk->Gp.w;
    a.Qu = (Real *)rk->Qn.u; a.Qv = (Real *)rk->Qn.v; a.Qw = (Real *)rk->Qn.w;
    for (int n = 0; n < OCN_MAX_TRACERS; ++n) { a.Pc[n] = (const Real *)rk->Gp.c[n]; a.Qc[n] = (Real *)rk->Qn.c[n]; }
    a.rk_a = Real(rk->a); a.rk_b = Real(rk->b);
  }
}

template <class Real, int R, int RK>
int launch_march_t(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G, const Rk3Fuse *rk, cudaStream_t s) {
  constexpr int TY = 7;
  MArgs<Real> ma;
  fill_hargs<Real>(ma.h, g, m, st, phy, G, rk);
  ma.nf = m.n_tracers + (m.momentum ? (m.hydrostatic ? 2 : 3) : 0);
  const int nbx = (g->Nx + 30) / 31, nby = (g->Ny + TY - 1) / TY;
  // z-chunks: >= 8 waves of 2 blocks per SM where the grid allows it, chunks of >= 16 planes (each chunk primes one face)
  int nch = (8 * 2 * 148 + nbx * nby - 1) / (nbx * nby);
  nch = std::max(1, std::min(nch, (g->Nz + 15) / 16));
  ma.kchunk = (g->Nz + nch - 1) / nch;
  nch = (g->Nz + ma.kchunk - 1) / ma.kchunk;
  const size_t smem = (size_t)ma.nf * (2 * (TY + 1) + 2 * TY) * 32 * sizeof(Real);
  auto kern = tend_hiorder_march_kernel<Real, R, TY, RK>;
  static OcnPerDeviceOnce attr_once;
  if (attr_once.first()) {
    OCN_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 11 * (2 * (TY + 1) + 2 * TY) * 32 * (int)sizeof(Real)));
  }
  dim3 block(32, TY + 1, 1), grid(nbx, nby, nch);
  kern<<<grid, block, smem, s>>>(ma);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "tend_hiorder_march_kernel launch");
}

// the staged kernel when its tiles fit two blocks per SM (<= 3 tracers in fp64 at R = 5), else *done stays false
constexpr int STAGED_TY = 8;                             // rows per tile = warps per block (>= the number of tendency fields)

// does the staged kernel apply?  3-D grid with every velocity component, <= 3 tracers, tiles that fit two blocks per SM
template <class Real, int R>
bool staged_fits(const ModelDev &m) {
  using SG = StagedGeom<Real, R, STAGED_TY>;
  const int nin = 3 + m.n_tracers, nf = m.n_tracers + (m.momentum ? (m.hydrostatic ? 2 : 3) : 0);
  if (nin > TMA_MAXIN || nf < 1 || nf > STAGED_TY) return false;
  return 2 * (SG::bytes(nin, nf, false) + 1024) <= 227 * 1024;
}

template <class Real, int R, int RK>
int launch_staged_t(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G, const Rk3Fuse *rk,
                    cudaStream_t s, bool *done) {
  constexpr int TY = STAGED_TY;
  using SG = StagedGeom<Real, R, TY>;
  *done = false;
  auto enc = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(ocn_tensormap_encoder());
  const int nin = 3 + m.n_tracers, nf = m.n_tracers + (m.momentum ? (m.hydrostatic ? 2 : 3) : 0);
  if (!enc || !staged_fits<Real, R>(m)) return OCN_OK;
  const bool zwin = 2 * (SG::bytes(nin, nf, true) + 1024) <= 227 * 1024;   // the per-thread z-windows, when two blocks per SM still fit
  const size_t smem = SG::bytes(nin, nf, zwin);
  TArgs<Real> ta;
  memset(&ta, 0, sizeof(ta));
  HArgs<Real> &a = ta.h;
  a.g = g->dev;
  a.m = m;
  a.u = (const Real *)st.u; a.v = (const Real *)st.v; a.w = (const Real *)st.w; a.phy = (const Real *)phy;
  a.Gu = (Real *)G.u; a.Gv = (Real *)G.v; a.Gw = (Real *)G.w;
  for (int n = 0; n < OCN_MAX_TRACERS; ++n) { a.c[n] = (const Real *)st.c[n]; a.Gc[n] = (Real *)G.c[n]; }
  ta.nf = nf; ta.nin = nin; ta.zwin = zwin ? 1 : 0;
  if (RK != 0) {
    const void *gp[TMA_MAXIN] = {rk->Gp.u, rk->Gp.v, rk->Gp.w, rk->Gp.c[0], rk->Gp.c[1], rk->Gp.c[2]};
    void *qn[TMA_MAXIN] = {rk->Qn.u, rk->Qn.v, rk->Qn.w, rk->Qn.c[0], rk->Qn.c[1], rk->Qn.c[2]};
    for (int f = 0; f < nin; ++f) { ta.Gp[f] = (const Real *)gp[f]; ta.Qn[f] = (Real *)qn[f]; }
    ta.rk_a = Real(rk->a); ta.rk_b = Real(rk->b);
  }
  const ocn_layout &L = g->lay;
  const void *in[TMA_MAXIN] = {st.u, st.v, st.w, st.c[0], st.c[1], st.c[2]};
  for (int f = 0; f < nin; ++f) {
    cuuint64_t dims[3] = {(cuuint64_t)L.stride_y, (cuuint64_t)L.ny_pad, (cuuint64_t)L.nz_pad};
    cuuint64_t strides[2] = {(cuuint64_t)L.stride_y * sizeof(Real), (cuuint64_t)L.stride_z * sizeof(Real)};
    cuuint32_t box[3] = {(cuuint32_t)SG::TW, (cuuint32_t)SG::TH, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(&ta.tmap[f], sizeof(Real) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3,
                     const_cast<void *>(in[f]), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return ocn_fail(OCN_ERR_CUDA, "tend_hiorder: cuTensorMapEncodeTiled failed (%d) for field %d", (int)r, f);
  }
  const int xoff = (int)(L.offset0 - (long long)L.hz * L.stride_z - (long long)L.hy * L.stride_y);   // array x of logical i = 1
  ta.xa_off = xoff - 1; ta.ya_off = L.hy - 1; ta.za_off = L.hz - 1;
  const int nbx = (g->Nx + 30) / 31, nby = (g->Ny + TY - 1) / TY;
  // z-chunks: >= 8 waves of 2 blocks per SM where the grid allows it, chunks of >= 16 planes (each chunk primes one face)
  int nch = (8 * 2 * 148 + nbx * nby - 1) / (nbx * nby);
  nch = std::max(1, std::min(nch, (g->Nz + 15) / 16));
  ta.kchunk = (g->Nz + nch - 1) / nch;
  nch = (g->Nz + ta.kchunk - 1) / ta.kchunk;
  auto kern = tend_hiorder_tma_kernel<Real, R, TY, RK>;
  static OcnPerDeviceOnce attr_once;
  if (attr_once.first()) OCN_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 113 * 1024));
  dim3 block(32, TY, 1), grid(nbx, nby, nch);
  kern<<<grid, block, smem, s>>>(ta);
  ocn_count_launch();
  *done = true;
  return ocn_check_cuda(cudaGetLastError(), "tend_hiorder_tma_kernel launch");
}

template <class Real, int R, int RK>
int launch_t(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G, const Rk3Fuse *rk, cudaStream_t s) {
  HArgs<Real> a;
  fill_hargs<Real>(a, g, m, st, phy, G, rk);
  dim3 block(32, 4, 1);
  dim3 grid((g->Nx + block.x - 1) / block.x, (g->Ny + block.y - 1) / block.y, g->Nz);
  tend_hiorder_kernel<Real, R, RK><<<grid, block, 0, s>>>(a);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "tend_hiorder_kernel launch");
}

}  // namespace

static int hiorder_order(const ModelDev &m) {
  int order = 0;
  for (int a = 0; a < 3; ++a)
    if (m.adv[a] == OCN_ADV_WENO7 || m.adv[a] == OCN_ADV_WENO9) order = m.adv[a];
  return order;
}

static bool march_applies(const ocn_grid *g, const FieldsDev &st) {
  return g->kernel != OCN_KERNEL_PERCELL && g->topo[0] != OCN_FLAT && g->topo[1] != OCN_FLAT && g->topo[2] != OCN_FLAT && st.u && st.v && st.w;
}

template <int RK>
static int dispatch_staged(const ocn_grid *g, const ModelDev &m, int order, const FieldsDev &st, const void *phy, const FieldsDev &G,
                           const Rk3Fuse *rk, cudaStream_t s, bool *done) {
  if (g->dtype == OCN_F64)
    return order == 7 ? launch_staged_t<double, 4, RK>(g, m, st, phy, G, rk, s, done) : launch_staged_t<double, 5, RK>(g, m, st, phy, G, rk, s, done);
  return order == 7 ? launch_staged_t<float, 4, RK>(g, m, st, phy, G, rk, s, done) : launch_staged_t<float, 5, RK>(g, m, st, phy, G, rk, s, done);
}

// Every WENO7/9 model can run ocn_tendencies_rk3: the TMA-staged marching kernel where it applies, else the global-load marching
// kernel or the per-cell kernel, each with the substage fused in (RK template parameter).
bool hiorder_rk3_applicable(const ocn_grid *g, const ModelDev &m, std::string *why) {
  auto no = [&](const char *w) { if (why) *why = w; return false; };
  if (!hiorder_order(m)) return no("no WENO7/WENO9 axis");
  if (m.momentum && !m.hydrostatic && g->topo[2] != OCN_FLAT && !g->uniform_z) return no("nonhydrostatic momentum on a stretched z axis");
  return true;
}

template <int RK>
static int dispatch_hiorder(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G, const Rk3Fuse *rk,
                            cudaStream_t s) {
  const int order = hiorder_order(m);
  if (!order) return ocn_fail(OCN_ERR_INVALID, "tend_hiorder: no WENO7/WENO9 axis");
  if (m.momentum && !m.hydrostatic && g->topo[2] != OCN_FLAT && !g->uniform_z)
    return ocn_fail(OCN_ERR_UNSUPPORTED, "tend_hiorder: nonhydrostatic momentum on a stretched z axis is not supported with WENO%d", order);
  // 3-D grids with a velocity along every axis: the marching kernels (every face flux once); anything else
  // (Flat axes, missing components) or OCN_KERNEL_PERCELL: the per-cell kernel
  if (march_applies(g, st)) {
    // the TMA-staged marching kernel where it applies (halo >= R is guaranteed by the scheme check of the API); the per-grid
    // flag OCN_DIAG_HI_NOSTAGE is a diagnostic switch that keeps the global-load marching kernel under test
    if (!(g->diag & OCN_DIAG_HI_NOSTAGE)) {
      bool done = false;
      const int rc = dispatch_staged<RK>(g, m, order, st, phy, G, rk, s, &done);
      if (rc || done) return rc;
    }
    if (g->dtype == OCN_F64)
      return order == 7 ? launch_march_t<double, 4, RK>(g, m, st, phy, G, rk, s) : launch_march_t<double, 5, RK>(g, m, st, phy, G, rk, s);
    return order == 7 ? launch_march_t<float, 4, RK>(g, m, st, phy, G, rk, s) : launch_march_t<float, 5, RK>(g, m, st, phy, G, rk, s);
  }
  if (g->dtype == OCN_F64)
    return order == 7 ? launch_t<double, 4, RK>(g, m, st, phy, G, rk, s) : launch_t<double, 5, RK>(g, m, st, phy, G, rk, s);
  return order == 7 ? launch_t<float, 4, RK>(g, m, st, phy, G, rk, s) : launch_t<float, 5, RK>(g, m, st, phy, G, rk, s);
}

int launch_tendencies_rk3_hiorder(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G,
                                  const Rk3Fuse &rk, cudaStream_t s) {
  return rk.use_prev ? dispatch_hiorder<2>(g, m, st, phy, G, &rk, s) : dispatch_hiorder<1>(g, m, st, phy, G, &rk, s);
}

int launch_tendencies_hiorder(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy,
                              const FieldsDev &G, cudaStream_t s) {
  return dispatch_hiorder<0>(g, m, st, phy, G, nullptr, s);
}
