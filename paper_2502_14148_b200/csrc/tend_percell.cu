// tend_percell.cu — OCN_KERNEL_PERCELL: one thread per interior cell, every term, every scheme and topology,
// operands straight from global memory (L1/L2).  It is the general kernel (small grids, 2-D, Upwind1 /
// Centered2 horizontally) and the "before" number for the fused 2.5-D kernels in tend_fused.cu.
//
// Discrete operators: SURVEY 8(c) c.4 / DESIGN.md "operators":
//   tracers   (B2),(B3) PAPER.md:990-1003   momentum flux form (7),(18),(B21) PAPER.md:329,512,1072-1074
//   Coriolis  eq. 6/17 PAPER.md:318,506     buoyancy eq. 4,6 PAPER.md:300,318    Laplacian eq. 8
// Tracers use the cancellation-free form (H1):  div(u c) = sum_faces u_f ([c]_f - c_ijk) + c_ijk div(u),
// with div(u) accumulated in double-double.
#include <cstring>

#include "ocn_internal.h"
#include "recon.cuh"

namespace {

using namespace ocn;

template <class Real>
struct Acc {
  const Real *__restrict__ q;
  long long sy, sz, o;   // o = flat offset of (i,j,k)
  __device__ __forceinline__ Real operator()(int di, int dj, int dk) const { return q[o + di + dj * sy + dk * sz]; }
};

template <class Real>
struct KArgs {
  GridDev g;
  ModelDev m;
  const Real *u, *v, *w, *phy;
  const Real *c[OCN_MAX_TRACERS];
  Real *Gu, *Gv, *Gw;
  Real *Gc[OCN_MAX_TRACERS];
  // fused substage (A4) (RK != 0): q_new = q + (rk_a G - rk_b G_prev) into the other state buffer of the ping-pong pair
  const Real *Pu, *Pv, *Pw;
  const Real *Pc[OCN_MAX_TRACERS];
  Real *Qu, *Qv, *Qw;
  Real *Qc[OCN_MAX_TRACERS];
  Real rk_a, rk_b;
};

// store G and, with the substage fused in, the new state (same arithmetic as rk3.cu: rk3_update); wall: G is 0 and q stays
template <int RK, class Real>
__device__ __forceinline__ void store_GQ(Real *Gf, const Real *Pf, Real *Qf, long long o, Real G, Real q, bool wall, Real rk_a, Real rk_b) {
  Gf[o] = G;
  if constexpr (RK != 0) {
    const Real qn = RK == 2 ? rk3_update(q, G, Pf[o], rk_a, rk_b) : rk3_update(q, G, rk_a);
    Qf[o] = wall ? q : qn;
  }
}

// 7-point Laplacian of a field centred in z (c, u, v): flux-divergence form (B2) on the rectilinear grid
template <class Real>
__device__ __forceinline__ Real lap_center(const GridDev &g, const Acc<Real> &q, int k, bool hx, bool hy, bool hz) {
  const Real q0 = q(0, 0, 0);
  Real s = Real(0);
  if (hx) s += ((q(1, 0, 0) - q0) - (q0 - q(-1, 0, 0))) * Real(g.rdx * g.rdx);
  if (hy) s += ((q(0, 1, 0) - q0) - (q0 - q(0, -1, 0))) * Real(g.rdy * g.rdy);
  if (hz) {
    const int z = g.zi(k);
    s += ((q(0, 0, 1) - q0) * Real(g.rdzf[z + 1]) - (q0 - q(0, 0, -1)) * Real(g.rdzf[z])) * Real(g.rdzc[z]);
  }
  return s;
}

// RK: 0 tendencies only, 1 fused substage without G_prev (zeta = 0), 2 with G_prev
template <class Real, int RK>
__global__ void __launch_bounds__(128) tend_percell_kernel(const KArgs<Real> a) {
  const GridDev &g = a.g;
  const ModelDev &m = a.m;
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1;
  const int j = blockIdx.y * blockDim.y + threadIdx.y + 1;
  const int k = blockIdx.z + 1;
  if (i > g.Nx || j > g.Ny) return;
  const long long o = g.idx(i, j, k);
  const bool hx = g.topo[0] != OCN_FLAT, hy = g.topo[1] != OCN_FLAT, hz = g.topo[2] != OCN_FLAT;
  const int sx_ = m.adv[0], sy_ = m.adv[1], sz_ = m.adv[2];
  const Real eps4 = Real(4.0 * m.weno_eps);
  const int zk = g.zi(k);
  const Real rdx = Real(g.rdx), rdy = Real(g.rdy);
  const Real rdzc = hz ? Real(g.rdzc[zk]) : Real(0);
  const Acc<Real> U{a.u, g.sy, g.sz, o}, V{a.v, g.sy, g.sz, o}, W{a.w, g.sy, g.sz, o};
  const bool haveu = hx && a.u != nullptr && sx_ != S_NONE;
  const bool havev = hy && a.v != nullptr && sy_ != S_NONE;
  const bool havew = hz && a.w != nullptr && sz_ != S_NONE;

  // ------------------------------------------------------------------ tracers
  if (m.n_tracers > 0) {
    const Real ul = haveu ? U(0, 0, 0) : Real(0), uh = haveu ? U(1, 0, 0) : Real(0);
    const Real vl = havev ? V(0, 0, 0) : Real(0), vh = havev ? V(0, 1, 0) : Real(0);
    const Real wl = havew ? W(0, 0, 0) : Real(0), wh = havew ? W(0, 0, 1) : Real(0);
    // velocity divergence D in double-double (the discrete divergence of the input is a rounding-level
    // quantity that multiplies the large tracer mean: it has to be reproduced, not dropped)
    double D = 0.0, Dlo = 0.0;
    if (haveu) dd_add_diff_scaled((double)uh, (double)ul, g.rdx, g.rdx_lo, D, Dlo);
    if (havev) dd_add_diff_scaled((double)vh, (double)vl, g.rdy, g.rdy_lo, D, Dlo);
    if (havew) dd_add_diff_scaled((double)wh, (double)wl, g.rdzc[zk], g.rdzc_lo[zk], D, Dlo);
    const double Dsum = D + Dlo;
    for (int n = 0; n < m.n_tracers; ++n) {
      const Acc<Real> C{a.c[n], g.sy, g.sz, o};
      const Real c0 = C(0, 0, 0);
      Real adv = Real(0);
      if (haveu) {
        const Real m3 = C(-3, 0, 0), m2 = C(-2, 0, 0), m1 = C(-1, 0, 0), p1 = C(1, 0, 0), p2 = C(2, 0, 0), p3 = C(3, 0, 0);
        const Real Rl = recon_rel<Real>(sx_, m3, m2, m1, c0, p1, p2, ul, c0, eps4);
        const Real Rh = recon_rel<Real>(sx_, m2, m1, c0, p1, p2, p3, uh, c0, eps4);
        adv += (uh * Rh - ul * Rl) * rdx;
      }
      if (havev) {
        const Real m3 = C(0, -3, 0), m2 = C(0, -2, 0), m1 = C(0, -1, 0), p1 = C(0, 1, 0), p2 = C(0, 2, 0), p3 = C(0, 3, 0);
        const Real Rl = recon_rel<Real>(sy_, m3, m2, m1, c0, p1, p2, vl, c0, eps4);
        const Real Rh = recon_rel<Real>(sy_, m2, m1, c0, p1, p2, p3, vh, c0, eps4);
        adv += (vh * Rh - vl * Rl) * rdy;
      }
      if (havew) {
        Real m3 = Real(0), p3 = Real(0);
        if (sz_ == S_WENO5) { m3 = C(0, 0, -3); p3 = C(0, 0, 3); }
        const Real m2 = C(0, 0, -2), m1 = C(0, 0, -1), p1 = C(0, 0, 1), p2 = C(0, 0, 2);
        const Real Rl = recon_rel<Real>(sz_, m3, m2, m1, c0, p1, p2, wl, c0, eps4);
        const Real Rh = recon_rel<Real>(sz_, m2, m1, c0, p1, p2, p3, wh, c0, eps4);
        adv += (wh * Rh - wl * Rl) * rdzc;
      }
      const Real cD = Real((double)c0 * Dsum);
      Real G = -adv - cD;
      if (m.kappa[n] != 0.0) G += Real(m.kappa[n]) * lap_center<Real>(g, C, k, hx, hy, hz && !m.vimplicit);
      store_GQ<RK, Real>(a.Gc[n], a.Pc[n], a.Qc[n], o, G, c0, false, a.rk_a, a.rk_b);
    }
  }
  if (!m.momentum) return;

  // ------------------------------------------------------------------ u at fcc
  if (a.Gu != nullptr) {
    Real G = Real(0);
    if (i >= first_face(g.topo[0])) {
      Real div = Real(0);
      if (hx && sx_ != S_NONE) {
        const Real m3 = U(-3, 0, 0), m2 = U(-2, 0, 0), m1 = U(-1, 0, 0), q0 = U(0, 0, 0), p1 = U(1, 0, 0), p2 = U(2, 0, 0), p3 = U(3, 0, 0);
        const Real ah = interp_adv<Real>(sx_, m1, q0, p1, p2);     // at centre i   (m = i+1)
        const Real al = interp_adv<Real>(sx_, m2, m1, q0, p1);     // at centre i-1 (m = i)
        const Real Fh = ah * recon_rel<Real>(sx_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sx_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdx;
      }
      if (hy && sy_ != S_NONE && a.v != nullptr) {
        const Real ah = interp_adv<Real>(sy_, V(-2, 1, 0), V(-1, 1, 0), V(0, 1, 0), V(1, 1, 0));   // v along x at y-face j+1
        const Real al = interp_adv<Real>(sy_, V(-2, 0, 0), V(-1, 0, 0), V(0, 0, 0), V(1, 0, 0));
        const Real m3 = U(0, -3, 0), m2 = U(0, -2, 0), m1 = U(0, -1, 0), q0 = U(0, 0, 0), p1 = U(0, 1, 0), p2 = U(0, 2, 0), p3 = U(0, 3, 0);
        const Real Fh = ah * recon_rel<Real>(sy_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sy_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdy;
      }
      if (hz && sz_ != S_NONE && a.w != nullptr) {
        const Real ah = interp_adv<Real>(sz_, W(-2, 0, 1), W(-1, 0, 1), W(0, 0, 1), W(1, 0, 1));   // w along x at z-face k+1
        const Real al = interp_adv<Real>(sz_, W(-2, 0, 0), W(-1, 0, 0), W(0, 0, 0), W(1, 0, 0));
        Real m3 = Real(0), p3 = Real(0);
        if (sz_ == S_WENO5) { m3 = U(0, 0, -3); p3 = U(0, 0, 3); }
        const Real m2 = U(0, 0, -2), m1 = U(0, 0, -1), q0 = U(0, 0, 0), p1 = U(0, 0, 1), p2 = U(0, 0, 2);
        const Real Fh = ah * recon_rel<Real>(sz_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sz_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdzc;
      }
      G = -div;
      if (m.coriolis && a.v != nullptr) {
        const double f = m.f0 + m.beta * ((j - 0.5) * g.dy - m.y0);
        G += Real(f) * (Real(0.25) * ((V(-1, 0, 0) + V(0, 0, 0)) + (V(-1, 1, 0) + V(0, 1, 0))));
      }
      if (m.nu != 0.0) G += Real(m.nu) * lap_center<Real>(g, U, k, hx, hy, hz && !m.vimplicit);
      if (m.hydrostatic && a.phy != nullptr) G -= (a.phy[o] - a.phy[o - 1]) * rdx;
    }
    store_GQ<RK, Real>(a.Gu, a.Pu, a.Qu, o, G, U(0, 0, 0), i < first_face(g.topo[0]), a.rk_a, a.rk_b);
  }

  // ------------------------------------------------------------------ v at cfc
  if (a.Gv != nullptr) {
    Real G = Real(0);
    if (j >= first_face(g.topo[1])) {
      Real div = Real(0);
      if (hx && sx_ != S_NONE && a.u != nullptr) {
        const Real ah = interp_adv<Real>(sx_, U(1, -2, 0), U(1, -1, 0), U(1, 0, 0), U(1, 1, 0));   // u along y at x-face i+1
        const Real al = interp_adv<Real>(sx_, U(0, -2, 0), U(0, -1, 0), U(0, 0, 0), U(0, 1, 0));
        const Real m3 = V(-3, 0, 0), m2 = V(-2, 0, 0), m1 = V(-1, 0, 0), q0 = V(0, 0, 0), p1 = V(1, 0, 0), p2 = V(2, 0, 0), p3 = V(3, 0, 0);
        const Real Fh = ah * recon_rel<Real>(sx_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sx_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdx;
      }
      if (hy && sy_ != S_NONE) {
        const Real m3 = V(0, -3, 0), m2 = V(0, -2, 0), m1 = V(0, -1, 0), q0 = V(0, 0, 0), p1 = V(0, 1, 0), p2 = V(0, 2, 0), p3 = V(0, 3, 0);
        const Real ah = interp_adv<Real>(sy_, m1, q0, p1, p2);
        const Real al = interp_adv<Real>(sy_, m2, m1, q0, p1);
        const Real Fh = ah * recon_rel<Real>(sy_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sy_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdy;
      }
      if (hz && sz_ != S_NONE && a.w != nullptr) {
        const Real ah = interp_adv<Real>(sz_, W(0, -2, 1), W(0, -1, 1), W(0, 0, 1), W(0, 1, 1));   // w along y at z-face k+1
        const Real al = interp_adv<Real>(sz_, W(0, -2, 0), W(0, -1, 0), W(0, 0, 0), W(0, 1, 0));
        Real m3 = Real(0), p3 = Real(0);
        if (sz_ == S_WENO5) { m3 = V(0, 0, -3); p3 = V(0, 0, 3); }
        const Real m2 = V(0, 0, -2), m1 = V(0, 0, -1), q0 = V(0, 0, 0), p1 = V(0, 0, 1), p2 = V(0, 0, 2);
        const Real Fh = ah * recon_rel<Real>(sz_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sz_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdzc;
      }
      G = -div;
      if (m.coriolis && a.u != nullptr) {
        const double f = m.f0 + m.beta * ((j - 1.0) * g.dy - m.y0);
        G -= Real(f) * (Real(0.25) * ((U(0, -1, 0) + U(1, -1, 0)) + (U(0, 0, 0) + U(1, 0, 0))));
      }
      if (m.nu != 0.0) G += Real(m.nu) * lap_center<Real>(g, V, k, hx, hy, hz && !m.vimplicit);
      if (m.hydrostatic && a.phy != nullptr) G -= (a.phy[o] - a.phy[o - g.sy]) * rdy;
    }
    store_GQ<RK, Real>(a.Gv, a.Pv, a.Qv, o, G, V(0, 0, 0), j < first_face(g.topo[1]), a.rk_a, a.rk_b);
  }

  // ------------------------------------------------------------------ w at ccf (nonhydrostatic)
  if (a.Gw != nullptr && !m.hydrostatic && hz) {
    Real G = Real(0);
    if (k >= first_face(g.topo[2])) {
      const Real rdzf = Real(g.rdzf[zk]);                 // 1/Δz_f[k]: thickness of the w control volume
      // Δz_c[k']/Δz_f[k] weights of the area-weighted vertical interpolation of u, v (1 on a uniform grid)
      Real a0 = Real(1), a1 = Real(1), a2 = Real(1), a3 = Real(1);
      if (!g.uniform_z) {
        a0 = Real(g.dzc[zk - 2] * g.rdzf[zk]); a1 = Real(g.dzc[zk - 1] * g.rdzf[zk]);
        a2 = Real(g.dzc[zk] * g.rdzf[zk]);     a3 = Real(g.dzc[zk + 1] * g.rdzf[zk]);
      }
      Real div = Real(0);
      if (hx && sx_ != S_NONE && a.u != nullptr) {
        const Real ah = interp_adv<Real>(sx_, a0 * U(1, 0, -2), a1 * U(1, 0, -1), a2 * U(1, 0, 0), a3 * U(1, 0, 1));   // u along z at x-face i+1
        const Real al = interp_adv<Real>(sx_, a0 * U(0, 0, -2), a1 * U(0, 0, -1), a2 * U(0, 0, 0), a3 * U(0, 0, 1));
        const Real m3 = W(-3, 0, 0), m2 = W(-2, 0, 0), m1 = W(-1, 0, 0), q0 = W(0, 0, 0), p1 = W(1, 0, 0), p2 = W(2, 0, 0), p3 = W(3, 0, 0);
        const Real Fh = ah * recon_rel<Real>(sx_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sx_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdx;
      }
      if (hy && sy_ != S_NONE && a.v != nullptr) {
        const Real ah = interp_adv<Real>(sy_, a0 * V(0, 1, -2), a1 * V(0, 1, -1), a2 * V(0, 1, 0), a3 * V(0, 1, 1));
        const Real al = interp_adv<Real>(sy_, a0 * V(0, 0, -2), a1 * V(0, 0, -1), a2 * V(0, 0, 0), a3 * V(0, 0, 1));
        const Real m3 = W(0, -3, 0), m2 = W(0, -2, 0), m1 = W(0, -1, 0), q0 = W(0, 0, 0), p1 = W(0, 1, 0), p2 = W(0, 2, 0), p3 = W(0, 3, 0);
        const Real Fh = ah * recon_rel<Real>(sy_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sy_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdy;
      }
      if (sz_ != S_NONE) {
        Real m3 = Real(0), p3 = Real(0);
        if (sz_ == S_WENO5) { m3 = W(0, 0, -3); p3 = W(0, 0, 3); }
        const Real m2 = W(0, 0, -2), m1 = W(0, 0, -1), q0 = W(0, 0, 0), p1 = W(0, 0, 1), p2 = W(0, 0, 2);
        const Real ah = interp_adv<Real>(sz_, m1, q0, p1, p2);     // at centre k   (m = k+1)
        const Real al = interp_adv<Real>(sz_, m2, m1, q0, p1);     // at centre k-1 (m = k)
        const Real Fh = ah * recon_rel<Real>(sz_, m2, m1, q0, p1, p2, p3, ah, Real(0), eps4);
        const Real Fl = al * recon_rel<Real>(sz_, m3, m2, m1, q0, p1, p2, al, Real(0), eps4);
        div += (Fh - Fl) * rdzf;
      }
      G = -div;
      if (m.buoyancy) {
        // b = g [alpha (T - Tref) - beta (S - Sref)] at k-1 and k, in double (cheap; keeps fp32 close to the oracle)
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
        const Real q0 = W(0, 0, 0);
        Real s = Real(0);
        if (hx) s += ((W(1, 0, 0) - q0) - (q0 - W(-1, 0, 0))) * Real(g.rdx * g.rdx);
        if (hy) s += ((W(0, 1, 0) - q0) - (q0 - W(0, -1, 0))) * Real(g.rdy * g.rdy);
        if (!m.vimplicit) s += ((W(0, 0, 1) - q0) * Real(g.rdzc[zk]) - (q0 - W(0, 0, -1)) * Real(g.rdzc[zk - 1])) * rdzf;
        G += Real(m.nu) * s;
      }
    }
    store_GQ<RK, Real>(a.Gw, a.Pw, a.Qw, o, G, W(0, 0, 0), k < first_face(g.topo[2]), a.rk_a, a.rk_b);
  }
}

template <class Real, int RK>
int launch_t(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G, const Rk3Fuse *rk, cudaStream_t s) {
  KArgs<Real> a;
  memset(&a, 0, sizeof(a));
  a.g = g->dev;
  a.m = m;
  a.u = (const Real *)st.u; a.v = (const Real *)st.v; a.w = (const Real *)st.w; a.phy = (const Real *)phy;
  a.Gu = (Real *)G.u; a.Gv = (Real *)G.v; a.Gw = (Real *)G.w;
  for (int n = 0; n < OCN_MAX_TRACERS; ++n) { a.c[n] = (const Real *)st.c[n]; a.Gc[n] = (Real *)G.c[n]; }
  if (RK != 0) {
    a.Pu = (const Real *)rk->Gp.u; a.Pv = (const Real *)rk->Gp.v; a.Pw = (const Real *)rk->Gp.w;
    a.Qu = (Real *)rk->Qn.u; a.Qv = (Real *)rk->Qn.v; a.Qw = (Real *)rk->Qn.w;
    for (int n = 0; n < OCN_MAX_TRACERS; ++n) { a.Pc[n] = (const Real *)rk->Gp.c[n]; a.Qc[n] = (Real *)rk->Qn.c[n]; }
    a.rk_a = Real(rk->a); a.rk_b = Real(rk->b);
  }
  dim3 block(32, 4, 1);
  dim3 grid((g->Nx + block.x - 1) / block.x, (g->Ny + block.y - 1) / block.y, g->Nz);
  tend_percell_kernel<Real, RK><<<grid, block, 0, s>>>(a);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "tend_percell_kernel launch");
}

}  // namespace

int launch_tendencies_percell(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy,
                              const FieldsDev &G, cudaStream_t s) {
  if (g->dtype == OCN_F64) return launch_t<double, 0>(g, m, st, phy, G, nullptr, s);
  return launch_t<float, 0>(g, m, st, phy, G, nullptr, s);
}

// tendencies + (A4) substage in one pass on the general kernel (every scheme and topology below WENO7): the path of ocn_tendencies_rk3
// where the TMA kernels do not apply (2-D grids such as C0, prescribed velocities, Upwind1 / Centered2, OCN_KERNEL_PERCELL)
int launch_tendencies_rk3_percell(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G,
                                  const Rk3Fuse &rk, cudaStream_t s) {
  if (g->dtype == OCN_F64)
    return rk.use_prev ? launch_t<double, 2>(g, m, st, phy, G, &rk, s) : launch_t<double, 1>(g, m, st, phy, G, &rk, s);
  return rk.use_prev ? launch_t<float, 2>(g, m, st, phy, G, &rk, s) : launch_t<float, 1>(g, m, st, phy, G, &rk, s);
}
