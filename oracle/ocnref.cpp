// oracle/ocnref.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU statement of the hot path of arXiv 2502.14148
// (Oceananigans): halo fill -> [w from continuity, hydrostatic pressure] -> tendencies
// (WENO5-Z / Centered / Upwind advection, Coriolis, linear-EOS buoyancy, Laplacian
// viscosity/diffusivity) -> low-storage RK3 substage, on a halo-padded Arakawa C-grid.
//
// * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
//   legs may load this library.  It shares no code with paper_2502_14148_b200/csrc.
// * The discrete operators ARE the definition; there is no blocking, fusion
//   or reordering: one function per operator, triple loops over padded arrays, every
//   function cites the passage of PAPER.md (or the DESIGN.md reading R#) it follows.
// * Evaluation type E: long double (x86 80-bit) = the parity reference ("the value of the
//   discrete formula on the given inputs"); double / float = the timed CPU baseline.
//   Storage type S: double or float arrays, dense padded, x fastest.
// * Pins: tests/test_oracle_pins.py (closed forms, invariants, paper constants, brute
//   force).  No function here is "parity unpinned".
//
// Index convention ("Face indices are left of cell indices"): interior cells
// i=1..Nx; face i lies at x_{i-1/2}; halo indices 1-H..0 and N+1..N+H.  Element (i,j,k) of
// any field lives at ((k-1+Hz)*(Ny+2Hy) + (j-1+Hy))*(Nx+2Hx) + (i-1+Hx).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <string>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { PERIODIC = 0, BOUNDED = 1, FLAT = 2 };
enum { ADV_NONE = 0, ADV_UPWIND1 = 1, ADV_CENTERED2 = 2, ADV_WENO5 = 5, ADV_WENO7 = 7, ADV_WENO9 = 9 };
enum { CENTER = 0, FACE = 1 };
constexpr int MAX_TRACERS = 8;

// ---------------------------------------------------------------------------------------
// Grid and metrics.  PAPER.md:940-947 (listing 15: faces given, centres are midpoints),
// PAPER.md:990-994 (volumes V and face areas Ax, Ay, Az of (B2)).  Only z may be stretched.
// ---------------------------------------------------------------------------------------
struct Grid {
  int Nx, Ny, Nz, H;
  int Hx, Hy, Hz;            // 0 on a Flat axis, else H
  int topo[3];
  double dx, dy;
  // z metrics, indexed k = 1-Hz .. Nz+Hz+1 through zi(k)
  std::vector<double> dzc;   // cell thickness  Δz_c[k]           (k = 1-Hz .. Nz+Hz)
  std::vector<double> dzf;   // centre spacing  Δz_f[k] = z_c[k]-z_c[k-1]
  std::vector<double> zc;    // centre height   z_c[k]
  std::vector<double> zf;    // face height     z_f[k]  (z_f[Nz+1] = 0 is the surface)
  long nxp, nyp, nzp;
  int zi(int k) const { return k - 1 + Hz + 1; }  // +1 slack so k-1 is always addressable
  long idx(int i, int j, int k) const {
    return ((long)(k - 1 + Hz) * nyp + (j - 1 + Hy)) * nxp + (i - 1 + Hx);
  }
  long nelem() const { return nxp * nyp * nzp; }
};

struct Params {
  int n_tracers, idx_T, idx_S;
  int adv[3];
  int momentum_prognostic;
  int hydrostatic;
  double weno_eps;
  double f0, beta_coriolis, y0;
  double g, alpha_T, beta_S;
  std::vector<double> T_ref, S_ref;   // Nz values each (empty = 0)
  double nu, kappa[MAX_TRACERS];
  int vimplicit = 0;   // N3 (A1) PAPER.md:785-789: vertical diffusion treated implicitly is NOT part of G
};

Grid *make_grid(int Nx, int Ny, int Nz, int H, double dx, double dy, const double *dz_c,
                double dz_uniform, const int topo[3]) {
  Grid *g = new Grid;
  g->Nx = Nx; g->Ny = Ny; g->Nz = Nz; g->H = H;
  for (int a = 0; a < 3; ++a) g->topo[a] = topo[a];
  g->Hx = topo[0] == FLAT ? 0 : H;
  g->Hy = topo[1] == FLAT ? 0 : H;
  g->Hz = topo[2] == FLAT ? 0 : H;
  g->dx = dx; g->dy = dy;
  g->nxp = Nx + 2 * g->Hx; g->nyp = Ny + 2 * g->Hy; g->nzp = Nz + 2 * g->Hz;
  const int Hz = g->Hz;
  const int n = Nz + 2 * Hz + 3;
  g->dzc.assign(n, 0.0); g->dzf.assign(n, 0.0); g->zc.assign(n, 0.0); g->zf.assign(n, 0.0);
  // interior thicknesses, bottom -> top
  for (int k = 1; k <= Nz; ++k) g->dzc[g->zi(k)] = dz_c ? dz_c[k - 1] : dz_uniform;
  // halo thicknesses: mirror on Bounded, wrap on Periodic; they only ever
  // multiply zero fluxes or periodic copies.
  for (int m = 1; m <= Hz; ++m) {
    if (topo[2] == PERIODIC) {
      g->dzc[g->zi(1 - m)] = g->dzc[g->zi(Nz + 1 - m)];
      g->dzc[g->zi(Nz + m)] = g->dzc[g->zi(m)];
    } else {
      g->dzc[g->zi(1 - m)] = g->dzc[g->zi(m)];
      g->dzc[g->zi(Nz + m)] = g->dzc[g->zi(Nz + 1 - m)];
    }
  }
  // faces: z_f[Nz+1] = 0 (surface), z_f[k] = z_f[k+1] - Δz_c[k]; summed in long double so
  // the metrics are the same numbers whatever E is.
  long double depth = 0;
  for (int k = 1; k <= Nz; ++k) depth += (long double)g->dzc[g->zi(k)];
  std::vector<long double> zf(n, 0.0L);
  zf[g->zi(1)] = -depth;
  for (int k = 1; k <= Nz + Hz; ++k) zf[g->zi(k + 1)] = zf[g->zi(k)] + (long double)g->dzc[g->zi(k)];
  for (int k = 0; k >= 1 - Hz; --k) zf[g->zi(k)] = zf[g->zi(k + 1)] - (long double)g->dzc[g->zi(k)];
  zf[g->zi(Nz + 1)] = 0.0L;  // exactly the surface
  for (int k = Nz + 1; k <= Nz + Hz; ++k) zf[g->zi(k + 1)] = zf[g->zi(k)] + (long double)g->dzc[g->zi(k)];
  for (int k = 1 - Hz; k <= Nz + Hz + 1; ++k) g->zf[g->zi(k)] = (double)zf[g->zi(k)];
  for (int k = 1 - Hz; k <= Nz + Hz; ++k) {
    long double c = 0.5L * (zf[g->zi(k)] + zf[g->zi(k + 1)]);   // listing 15: midpoint
    g->zc[g->zi(k)] = (double)c;
  }
  for (int k = 2 - Hz; k <= Nz + Hz; ++k) {
    long double cm = 0.5L * (zf[g->zi(k - 1)] + zf[g->zi(k)]);
    long double cp = 0.5L * (zf[g->zi(k)] + zf[g->zi(k + 1)]);
    g->dzf[g->zi(k)] = (double)(cp - cm);
  }
  // spacing across the outermost stored face (only ever multiplies mirrored zero gradients)
  if (Hz > 0) {
    g->dzf[g->zi(1 - Hz)] = g->dzc[g->zi(1 - Hz)];
    g->dzf[g->zi(Nz + Hz + 1)] = g->dzc[g->zi(Nz + Hz)];
  } else {
    g->dzf[g->zi(1)] = g->dzc[g->zi(1)];
    g->dzf[g->zi(2)] = g->dzc[g->zi(1)];
  }
  return g;
}

// ---------------------------------------------------------------------------------------
// One-dimensional building blocks.  `q(m)` is a 1-D sequence; the target
// point lies midway between q(m-1) and q(m).
// ---------------------------------------------------------------------------------------

// (B4) PAPER.md:1007  Centered(order=2): <c>_i = (c_i + c_{i-1})/2
template <class E, class Q> E C2(Q q, int m) { return (q(m - 1) + q(m)) / E(2); }

// Centered(order=4): the symmetric part of UpwindBiased(order=3) (B5)/(B7)
template <class E, class Q> E C4(Q q, int m) {
  return (-q(m - 2) + E(7) * q(m - 1) + E(7) * q(m) - q(m + 1)) / E(12);
}

// (B5) PAPER.md:1013  UpwindBiased(order=3), u>0 and u<0 branches
template <class E, class Q> E U3L(Q q, int m) { return (-q(m - 2) + E(5) * q(m - 1) + E(2) * q(m)) / E(6); }
template <class E, class Q> E U3R(Q q, int m) { return (E(2) * q(m - 1) + E(5) * q(m) - q(m + 1)) / E(6); }

// WENO5 with WENO-Z weights from five values (a,b,c,d,e), biased towards a.
// Candidates: (B9) PAPER.md:1039; convex combination: (B8) PAPER.md:1034; weights: WENO-Z
// with the classical 5th-order smoothness indicators and ideal weights
// (1/10, 6/10, 3/10) — DESIGN.md readings R1, R2 (not printed in the paper).
template <class E> E weno5z(E a, E b, E c, E d, E e, E eps) {
  const E p_p1 = (E(2) * a - E(7) * b + E(11) * c) / E(6);   // s = +1  [c]^{3,1}
  const E p_0 = (-b + E(5) * c + E(2) * d) / E(6);           // s =  0  [c]^{3,0}
  const E p_m1 = (E(2) * c + E(5) * d - e) / E(6);           // s = -1  [c]^{3,-1}
  const E t1 = a - E(2) * b + c, u1 = a - E(4) * b + E(3) * c;
  const E t0 = b - E(2) * c + d, u0 = b - d;
  const E tm = c - E(2) * d + e, um = E(3) * c - E(4) * d + e;
  const E b_p1 = E(13) / E(12) * t1 * t1 + E(1) / E(4) * u1 * u1;
  const E b_0 = E(13) / E(12) * t0 * t0 + E(1) / E(4) * u0 * u0;
  const E b_m1 = E(13) / E(12) * tm * tm + E(1) / E(4) * um * um;
  const E tau5 = std::fabs(b_p1 - b_m1);
  const E r1 = tau5 / (b_p1 + eps), r0 = tau5 / (b_0 + eps), rm = tau5 / (b_m1 + eps);
  const E a_p1 = E(1) / E(10) * (E(1) + r1 * r1);
  const E a_0 = E(6) / E(10) * (E(1) + r0 * r0);
  const E a_m1 = E(3) / E(10) * (E(1) + rm * rm);
  const E s = a_p1 + a_0 + a_m1;
  return (a_p1 / s) * p_p1 + (a_0 / s) * p_0 + (a_m1 / s) * p_m1;
}

// left-biased (flow in +direction) and right-biased (mirror image, reading R3)
template <class E, class Q> E W5L(Q q, int m, E eps) { return weno5z<E>(q(m - 3), q(m - 2), q(m - 1), q(m), q(m + 1), eps); }
template <class E, class Q> E W5R(Q q, int m, E eps) { return weno5z<E>(q(m + 2), q(m + 1), q(m), q(m - 1), q(m - 2), eps); }

// ---- WENO(2r-1)-Z for r = 3, 4, 5 from the DEFINITION ("orders up to 11",
// PAPER.md:1030-1042 (B8)/(B9), WENO-Z PAPER.md:1042; readings R1, R2, R20).  Tables: oracle/weno_tables.inc, exact
// rationals written by oracle/gen_weno_tables.py (candidate polynomials matching cell averages, Jiang-Shu
// smoothness integrals, ideal weights, tau combinations).
#define Q(n, d) ((long double)(n) / (long double)(d))
#include "weno_tables.inc"
#undef Q
struct WenoTab { int r; const long double *ainv, *imat, *d, *tau; };
inline WenoTab weno_tab(int r) {
  if (r == 3) return {3, &WENO5_AINV[0][0][0], &WENO5_IMAT[0][0], WENO5_D, WENO5_TAU};
  if (r == 4) return {4, &WENO7_AINV[0][0][0], &WENO7_IMAT[0][0], WENO7_D, WENO7_TAU};
  return {5, &WENO9_AINV[0][0][0], &WENO9_IMAT[0][0], WENO9_D, WENO9_TAU};
}
// v[0..2r-2]: the 2r-1 cell values, v[0] the most upwind one, v[r-1] the upwind cell of the face (cell 0 of the
// generator).  Step by step: (1) for each candidate stencil k the monomial coefficients a_n of the polynomial p_k
// whose cell averages are the data — taken of the data MINUS v[r-1] (p_k of shifted data is p_k minus the shift;
// the derivatives do not see it), which keeps the arithmetic free of the field's mean; (2) p_k(1/2);
// (3) beta_k = sum_l int (d^l p_k)^2; (4) tau = |sum_k TAU_k beta_k|; (5) alpha_k = d_k (1 + (tau/(beta_k+eps))^2);
// (6) the convex combination (B8).
template <class E> E wenoz_general(int r, const E *v, E eps) {
  const WenoTab t = weno_tab(r);
  const E vc = v[r - 1];
  E p[5], beta[5];
  for (int k = 0; k < r; ++k) {
    E a[5];
    for (int n = 0; n < r; ++n) {
      E s = E(0);
      for (int jj = 0; jj < r; ++jj) s += (E)t.ainv[(k * r + n) * r + jj] * (v[k + jj] - vc);
      a[n] = s;
    }
    E val = E(0), half = E(1);
    for (int n = 0; n < r; ++n) { val += a[n] * half; half /= E(2); }
    p[k] = vc + val;
    E b = E(0);
    for (int n = 1; n < r; ++n)
      for (int m = 1; m < r; ++m) b += (E)t.imat[n * r + m] * a[n] * a[m];
    beta[k] = b;
  }
  E tau = E(0);
  for (int k = 0; k < r; ++k) tau += (E)t.tau[k] * beta[k];
  tau = std::fabs(tau);
  E alpha[5], sum = E(0);
  for (int k = 0; k < r; ++k) {
    const E q = tau / (beta[k] + eps);
    alpha[k] = (E)t.d[k] * (E(1) + q * q);
    sum += alpha[k];
  }
  E out = E(0);
  for (int k = 0; k < r; ++k) out += (alpha[k] / sum) * p[k];
  return out;
}
// left-biased: cells m-r .. m+r-2 (upwind cell m-1); right-biased: the mirror image m+r-1 .. m-r+1 (reading R3)
template <class E, class Q_> E WGL(int r, Q_ q, int m, E eps) {
  E v[9];
  for (int t = 0; t < 2 * r - 1; ++t) v[t] = q(m - r + t);
  return wenoz_general<E>(r, v, eps);
}
template <class E, class Q_> E WGR(int r, Q_ q, int m, E eps) {
  E v[9];
  for (int t = 0; t < 2 * r - 1; ++t) v[t] = q(m + r - 1 - t);
  return wenoz_general<E>(r, v, eps);
}
// Centered(6), Centered(8): symmetric part of UpwindBiased(5), UpwindBiased(7) (reading R4); q[m-n/2] .. q[m+n/2-1]
template <class E, class Q_> E CN(int order, Q_ q, int m) {
  const long double *w = order == 4 ? CENTERED4_W : (order == 6 ? CENTERED6_W : CENTERED8_W);
  E s = E(0);
  for (int t = 0; t < order; ++t) s += (E)w[t] * q(m - order / 2 + t);
  return s;
}

// Upwinded product  a~ * reconstruct(q; m)   (B5) PAPER.md:1013-1016 ("= 0 if u = 0")
template <class E, class Q> E UP(int scheme, E a, Q q, int m, E eps) {
  switch (scheme) {
    case ADV_CENTERED2: return a * C2<E>(q, m);
    case ADV_UPWIND1: return a * (a > E(0) ? q(m - 1) : q(m));
    case ADV_WENO5: return a * (a > E(0) ? W5L<E>(q, m, eps) : W5R<E>(q, m, eps));
    case ADV_WENO7: return a * (a > E(0) ? WGL<E>(4, q, m, eps) : WGR<E>(4, q, m, eps));
    case ADV_WENO9: return a * (a > E(0) ? WGL<E>(5, q, m, eps) : WGR<E>(5, q, m, eps));
    default: return E(0);
  }
}

// "high-order Centered" advecting-velocity interpolation, PAPER.md:1074 (B21), reading R4:
// Centered(N-1) where the flux direction uses WENO(N) (4, 6, 8 for N = 5, 7, 9), Centered(2) otherwise.
template <class E, class Q> E IX(int scheme, Q q, int m) {
  if (scheme == ADV_WENO5) return C4<E>(q, m);
  if (scheme == ADV_WENO7) return CN<E>(6, q, m);
  if (scheme == ADV_WENO9) return CN<E>(8, q, m);
  return C2<E>(q, m);
}

// ---------------------------------------------------------------------------------------
// The model: all operators over padded arrays of storage type S, evaluated in E.
// ---------------------------------------------------------------------------------------
template <class S, class E> struct Model {
  const Grid &g;
  const Params &p;
  const S *u, *v, *w;
  const S *c[MAX_TRACERS];
  const S *phy;
  Model(const Grid &g_, const Params &p_) : g(g_), p(p_), u(nullptr), v(nullptr), w(nullptr), phy(nullptr) {
    for (auto &x : c) x = nullptr;
  }
  E at(const S *q, int i, int j, int k) const { return (E)q[g.idx(i, j, k)]; }
  E dzc(int k) const { return (E)g.dzc[g.zi(k)]; }
  E dzf(int k) const { return (E)g.dzf[g.zi(k)]; }
  bool hasx() const { return g.topo[0] != FLAT; }
  bool hasy() const { return g.topo[1] != FLAT; }
  bool hasz() const { return g.topo[2] != FLAT; }
  E eps() const { return (E)p.weno_eps; }

  // linear equation of state, reading R9 (PAPER.md:300 b = -g rho'/rho0)
  E buoyancy(int i, int j, int k) const {
    // reference profiles are indexed by interior level; halo levels mirror (Bounded z)
    int kk = k < 1 ? 1 - k : (k > g.Nz ? 2 * g.Nz + 1 - k : k);
    if (g.topo[2] == PERIODIC) kk = ((k - 1) % g.Nz + g.Nz) % g.Nz + 1;
    const E Tr = p.T_ref.empty() ? E(0) : (E)p.T_ref[kk - 1];
    const E Sr = p.S_ref.empty() ? E(0) : (E)p.S_ref[kk - 1];
    const E T = p.idx_T >= 0 ? at(c[p.idx_T], i, j, k) - Tr : E(0);
    const E Sa = p.idx_S >= 0 ? at(c[p.idx_S], i, j, k) - Sr : E(0);
    return (E)p.g * ((E)p.alpha_T * T - (E)p.beta_S * Sa);
  }

  // 7-point Laplacian in flux-divergence form (B2) with J = -coef * grad q: PAPER.md:340 (eq 8,
  // first row), PAPER.md:983 (δ²x), PAPER.md:990-994 (B2).  zloc = CENTER for fields centred in
  // z (c, u, v), FACE for w.
  E laplacian(const S *q, int i, int j, int k, int zloc) const {
    const E dx = (E)g.dx, dy = (E)g.dy;
    const E dzv = zloc == CENTER ? dzc(k) : dzf(k);     // thickness of this control volume
    const E V = dx * dy * dzv, Ax = dy * dzv, Ay = dx * dzv, Az = dx * dy;
    E s = E(0);
    if (hasx()) s += Ax * (at(q, i + 1, j, k) - at(q, i, j, k)) / dx - Ax * (at(q, i, j, k) - at(q, i - 1, j, k)) / dx;
    if (hasy()) s += Ay * (at(q, i, j + 1, k) - at(q, i, j, k)) / dy - Ay * (at(q, i, j, k) - at(q, i, j - 1, k)) / dy;
    if (hasz() && !p.vimplicit) {   // (A1): "vertical diffusion treated with an ExplicitTimeDiscretization is absorbed into G"
      // spacing between this point and its upper / lower neighbour
      const E dup = zloc == CENTER ? dzf(k + 1) : dzc(k);
      const E ddn = zloc == CENTER ? dzf(k) : dzc(k - 1);
      s += Az * (at(q, i, j, k + 1) - at(q, i, j, k)) / dup - Az * (at(q, i, j, k) - at(q, i, j, k - 1)) / ddn;
    }
    return s / V;
  }

  // ---- tracer tendency at ccc: (B3) PAPER.md:996-1003 + diffusion; SURVEY c.4 ----
  E G_tracer(int n, int i, int j, int k) const {
    const S *cc = c[n];
    const E dx = (E)g.dx, dy = (E)g.dy, dz = dzc(k);
    const E V = dx * dy * dz, Ax = dy * dz, Ay = dx * dz, Az = dx * dy;
    E div = E(0);
    if (hasx() && u) {
      auto cx = [&](int m) { return at(cc, m, j, k); };
      const E Fl = UP<E>(p.adv[0], at(u, i, j, k), cx, i, eps());          // at fcc, face i
      const E Fh = UP<E>(p.adv[0], at(u, i + 1, j, k), cx, i + 1, eps());  // face i+1
      div += Ax * Fh - Ax * Fl;
    }
    if (hasy() && v) {
      auto cy = [&](int m) { return at(cc, i, m, k); };
      const E Fl = UP<E>(p.adv[1], at(v, i, j, k), cy, j, eps());
      const E Fh = UP<E>(p.adv[1], at(v, i, j + 1, k), cy, j + 1, eps());
      div += Ay * Fh - Ay * Fl;
    }
    if (hasz() && w) {
      auto cz = [&](int m) { return at(cc, i, j, m); };
      const E Fl = UP<E>(p.adv[2], at(w, i, j, k), cz, k, eps());
      const E Fh = UP<E>(p.adv[2], at(w, i, j, k + 1), cz, k + 1, eps());
      div += Az * Fh - Az * Fl;
    }
    return -div / V + (E)p.kappa[n] * laplacian(cc, i, j, k, CENTER);
  }

  // ---- u tendency at fcc: eq (6)/(17) PAPER.md:318,506; flux form (7)/(18); (B21) ----
  E G_u(int i, int j, int k) const {
    const E dx = (E)g.dx, dy = (E)g.dy, dz = dzc(k);
    const E V = dx * dy * dz, Ax = dy * dz, Ay = dx * dz, Az = dx * dy;
    E div = E(0);
    if (hasx()) {
      auto ux = [&](int m) { return at(u, m, j, k); };
      auto Axu = [&](int m) { return Ax * at(u, m, j, k); };
      // x-faces of the u control volume are the cell centres i-1 and i
      const E Fh = UP<E>(p.adv[0], IX<E>(p.adv[0], Axu, i + 1), ux, i + 1, eps());  // centre i
      const E Fl = UP<E>(p.adv[0], IX<E>(p.adv[0], Axu, i), ux, i, eps());          // centre i-1
      div += Fh - Fl;
    }
    if (hasy() && v) {
      auto uy = [&](int m) { return at(u, i, m, k); };
      auto Ayv_h = [&](int m) { return Ay * at(v, m, j + 1, k); };   // v along x at y-face j+1
      auto Ayv_l = [&](int m) { return Ay * at(v, m, j, k); };       // v along x at y-face j
      const E Fh = UP<E>(p.adv[1], IX<E>(p.adv[1], Ayv_h, i), uy, j + 1, eps());   // at ffc (i, j+1)
      const E Fl = UP<E>(p.adv[1], IX<E>(p.adv[1], Ayv_l, i), uy, j, eps());       // at ffc (i, j)
      div += Fh - Fl;
    }
    if (hasz() && w) {
      auto uz = [&](int m) { return at(u, i, j, m); };
      auto Azw_h = [&](int m) { return Az * at(w, m, j, k + 1); };
      auto Azw_l = [&](int m) { return Az * at(w, m, j, k); };
      const E Fh = UP<E>(p.adv[2], IX<E>(p.adv[2], Azw_h, i), uz, k + 1, eps());   // at fcf (i, k+1)
      const E Fl = UP<E>(p.adv[2], IX<E>(p.adv[2], Azw_l, i), uz, k, eps());
      div += Fh - Fl;
    }
    E G = -div / V;
    // Coriolis -f x u, reading R8: 4-point average of v to fcc, f at this point's own y
    if (v && (p.f0 != 0.0 || p.beta_coriolis != 0.0)) {
      const E yc = (E(j) - E(1) / E(2)) * dy;
      const E f = (E)p.f0 + (E)p.beta_coriolis * (yc - (E)p.y0);
      G += f * (at(v, i - 1, j, k) + at(v, i, j, k) + at(v, i - 1, j + 1, k) + at(v, i, j + 1, k)) / E(4);
    }
    G += (E)p.nu * laplacian(u, i, j, k, CENTER);
    // hydrostatic pressure gradient -∂x p_hy, eq (17), (A6) PAPER.md:817-822
    if (p.hydrostatic && phy) G -= (at(phy, i, j, k) - at(phy, i - 1, j, k)) / dx;
    return G;
  }

  // ---- v tendency at cfc (mirror of u with x <-> y) ----
  E G_v(int i, int j, int k) const {
    const E dx = (E)g.dx, dy = (E)g.dy, dz = dzc(k);
    const E V = dx * dy * dz, Ax = dy * dz, Ay = dx * dz, Az = dx * dy;
    E div = E(0);
    if (hasx() && u) {
      auto vx = [&](int m) { return at(v, m, j, k); };
      auto Axu_h = [&](int m) { return Ax * at(u, i + 1, m, k); };   // u along y at x-face i+1
      auto Axu_l = [&](int m) { return Ax * at(u, i, m, k); };
      const E Fh = UP<E>(p.adv[0], IX<E>(p.adv[0], Axu_h, j), vx, i + 1, eps());   // at ffc (i+1, j)
      const E Fl = UP<E>(p.adv[0], IX<E>(p.adv[0], Axu_l, j), vx, i, eps());
      div += Fh - Fl;
    }
    if (hasy()) {
      auto vy = [&](int m) { return at(v, i, m, k); };
      auto Ayv = [&](int m) { return Ay * at(v, i, m, k); };
      const E Fh = UP<E>(p.adv[1], IX<E>(p.adv[1], Ayv, j + 1), vy, j + 1, eps());  // centre j
      const E Fl = UP<E>(p.adv[1], IX<E>(p.adv[1], Ayv, j), vy, j, eps());          // centre j-1
      div += Fh - Fl;
    }
    if (hasz() && w) {
      auto vz = [&](int m) { return at(v, i, j, m); };
      auto Azw_h = [&](int m) { return Az * at(w, i, m, k + 1); };
      auto Azw_l = [&](int m) { return Az * at(w, i, m, k); };
      const E Fh = UP<E>(p.adv[2], IX<E>(p.adv[2], Azw_h, j), vz, k + 1, eps());   // at cff (j, k+1)
      const E Fl = UP<E>(p.adv[2], IX<E>(p.adv[2], Azw_l, j), vz, k, eps());
      div += Fh - Fl;
    }
    E G = -div / V;
    if (u && (p.f0 != 0.0 || p.beta_coriolis != 0.0)) {
      const E yf = (E(j) - E(1)) * dy;
      const E f = (E)p.f0 + (E)p.beta_coriolis * (yf - (E)p.y0);
      G -= f * (at(u, i, j - 1, k) + at(u, i + 1, j - 1, k) + at(u, i, j, k) + at(u, i + 1, j, k)) / E(4);
    }
    G += (E)p.nu * laplacian(v, i, j, k, CENTER);
    if (p.hydrostatic && phy) G -= (at(phy, i, j, k) - at(phy, i, j - 1, k)) / dy;
    return G;
  }

  // ---- w tendency at ccf (nonhydrostatic only); control volume thickness Δz_f[k] ----
  E G_w(int i, int j, int k) const {
    const E dx = (E)g.dx, dy = (E)g.dy, dz = dzf(k);
    const E V = dx * dy * dz, Az = dx * dy;
    E div = E(0);
    if (hasx()) {
      auto wx = [&](int m) { return at(w, m, j, k); };
      // advecting u at fcf: interpolate the area flux Ax*u in z (Ax = Δy Δz_c[k'])
      auto Axu_h = [&](int m) { return dy * dzc(m) * at(u, i + 1, j, m); };
      auto Axu_l = [&](int m) { return dy * dzc(m) * at(u, i, j, m); };
      const E Fh = UP<E>(p.adv[0], IX<E>(p.adv[0], Axu_h, k), wx, i + 1, eps());
      const E Fl = UP<E>(p.adv[0], IX<E>(p.adv[0], Axu_l, k), wx, i, eps());
      div += Fh - Fl;
    }
    if (hasy()) {
      auto wy = [&](int m) { return at(w, i, m, k); };
      auto Ayv_h = [&](int m) { return dx * dzc(m) * at(v, i, j + 1, m); };
      auto Ayv_l = [&](int m) { return dx * dzc(m) * at(v, i, j, m); };
      const E Fh = UP<E>(p.adv[1], IX<E>(p.adv[1], Ayv_h, k), wy, j + 1, eps());
      const E Fl = UP<E>(p.adv[1], IX<E>(p.adv[1], Ayv_l, k), wy, j, eps());
      div += Fh - Fl;
    }
    {
      auto wz = [&](int m) { return at(w, i, j, m); };
      auto Azw = [&](int m) { return Az * at(w, i, j, m); };
      // z-faces of the w control volume are the cell centres k-1 and k
      const E Fh = UP<E>(p.adv[2], IX<E>(p.adv[2], Azw, k + 1), wz, k + 1, eps());  // centre k
      const E Fl = UP<E>(p.adv[2], IX<E>(p.adv[2], Azw, k), wz, k, eps());          // centre k-1
      div += Fh - Fl;
    }
    E G = -div / V;
    // buoyancy  -b g^ with g^ = -z^ (eq 6), reading R10: interpolated to ccf
    if (p.idx_T >= 0 || p.idx_S >= 0) G += (buoyancy(i, j, k - 1) + buoyancy(i, j, k)) / E(2);
    G += (E)p.nu * laplacian(w, i, j, k, FACE);
    return G;
  }
};

// ---------------------------------------------------------------------------------------
// Halo fill (a1): PAPER.md:1078 ("halo cells are updated before the computation of
// tendencies"), default no-flux / impenetrable walls PAPER.md:349-353, readings R5, R6.
// x, then y over the x-filled range, then z over the xy-filled range => edges and corners.
// ---------------------------------------------------------------------------------------
template <class S> void fill_halos_field(const Grid &g, S *q, const int loc[3]) {
  const int N[3] = {g.Nx, g.Ny, g.Nz};
  const int Hh[3] = {g.Hx, g.Hy, g.Hz};
  for (int ax = 0; ax < 3; ++ax) {
    const int H = Hh[ax], Na = N[ax], topo = g.topo[ax];
    if (topo == FLAT || H == 0) continue;
    // sweep the full padded range of the two other axes: rows whose other-axis halos are not
    // filled yet are overwritten by the later passes, so the final result is the same as
    // mapping each coordinate independently (edges and corners included).
    int lo[3], hi[3];
    for (int b = 0; b < 3; ++b) { lo[b] = 1 - Hh[b]; hi[b] = N[b] + Hh[b]; }
    auto at = [&](int a, int b1, int b2) -> S & {
      int ijk[3];
      ijk[ax] = a; ijk[(ax + 1) % 3] = b1; ijk[(ax + 2) % 3] = b2;
      return q[g.idx(ijk[0], ijk[1], ijk[2])];
    };
    const int B1 = (ax + 1) % 3, B2 = (ax + 2) % 3;
    for (int b2 = lo[B2]; b2 <= hi[B2]; ++b2)
      for (int b1 = lo[B1]; b1 <= hi[B1]; ++b1) {
        if (topo == PERIODIC) {
          for (int m = 1; m <= H; ++m) { at(1 - m, b1, b2) = at(Na + 1 - m, b1, b2); at(Na + m, b1, b2) = at(m, b1, b2); }
        } else if (loc[ax] == CENTER) {   // Bounded, centre-located: even mirror (no-flux)
          for (int m = 1; m <= H; ++m) { at(1 - m, b1, b2) = at(m, b1, b2); at(Na + m, b1, b2) = at(Na + 1 - m, b1, b2); }
        } else {                          // Bounded, wall-normal velocity: walls and beyond = 0
          at(1, b1, b2) = S(0);
          for (int m = 1; m <= H; ++m) { at(1 - m, b1, b2) = S(0); at(Na + m, b1, b2) = S(0); }
        }
      }
  }
}

// (15) PAPER.md:456-458: w from continuity, column integration from the bottom; R11: w_top kept.
template <class S, class E> void compute_w(const Grid &g, const S *u, const S *v, S *w) {
  const E dx = (E)g.dx, dy = (E)g.dy;
  const bool hx = g.topo[0] != FLAT, hy = g.topo[1] != FLAT;
  const int ihi = hx ? g.Nx + g.Hx - 1 : g.Nx, jhi = hy ? g.Ny + g.Hy - 1 : g.Ny;
#pragma omp parallel for schedule(static)
  for (int j = 1 - g.Hy; j <= jhi; ++j)
    for (int i = 1 - g.Hx; i <= ihi; ++i) {
      E wk = E(0);
      w[g.idx(i, j, 1)] = S(0);
      for (int k = 1; k <= g.Nz; ++k) {
        E d = E(0);
        if (hx) d += ((E)u[g.idx(i + 1, j, k)] - (E)u[g.idx(i, j, k)]) / dx;
        if (hy) d += ((E)v[g.idx(i, j + 1, k)] - (E)v[g.idx(i, j, k)]) / dy;
        wk = wk - (E)g.dzc[g.zi(k)] * d;
        w[g.idx(i, j, k + 1)] = (S)wk;
        wk = (E)(S)wk;   // the stored value is what the next level integrates from
      }
    }
}

// (14) PAPER.md:452-454, (A6) PAPER.md:817-822: ∂z p_hy = b, p(z=0) = 0, integrated downward.
template <class S, class E> void compute_phy(const Grid &g, const Params &p, const S *T, const S *Sa, S *phy) {
  Model<S, E> m(g, p);
  if (p.idx_T >= 0) m.c[p.idx_T] = T;
  if (p.idx_S >= 0) m.c[p.idx_S] = Sa;
#pragma omp parallel for schedule(static)
  for (int j = 1 - g.Hy; j <= g.Ny + g.Hy; ++j)
    for (int i = 1 - g.Hx; i <= g.Nx + g.Hx; ++i) {
      E pk = -m.buoyancy(i, j, g.Nz) * m.dzc(g.Nz) / E(2);
      phy[g.idx(i, j, g.Nz)] = (S)pk;
      for (int k = g.Nz; k >= 2; --k) {
        pk = (E)(S)pk - (m.buoyancy(i, j, k) + m.buoyancy(i, j, k - 1)) / E(2) * m.dzf(k);
        phy[g.idx(i, j, k - 1)] = (S)pk;
      }
    }
}

// first index of the prognostic range of a face-located field along an axis: wall face 1 excluded
inline int first_face(const Grid &g, int ax) { return g.topo[ax] == BOUNDED ? 2 : 1; }

template <class S, class E>
void compute_tendencies(const Grid &g, const Params &p, const S *u, const S *v, const S *w, const S *const *c,
                        const S *phy, S *Gu, S *Gv, S *Gw, S *const *Gc) {
  Model<S, E> m(g, p);
  m.u = u; m.v = v; m.w = w; m.phy = phy;
  for (int n = 0; n < p.n_tracers; ++n) m.c[n] = c[n];
#pragma omp parallel for collapse(2) schedule(static)
  for (int k = 1; k <= g.Nz; ++k)
    for (int j = 1; j <= g.Ny; ++j)
      for (int i = 1; i <= g.Nx; ++i) {
        const long id = g.idx(i, j, k);
        for (int n = 0; n < p.n_tracers; ++n) Gc[n][id] = (S)m.G_tracer(n, i, j, k);
        if (p.momentum_prognostic) {
          if (Gu) Gu[id] = i >= first_face(g, 0) ? (S)m.G_u(i, j, k) : S(0);   // wall faces: G = 0
          if (Gv) Gv[id] = j >= first_face(g, 1) ? (S)m.G_v(i, j, k) : S(0);
          if (Gw && !p.hydrostatic && g.topo[2] != FLAT) Gw[id] = k >= first_face(g, 2) ? (S)m.G_w(i, j, k) : S(0);
        }
      }
}

// tendencies at a list of sample points (for parity at full benchmark sizes): out[s*nf + f],
// field order u, v, w, c0..; fields that do not exist give 0.
template <class S, class E>
void tendencies_at(const Grid &g, const Params &p, const S *u, const S *v, const S *w, const S *const *c,
                   const S *phy, long ns, const int *ijk, double *out) {
  Model<S, E> m(g, p);
  m.u = u; m.v = v; m.w = w; m.phy = phy;
  for (int n = 0; n < p.n_tracers; ++n) m.c[n] = c[n];
  const int nf = 3 + p.n_tracers;
#pragma omp parallel for schedule(static)
  for (long s = 0; s < ns; ++s) {
    const int i = ijk[3 * s], j = ijk[3 * s + 1], k = ijk[3 * s + 2];
    double *o = out + s * nf;
    o[0] = o[1] = o[2] = 0.0;
    if (p.momentum_prognostic) {
      if (u) o[0] = i >= first_face(g, 0) ? (double)(S)m.G_u(i, j, k) : 0.0;
      if (v) o[1] = j >= first_face(g, 1) ? (double)(S)m.G_v(i, j, k) : 0.0;
      if (w && !p.hydrostatic && g.topo[2] != FLAT) o[2] = k >= first_face(g, 2) ? (double)(S)m.G_w(i, j, k) : 0.0;
    }
    for (int n = 0; n < p.n_tracers; ++n) o[3 + n] = (double)(S)m.G_tracer(n, i, j, k);
  }
}

// (A4) PAPER.md:797-801: q <- q + Δt (γ G^m - ζ G^{m-1}) on interior non-wall points (reading R14)
template <class S, class E>
void substage_field(const Grid &g, S *q, const S *G, const S *Gp, E gamma, E zeta, E dt, const int loc[3]) {
  const int i0 = loc[0] == FACE ? first_face(g, 0) : 1;
  const int j0 = loc[1] == FACE ? first_face(g, 1) : 1;
  const int k0 = loc[2] == FACE ? first_face(g, 2) : 1;
#pragma omp parallel for collapse(2) schedule(static)
  for (int k = k0; k <= g.Nz; ++k)
    for (int j = j0; j <= g.Ny; ++j)
      for (int i = i0; i <= g.Nx; ++i) {
        const long id = g.idx(i, j, k);
        const E gp = (Gp && zeta != E(0)) ? (E)Gp[id] : E(0);
        q[id] = (S)((E)q[id] + dt * (gamma * (E)G[id] - zeta * gp));
      }
}

thread_local std::string g_err;

}  // namespace

// =========================================================================================
// C ABI.  eval: 0 = long double (parity reference), 1 = double, 2 = float.
// Arrays are double (`_f64`) or float (`_f32`) host pointers, dense padded, x fastest.
// =========================================================================================
extern "C" {

struct ocnref_params {
  int n_tracers, idx_T, idx_S;
  int adv_x, adv_y, adv_z;
  int momentum_prognostic;
  int hydrostatic;
  double weno_eps;
  double f0, beta_coriolis, y0;
  double g, alpha_T, beta_S;
  const double *T_ref, *S_ref;
  double nu, kappa[MAX_TRACERS];
  int implicit_vertical_diffusion;
};

static Params to_params(const Grid &g, const ocnref_params *pp) {
  Params p;
  p.n_tracers = pp->n_tracers; p.idx_T = pp->idx_T; p.idx_S = pp->idx_S;
  p.adv[0] = pp->adv_x; p.adv[1] = pp->adv_y; p.adv[2] = pp->adv_z;
  p.momentum_prognostic = pp->momentum_prognostic; p.hydrostatic = pp->hydrostatic;
  p.weno_eps = pp->weno_eps;
  p.f0 = pp->f0; p.beta_coriolis = pp->beta_coriolis; p.y0 = pp->y0;
  p.g = pp->g; p.alpha_T = pp->alpha_T; p.beta_S = pp->beta_S;
  if (pp->T_ref) p.T_ref.assign(pp->T_ref, pp->T_ref + g.Nz);
  if (pp->S_ref) p.S_ref.assign(pp->S_ref, pp->S_ref + g.Nz);
  p.nu = pp->nu;
  for (int n = 0; n < MAX_TRACERS; ++n) p.kappa[n] = pp->kappa[n];
  p.vimplicit = pp->implicit_vertical_diffusion ? 1 : 0;
  return p;
}

void *ocnref_grid_create(int Nx, int Ny, int Nz, int halo, double dx, double dy, const double *dz_c,
                         double dz_uniform, const int *topology) {
  return make_grid(Nx, Ny, Nz, halo, dx, dy, dz_c, dz_uniform, topology);
}
void ocnref_grid_destroy(void *g) { delete (Grid *)g; }
void ocnref_grid_dims(const void *gv, long *nxp, long *nyp, long *nzp, int *hx, int *hy, int *hz) {
  const Grid *g = (const Grid *)gv;
  *nxp = g->nxp; *nyp = g->nyp; *nzp = g->nzp; *hx = g->Hx; *hy = g->Hy; *hz = g->Hz;
}
// which: 0 = z_f (k=1..Nz+1), 1 = z_c (1..Nz), 2 = Δz_c (1..Nz), 3 = Δz_f (2..Nz)
void ocnref_grid_metric(const void *gv, int which, double *out) {
  const Grid *g = (const Grid *)gv;
  if (which == 0) for (int k = 1; k <= g->Nz + 1; ++k) out[k - 1] = g->zf[g->zi(k)];
  if (which == 1) for (int k = 1; k <= g->Nz; ++k) out[k - 1] = g->zc[g->zi(k)];
  if (which == 2) for (int k = 1; k <= g->Nz; ++k) out[k - 1] = g->dzc[g->zi(k)];
  if (which == 3) for (int k = 2; k <= g->Nz; ++k) out[k - 2] = g->dzf[g->zi(k)];
}
int ocnref_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void ocnref_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

// ---- 1-D building blocks, for the pins ----
double ocnref_weno5z(const double *q5, double eps, int eval) {
  if (eval == 0) return (double)weno5z<long double>(q5[0], q5[1], q5[2], q5[3], q5[4], eps);
  if (eval == 1) return weno5z<double>(q5[0], q5[1], q5[2], q5[3], q5[4], eps);
  return (double)weno5z<float>((float)q5[0], (float)q5[1], (float)q5[2], (float)q5[3], (float)q5[4], (float)eps);
}
// reconstruct a 1-D sequence q[0..n) at the point between q[m-1] and q[m]
// kind: 2 = C2, 4 = C4, 6 = C6, 8 = C8, 1 = U1L, -1 = U1R, 3 = U3L, -3 = U3R, 5 = W5L, -5 = W5R, +-7, +-9 = WENO7/9,
//       +-55 = WENO5 through the general routine, 44 = Centered(4) through the generated table
double ocnref_reconstruct(const double *q, int m, int kind, double eps) {
  typedef long double E;
  auto f = [&](int mm) { return (E)q[mm]; };
  switch (kind) {
    case 2: return (double)C2<E>(f, m);
    case 4: return (double)C4<E>(f, m);
    case 1: return (double)f(m - 1);
    case -1: return (double)f(m);
    case 3: return (double)U3L<E>(f, m);
    case -3: return (double)U3R<E>(f, m);
    case 5: return (double)W5L<E>(f, m, (E)eps);
    case -5: return (double)W5R<E>(f, m, (E)eps);
    case 6: return (double)CN<E>(6, f, m);
    case 8: return (double)CN<E>(8, f, m);
    case 44: return (double)CN<E>(4, f, m);            // Centered(4) through the generated table (pin vs C4)
    case 55: return (double)WGL<E>(3, f, m, (E)eps);   // WENO5 through the general routine (pin vs weno5z)
    case -55: return (double)WGR<E>(3, f, m, (E)eps);
    case 7: return (double)WGL<E>(4, f, m, (E)eps);
    case -7: return (double)WGR<E>(4, f, m, (E)eps);
    case 9: return (double)WGL<E>(5, f, m, (E)eps);
    case -9: return (double)WGR<E>(5, f, m, (E)eps);
  }
  return 0.0;
}
// upwinded product a * reconstruct(q; m) with scheme in {1,2,5}
double ocnref_upwind_flux(const double *q, int m, int scheme, double a, double eps) {
  typedef long double E;
  auto f = [&](int mm) { return (E)q[mm]; };
  return (double)UP<E>(scheme, (E)a, f, m, (E)eps);
}

#define DISPATCH_F64(CALL_LD, CALL_D) do { if (eval == 0) { CALL_LD; } else { CALL_D; } } while (0)

void ocnref_fill_halos_field_f64(const void *g, double *q, const int *loc) { fill_halos_field<double>(*(const Grid *)g, q, loc); }
void ocnref_fill_halos_field_f32(const void *g, float *q, const int *loc) { fill_halos_field<float>(*(const Grid *)g, q, loc); }

void ocnref_compute_w_f64(const void *g, const double *u, const double *v, double *w, int eval) {
  DISPATCH_F64((compute_w<double, long double>(*(const Grid *)g, u, v, w)), (compute_w<double, double>(*(const Grid *)g, u, v, w)));
}
void ocnref_compute_w_f32(const void *g, const float *u, const float *v, float *w) { compute_w<float, float>(*(const Grid *)g, u, v, w); }

void ocnref_compute_phy_f64(const void *gv, const ocnref_params *pp, const double *T, const double *S, double *phy, int eval) {
  const Grid &g = *(const Grid *)gv; Params p = to_params(g, pp);
  DISPATCH_F64((compute_phy<double, long double>(g, p, T, S, phy)), (compute_phy<double, double>(g, p, T, S, phy)));
}
void ocnref_compute_phy_f32(const void *gv, const ocnref_params *pp, const float *T, const float *S, float *phy) {
  const Grid &g = *(const Grid *)gv; Params p = to_params(g, pp);
  compute_phy<float, float>(g, p, T, S, phy);
}

void ocnref_compute_tendencies_f64(const void *gv, const ocnref_params *pp, const double *u, const double *v, const double *w,
                                   const double *const *c, const double *phy, double *Gu, double *Gv, double *Gw,
                                   double *const *Gc, int eval) {
  const Grid &g = *(const Grid *)gv; Params p = to_params(g, pp);
  DISPATCH_F64((compute_tendencies<double, long double>(g, p, u, v, w, c, phy, Gu, Gv, Gw, Gc)),
               (compute_tendencies<double, double>(g, p, u, v, w, c, phy, Gu, Gv, Gw, Gc)));
}
void ocnref_compute_tendencies_f32(const void *gv, const ocnref_params *pp, const float *u, const float *v, const float *w,
                                   const float *const *c, const float *phy, float *Gu, float *Gv, float *Gw, float *const *Gc) {
  const Grid &g = *(const Grid *)gv; Params p = to_params(g, pp);
  compute_tendencies<float, float>(g, p, u, v, w, c, phy, Gu, Gv, Gw, Gc);
}
void ocnref_tendencies_at_f64(const void *gv, const ocnref_params *pp, const double *u, const double *v, const double *w,
                              const double *const *c, const double *phy, long ns, const int *ijk, double *out, int eval) {
  const Grid &g = *(const Grid *)gv; Params p = to_params(g, pp);
  DISPATCH_F64((tendencies_at<double, long double>(g, p, u, v, w, c, phy, ns, ijk, out)),
               (tendencies_at<double, double>(g, p, u, v, w, c, phy, ns, ijk, out)));
}
void ocnref_substage_field_f64(const void *g, double *q, const double *G, const double *Gp, double gamma, double zeta,
                               double dt, const int *loc, int eval) {
  DISPATCH_F64((substage_field<double, long double>(*(const Grid *)g, q, G, Gp, gamma, zeta, dt, loc)),
               (substage_field<double, double>(*(const Grid *)g, q, G, Gp, gamma, zeta, dt, loc)));
}
void ocnref_substage_field_f32(const void *g, float *q, const float *G, const float *Gp, double gamma, double zeta,
                               double dt, const int *loc) {
  substage_field<float, float>(*(const Grid *)g, q, G, Gp, (float)gamma, (float)zeta, (float)dt, loc);
}
// (A4) constants.  Exposed so the pins test the numbers the oracle actually uses.
void ocnref_rk3_coefficients(int stage, long double *gamma, long double *zeta) {
  static const long double G[3] = {8.0L / 15.0L, 5.0L / 12.0L, 3.0L / 4.0L};
  static const long double Z[3] = {0.0L, 17.0L / 60.0L, 5.0L / 12.0L};
  *gamma = G[stage - 1]; *zeta = Z[stage - 1];
}
void ocnref_rk3_substage_field_f64(const void *g, double *q, const double *G, const double *Gp, int stage, double dt,
                                   const int *loc, int eval) {
  long double ga, ze; ocnref_rk3_coefficients(stage, &ga, &ze);
  if (eval == 0) substage_field<double, long double>(*(const Grid *)g, q, G, Gp, ga, ze, (long double)dt, loc);
  else substage_field<double, double>(*(const Grid *)g, q, G, Gp, (double)ga, (double)ze, dt, loc);
}
void ocnref_rk3_substage_field_f32(const void *g, float *q, const float *G, const float *Gp, int stage, double dt, const int *loc) {
  long double ga, ze; ocnref_rk3_coefficients(stage, &ga, &ze);
  substage_field<float, float>(*(const Grid *)g, q, G, Gp, (float)ga, (float)ze, (float)dt, loc);
}
void ocnref_rk3_coefficients_f64(int stage, double *gamma, double *zeta) {
  long double ga, ze; ocnref_rk3_coefficients(stage, &ga, &ze); *gamma = (double)ga; *zeta = (double)ze;
}

}  // extern "C"

// N2 / N3 (pressure correction, vertically-implicit diffusion): PAPER.md:785-851
#include "ocnref_solvers.inc"
