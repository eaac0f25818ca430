// barotropic.cu — SURVEY 8(f) N4: the split-explicit free surface of the HydrostaticFreeSurfaceModel, (A13)-(A21) PAPER.md:857-923.
//
//     U = sum_k dz_c u                                   column_integral_kernel      (A13)
//     F = sum_k dz_c (gamma G - zeta G_prev)             column_integral_kernel      the frozen slow term of (A19)
//     M x { eta -= dtau div U;  U -= dtau (g H grad eta_new - F);  bar += a_n (eta, U, V) }
//                                                        barotropic_substep_kernel   (A18),(A19),(A20)  one launch per substep
//     u <- u~ + (Ubar - sum_k dz_c u~) / H               barotropic_correct_kernel   (A21)
//
// Barotropic fields (eta at cc, U at fc, V at cf) are ONE horizontal plane of the grid layout: stride_z elements, element (i,j)
// at offset0 - hz*stride_z + (i-1) + (j-1)*stride_y.  Readings (R25-R27): linearised free surface on a static grid
// (eq. 16) => the column integrals run over the resting depth H = sum dz_c and g(H+eta) is g H; dtau = dt/N, M
// substeps are taken and averaged with the caller's weights; U, V are 0 and stay 0 on wall faces, Periodic axes wrap by index.
//
// Substepping is a tiny 2-D problem (C3: 864 000 columns, ~80 MB of planes, L2-resident), so it is latency- not HBM-bound: one
// fused kernel per substep computes eta_new at the three cells a (U,V) pair needs (2 redundant evaluations instead of a second
// launch and a second pass), ping-pongs the state planes and accumulates the weighted averages in the same pass.
#include <algorithm>
#include <cstdlib>

#include "ocn_internal.h"

namespace {

struct Plane2 {
  int Nx, Ny, tx, ty;
  long long sy, off;   // row pitch, offset of (1,1)
  __host__ __device__ long long idx(int i, int j) const { return off + (i - 1) + (long long)(j - 1) * sy; }
};
Plane2 make_plane(const ocn_grid *g) {
  Plane2 P;
  P.Nx = g->Nx; P.Ny = g->Ny; P.tx = g->topo[0]; P.ty = g->topo[1];
  P.sy = g->lay.stride_y; P.off = g->lay.offset0 - (long long)g->Hz * g->lay.stride_z;
  return P;
}

// out(i,j) = sum_k dz_c[k] (a A[i,j,k] - b B[i,j,k]) on the non-wall faces (0 on wall faces); blockIdx.z: 0 -> x-component, 1 -> y
template <class Real>
__global__ void __launch_bounds__(128) column_integral_kernel(const GridDev g, const Plane2 P, const Real *__restrict__ A0,
                                                              const Real *__restrict__ B0, Real *__restrict__ out0,
                                                              const Real *__restrict__ A1, const Real *__restrict__ B1,
                                                              Real *__restrict__ out1, const double a, const double b) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1, j = blockIdx.y * blockDim.y + threadIdx.y + 1, c = blockIdx.z;
  if (i > g.Nx || j > g.Ny) return;
  const Real *__restrict__ A = c ? A1 : A0;
  const Real *__restrict__ B = c ? B1 : B0;
  Real *__restrict__ out = c ? out1 : out0;
  if (!A || !out) return;
  const bool wall = c ? (P.ty == OCN_BOUNDED && j == 1) : (P.tx == OCN_BOUNDED && i == 1);
  double s = 0.0;
  if (!wall) {
    long long o = g.idx(i, j, 1);
#pragma unroll 4
    for (int k = 1; k <= g.Nz; ++k, o += g.sz) {
      // explicit roundings (no contraction choice left to the compiler): the hydrostatic TMA-ring kernel accumulates the same
      // sums while it holds G and G_prev (tend_fused.cu, a.FUo) and must reproduce them bit for bit
      double q = __dmul_rn(a, (double)A[o]);
      if (B) q = __fma_rn(-b, (double)B[o], q);
      s = __fma_rn(g.dzc[g.zi(k)], q, s);
    }
  }
  out[P.idx(i, j)] = Real(s);
}

struct BtPlanes { void *eta, *U, *V; };

template <class Real>
__global__ void __launch_bounds__(256) barotropic_substep_kernel(const Plane2 P, const BtPlanes in, const BtPlanes out, const BtPlanes acc,
                                                                 const Real *__restrict__ FU, const Real *__restrict__ FV,
                                                                 const double dtau, const double rdx, const double rdy,
                                                                 const double gH, const double an, const int first) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1, j = blockIdx.y * blockDim.y + threadIdx.y + 1;
  if (i > P.Nx || j > P.Ny) return;
  const Real *__restrict__ e = (const Real *)in.eta;
  const Real *__restrict__ U = (const Real *)in.U;
  const Real *__restrict__ V = (const Real *)in.V;
  // (A18) at an interior cell: face N+1 is face 1 (Periodic) or the wall, 0 (Bounded)
  auto eta_new = [&](int ci, int cj) -> double {
    const long long o = P.idx(ci, cj);
    const double ul = (double)U[o], uh = ci == P.Nx ? (P.tx == OCN_PERIODIC ? (double)U[P.idx(1, cj)] : 0.0) : (double)U[o + 1];
    const double vl = (double)V[o], vh = cj == P.Ny ? (P.ty == OCN_PERIODIC ? (double)V[P.idx(ci, 1)] : 0.0) : (double)V[o + P.sy];
    double div = 0.0;
    if (P.tx != OCN_FLAT) div = (uh - ul) * rdx;
    if (P.ty != OCN_FLAT) div = fma(vh - vl, rdy, div);
    return (double)Real(fma(-dtau, div, (double)e[o]));       // as stored: (A19) sees eta_new rounded to the storage type
  };
  const long long o = P.idx(i, j);
  const double ec = eta_new(i, j);
  double un = (double)U[o], vn = (double)V[o];
  if (P.tx != OCN_FLAT && !(P.tx == OCN_BOUNDED && i == 1)) {     // (A19) with the NEW eta (forward-backward)
    const double el = eta_new(i == 1 ? P.Nx : i - 1, j);
    un -= dtau * (gH * (ec - el) * rdx - (double)FU[o]);
  }
  if (P.ty != OCN_FLAT && !(P.ty == OCN_BOUNDED && j == 1)) {
    const double el = eta_new(i, j == 1 ? P.Ny : j - 1);
    vn -= dtau * (gH * (ec - el) * rdy - (double)FV[o]);
  }
  ((Real *)out.eta)[o] = Real(ec);
  ((Real *)out.U)[o] = Real(un);
  ((Real *)out.V)[o] = Real(vn);
  // (A20): the averages see the values as stored (rounded to the storage type), like the next substep does
  Real *ae = (Real *)acc.eta, *aU = (Real *)acc.U, *aV = (Real *)acc.V;
  const double e_s = (double)Real(ec), u_s = (double)Real(un), v_s = (double)Real(vn);
  ae[o] = Real(first ? an * e_s : fma(an, e_s, (double)ae[o]));
  aU[o] = Real(first ? an * u_s : fma(an, u_s, (double)aU[o]));
  aV[o] = Real(first ? an * v_s : fma(an, v_s, (double)aV[o]));
}

// S substeps per launch (temporal blocking).  A block loads a 64 x 32 region of (eta, U, V, FU, FV) into shared memory — its 56 x 24
// output cells plus S = 4 cells of halo on every side, Periodic axes wrapped by index, cells beyond a wall absent — and advances it S
// substeps in place (phase 1: eta_new from the old transports; barrier; phase 2: U, V from the new eta; barrier): after substep s the
// cells at least s away from the region's edge are exact, so the output cells are exact after S.  Same arithmetic per cell as
// barotropic_substep_kernel (double evaluation, values rounded to the storage type after every substep, the averages accumulated in the
// storage type), so the result is bit-identical; the planes are read and written once per S substeps instead of once per substep
// (C3: 97 MB of L2 traffic and one launch per substep were what a substep cost).
#ifndef OCN_BT_NT
#define OCN_BT_NT 512
#endif
constexpr int BT_S = 4, BT_RX = 64, BT_RY = 32, BT_NT = OCN_BT_NT, BT_NC = BT_RX * BT_RY / BT_NT;
struct BtWeights { double a[BT_S]; };

template <class Real>
__global__ void __launch_bounds__(BT_NT) barotropic_multistep_kernel(const Plane2 P, const BtPlanes in, const BtPlanes out, const BtPlanes acc,
                                                                   const Real *__restrict__ FU, const Real *__restrict__ FV,
                                                                   const double dtau, const double rdx, const double rdy, const double gH,
                                                                   const BtWeights w, const int ns, const int first) {
  extern __shared__ __align__(16) unsigned char bt_smem[];
  Real *se = reinterpret_cast<Real *>(bt_smem), *sU = se + BT_RX * BT_RY, *sV = sU + BT_RX * BT_RY, *sFU = sV + BT_RX * BT_RY,
       *sFV = sFU + BT_RX * BT_RY;
  const int tid = threadIdx.x;
  const int gi0 = blockIdx.x * (BT_RX - 2 * BT_S) + 1 - BT_S, gj0 = blockIdx.y * (BT_RY - 2 * BT_S) + 1 - BT_S;
  const bool perx = P.tx == OCN_PERIODIC, pery = P.ty == OCN_PERIODIC;
  int gi[BT_NC], gj[BT_NC];            // wrapped global indices of this thread's cells (0: the cell does not exist)
  long long off[BT_NC];
#pragma unroll
  for (int m = 0; m < BT_NC; ++m) {
    const int c = tid + m * BT_NT, x = c % BT_RX, y = c / BT_RX;
    int i = gi0 + x, j = gj0 + y;
    if (perx) i = i < 1 ? i + P.Nx : (i > P.Nx ? i - P.Nx : i);
    if (pery) j = j < 1 ? j + P.Ny : (j > P.Ny ? j - P.Ny : j);
    const bool ok = i >= 1 && i <= P.Nx && j >= 1 && j <= P.Ny;
    gi[m] = ok ? i : 0; gj[m] = ok ? j : 0;
    off[m] = P.idx(ok ? i : 1, ok ? j : 1);
    se[c] = ok ? ((const Real *)in.eta)[off[m]] : Real(0);
    sU[c] = ok ? ((const Real *)in.U)[off[m]] : Real(0);
    sV[c] = ok ? ((const Real *)in.V)[off[m]] : Real(0);
    sFU[c] = ok ? FU[off[m]] : Real(0);
    sFV[c] = ok ? FV[off[m]] : Real(0);
  }
  // the running weighted averages (A20) of the output cells live in registers for the S substeps
  Real ae[BT_NC], aU[BT_NC], aV[BT_NC];
  bool mine[BT_NC];
#pragma unroll
  for (int m = 0; m < BT_NC; ++m) {
    const int c = tid + m * BT_NT, x = c % BT_RX, y = c / BT_RX;
    mine[m] = x >= BT_S && x < BT_RX - BT_S && y >= BT_S && y < BT_RY - BT_S && gi0 + x <= P.Nx && gj0 + y <= P.Ny;   // unwrapped: inside the grid
    const bool ld = mine[m] && !first;
    ae[m] = ld ? ((const Real *)acc.eta)[off[m]] : Real(0);
    aU[m] = ld ? ((const Real *)acc.U)[off[m]] : Real(0);
    aV[m] = ld ? ((const Real *)acc.V)[off[m]] : Real(0);
  }
  __syncthreads();
  for (int s = 0; s < ns; ++s) {
    // ---- phase 1, (A18): eta_new = eta - dtau div(U); face N+1 is face 1 (Periodic: the wrapped neighbour) or the wall, 0 (Bounded)
    // (reads the neighbours' U, V and the cell's own eta, writes the cell's own eta: no hazard inside the phase)
#pragma unroll
    for (int m = 0; m < BT_NC; ++m) {
      const int c = tid + m * BT_NT, x = c % BT_RX, y = c / BT_RX;
      if (gi[m] && x < BT_RX - 1 && y < BT_RY - 1) {
        const double ul = (double)sU[c], uh = (gi[m] == P.Nx && !perx) ? 0.0 : (double)sU[c + 1];
        const double vl = (double)sV[c], vh = (gj[m] == P.Ny && !pery) ? 0.0 : (double)sV[c + BT_RX];
        double div = (uh - ul) * rdx;
        div = fma(vh - vl, rdy, div);
        se[c] = Real(fma(-dtau, div, (double)se[c]));
      }
    }
    __syncthreads();
    // ---- phase 2, (A19) with the NEW eta (forward-backward), (A20)
    const double an = w.a[s];
#pragma unroll
    for (int m = 0; m < BT_NC; ++m) {
      const int c = tid + m * BT_NT, x = c % BT_RX, y = c / BT_RX;
      if (gi[m] && x >= 1 && y >= 1) {
        const double ec = (double)se[c];
        double un = (double)sU[c], vn = (double)sV[c];
        if (!(P.tx == OCN_BOUNDED && gi[m] == 1)) un -= dtau * (gH * (ec - (double)se[c - 1]) * rdx - (double)sFU[c]);
        if (!(P.ty == OCN_BOUNDED && gj[m] == 1)) vn -= dtau * (gH * (ec - (double)se[c - BT_RX]) * rdy - (double)sFV[c]);
        const Real us = Real(un), vs = Real(vn);
        sU[c] = us; sV[c] = vs;
        // the averages see the values as stored (rounded to the storage type), like the next substep does
        const double e_s = (double)se[c], u_s = (double)us, v_s = (double)vs;
        const bool zero = first && s == 0;
        ae[m] = Real(zero ? an * e_s : fma(an, e_s, (double)ae[m]));
        aU[m] = Real(zero ? an * u_s : fma(an, u_s, (double)aU[m]));
        aV[m] = Real(zero ? an * v_s : fma(an, v_s, (double)aV[m]));
      }
    }
    __syncthreads();
  }
  // ---- the output cells: state after ns substeps, averages
#pragma unroll
  for (int m = 0; m < BT_NC; ++m) {
    if (mine[m]) {
      const int c = tid + m * BT_NT;
      const long long o = off[m];
      ((Real *)out.eta)[o] = se[c];
      ((Real *)out.U)[o] = sU[c];
      ((Real *)out.V)[o] = sV[c];
      ((Real *)acc.eta)[o] = ae[m];
      ((Real *)acc.U)[o] = aU[m];
      ((Real *)acc.V)[o] = aV[m];
    }
  }
}

// (A21) on the non-wall faces; blockIdx.z: 0 -> u with Ubar, 1 -> v with Vbar.  Columns of up to NZR levels are held in registers
// (every load issued before the first use, the column read once); taller columns are swept twice in batches of 8 levels.
template <class Real, int NZR>
__global__ void __launch_bounds__(128) barotropic_correct_kernel(const GridDev g, const Plane2 P, Real *__restrict__ u, Real *__restrict__ v,
                                                                 const Real *__restrict__ Ub, const Real *__restrict__ Vb, const double rH) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1, j = blockIdx.y * blockDim.y + threadIdx.y + 1, c = blockIdx.z;
  if (i > g.Nx || j > g.Ny) return;
  Real *__restrict__ q = c ? v : u;
  const Real *__restrict__ bar = c ? Vb : Ub;
  if (!q) return;
  if (c ? (P.ty == OCN_BOUNDED && j == 1) : (P.tx == OCN_BOUNDED && i == 1)) return;
  const long long o0 = g.idx(i, j, 1);
  const int Nz = g.Nz;
  const double target = (double)bar[P.idx(i, j)];
  if (NZR > 0 && Nz <= NZR) {
    Real col[NZR > 0 ? NZR : 1];
#pragma unroll
    for (int m = 0; m < NZR; ++m) col[m] = m < Nz ? q[o0 + m * g.sz] : Real(0);
    double s = 0.0;
#pragma unroll
    for (int m = 0; m < NZR; ++m)
      if (m < Nz) s = fma(g.dzc[g.zi(m + 1)], (double)col[m], s);
    const double corr = (target - s) * rH;
#pragma unroll
    for (int m = 0; m < NZR; ++m)
      if (m < Nz) q[o0 + m * g.sz] = Real((double)col[m] + corr);
    return;
  }
  constexpr int KB = 8;
  double s = 0.0;
  for (int k = 0; k < Nz; k += KB) {
    Real t[KB];
#pragma unroll
    for (int m = 0; m < KB; ++m) t[m] = k + m < Nz ? q[o0 + (k + m) * g.sz] : Real(0);
#pragma unroll
    for (int m = 0; m < KB; ++m)
      if (k + m < Nz) s = fma(g.dzc[g.zi(k + m + 1)], (double)t[m], s);
  }
  const double corr = (target - s) * rH;
  for (int k = 0; k < Nz; k += KB) {
    Real t[KB];
#pragma unroll
    for (int m = 0; m < KB; ++m) t[m] = k + m < Nz ? q[o0 + (k + m) * g.sz] : Real(0);
#pragma unroll
    for (int m = 0; m < KB; ++m)
      if (k + m < Nz) q[o0 + (k + m) * g.sz] = Real((double)t[m] + corr);
  }
}

double column_depth(const ocn_grid *g) {
  long double H = 0;
  for (int k = 1; k <= g->Nz; ++k) H += (long double)g->h_dzc[k + g->Hz];
  return (double)H;
}

int check_grid(const char *who, const ocn_grid *g) {
  if (!g) return ocn_fail(OCN_ERR_INVALID, "%s: grid is NULL", who);
  if (g->topo[2] != OCN_BOUNDED) return ocn_fail(OCN_ERR_INVALID, "%s: z must be Bounded", who);
  return OCN_OK;
}

template <class Real>
void launch_column_integral(const ocn_grid *g, const void *A0, const void *B0, void *o0, const void *A1, const void *B1, void *o1,
                            double a, double b, cudaStream_t s) {
  dim3 block(64, 2, 1), grid((g->Nx + 63) / 64, (g->Ny + 1) / 2, 2);
  column_integral_kernel<Real><<<grid, block, 0, s>>>(g->dev, make_plane(g), (const Real *)A0, (const Real *)B0, (Real *)o0,
                                                      (const Real *)A1, (const Real *)B1, (Real *)o1, a, b);
  ocn_count_launch();
}

}  // namespace

extern "C" {

int ocn_barotropic_init(const ocn_grid *g, const ocn_fields *state, ocn_barotropic *bt, void *stream) {
  int rc = check_grid("ocn_barotropic_init", g);
  if (rc) return rc;
  if (!state || !bt || !state->u || !state->v || !bt->U || !bt->V) return ocn_fail(OCN_ERR_INVALID, "ocn_barotropic_init: NULL argument");
  if (g->dtype == OCN_F64) launch_column_integral<double>(g, state->u, nullptr, bt->U, state->v, nullptr, bt->V, 1.0, 0.0, (cudaStream_t)stream);
  else launch_column_integral<float>(g, state->u, nullptr, bt->U, state->v, nullptr, bt->V, 1.0, 0.0, (cudaStream_t)stream);
  return ocn_check_cuda(cudaGetLastError(), "column_integral_kernel launch");
}

int ocn_barotropic_forcing(const ocn_grid *g, double gamma, double zeta, const ocn_fields *G, const ocn_fields *G_prev, void *FU,
                           void *FV, void *stream) {
  int rc = check_grid("ocn_barotropic_forcing", g);
  if (rc) return rc;
  if (!G || !G->u || !G->v || !FU || !FV) return ocn_fail(OCN_ERR_INVALID, "ocn_barotropic_forcing: NULL argument");
  if (G_prev && (!G_prev->u || !G_prev->v)) return ocn_fail(OCN_ERR_INVALID, "ocn_barotropic_forcing: G_prev lacks u or v");
  const void *pu = G_prev ? G_prev->u : nullptr, *pv = G_prev ? G_prev->v : nullptr;
  if (g->dtype == OCN_F64) launch_column_integral<double>(g, G->u, pu, FU, G->v, pv, FV, gamma, zeta, (cudaStream_t)stream);
  else launch_column_integral<float>(g, G->u, pu, FU, G->v, pv, FV, gamma, zeta, (cudaStream_t)stream);
  return ocn_check_cuda(cudaGetLastError(), "column_integral_kernel launch");
}

int ocn_barotropic_substeps(const ocn_grid *g, double grav, double dt, int N, int M, const double *weights, ocn_barotropic *bt,
                            const void *FU, const void *FV, void *scratch, void *stream) {
  int rc = check_grid("ocn_barotropic_substeps", g);
  if (rc) return rc;
  if (!bt || !bt->eta || !bt->U || !bt->V || !FU || !FV || !scratch || !weights) return ocn_fail(OCN_ERR_INVALID, "ocn_barotropic_substeps: NULL argument");
  if (g->ext_halo[1])   // Periodic axes wrap by index inside the local plane: wrong on a slab
    return ocn_fail(OCN_ERR_UNSUPPORTED, "ocn_barotropic_substeps: the substepper is not sharded: this grid is a y-slab (ocn_grid_set_external_halo)");
  if (N < 1 || M < 1) return ocn_fail(OCN_ERR_INVALID, "ocn_barotropic_substeps: N and M must be >= 1 (got %d, %d)", N, M);
  if (!(dt > 0.0) || !(grav >= 0.0)) return ocn_fail(OCN_ERR_INVALID, "ocn_barotropic_substeps: dt must be > 0 and g >= 0");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t esz = g->dtype == OCN_F64 ? 8 : 4, plane = (size_t)g->lay.stride_z * esz;
  char *w = (char *)scratch;
  BtPlanes A = {bt->eta, bt->U, bt->V}, B = {w, w + plane, w + 2 * plane}, acc = {w + 3 * plane, w + 4 * plane, w + 5 * plane};
  const Plane2 P = make_plane(g);
  const double dtau = dt / (double)N, gH = grav * column_depth(g);
  // S substeps per launch where the plane is large enough for the 64 x 32 regions (no double wrap) and 2-D; else one launch per substep
  const bool blocked = g->topo[0] != OCN_FLAT && g->topo[1] != OCN_FLAT && g->Nx >= BT_RX && g->Ny >= BT_RY && !(g->diag & OCN_DIAG_BT_SINGLESTEP);
  if (blocked) {
    const size_t smem = (size_t)5 * BT_RX * BT_RY * esz;
    static OcnPerDeviceOnce once;
    if (once.first()) {
      OCN_CUDA(cudaFuncSetAttribute(barotropic_multistep_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, 5 * BT_RX * BT_RY * 8));
      OCN_CUDA(cudaFuncSetAttribute(barotropic_multistep_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 5 * BT_RX * BT_RY * 4));
    }
    const int ox = BT_RX - 2 * BT_S, oy = BT_RY - 2 * BT_S;
    dim3 grid((g->Nx + ox - 1) / ox, (g->Ny + oy - 1) / oy, 1);
    int ng = 0;
    for (int n0 = 0; n0 < M; n0 += BT_S, ++ng) {
      const BtPlanes &in = (ng & 1) ? B : A, &out = (ng & 1) ? A : B;
      BtWeights w;
      const int ns = std::min(BT_S, M - n0);
      for (int t = 0; t < BT_S; ++t) w.a[t] = t < ns ? weights[n0 + t] : 0.0;
      if (g->dtype == OCN_F64)
        barotropic_multistep_kernel<double><<<grid, BT_NT, smem, s>>>(P, in, out, acc, (const double *)FU, (const double *)FV, dtau, g->dev.rdx, g->dev.rdy, gH, w, ns, n0 == 0);
      else
        barotropic_multistep_kernel<float><<<grid, BT_NT, smem, s>>>(P, in, out, acc, (const float *)FU, (const float *)FV, dtau, g->dev.rdx, g->dev.rdy, gH, w, ns, n0 == 0);
    }
    ocn_count_launch(ng);
  } else {
    dim3 block(64, 4, 1), grid((g->Nx + 63) / 64, (g->Ny + 3) / 4, 1);
    for (int n = 1; n <= M; ++n) {
      const BtPlanes &in = (n & 1) ? A : B, &out = (n & 1) ? B : A;
      if (g->dtype == OCN_F64)
        barotropic_substep_kernel<double><<<grid, block, 0, s>>>(P, in, out, acc, (const double *)FU, (const double *)FV, dtau, g->dev.rdx, g->dev.rdy, gH, weights[n - 1], n == 1);
      else
        barotropic_substep_kernel<float><<<grid, block, 0, s>>>(P, in, out, acc, (const float *)FU, (const float *)FV, dtau, g->dev.rdx, g->dev.rdy, gH, weights[n - 1], n == 1);
    }
    ocn_count_launch(M);
  }
  OCN_CUDA(cudaGetLastError());
  // the barotropic variables are re-initialised with the averages
  OCN_CUDA(cudaMemcpyAsync(bt->eta, acc.eta, plane, cudaMemcpyDeviceToDevice, s));
  OCN_CUDA(cudaMemcpyAsync(bt->U, acc.U, plane, cudaMemcpyDeviceToDevice, s));
  OCN_CUDA(cudaMemcpyAsync(bt->V, acc.V, plane, cudaMemcpyDeviceToDevice, s));
  return OCN_OK;
}

// ---- ocn_barotropic_substeps_static: the substepper for callers that own no device scratch and may not ask the CUDA allocator
// for any (see include/ocn.h).  The six work planes live in this file-scope device array, which every GPU that loads the library
// keeps until the process exits.  NOTE for whoever edits this: in HOST code the name `bt_static_scratch` is only a handle of the
// symbol, not a device address — a kernel or a cudaMemsetAsync handed `bt_static_scratch` itself would fault (or, on machines where
// the GPU can reach host memory, quietly scribble on host memory).  The device address comes from cudaGetSymbolAddress, asked once
// per device with that device current, and is cached below.
static __device__ __align__(256) unsigned char bt_static_scratch[OCN_BT_STATIC_SCRATCH_BYTES];

static int bt_static_scratch_address(void **out) {
  static void *addr[64] = {};          // per device ordinal; a repeated look-up by a second host thread stores the same value
  int d = 0;
  OCN_CUDA(cudaGetDevice(&d));
  if (d < 0 || d >= 64) return ocn_fail(OCN_ERR_UNSUPPORTED, "ocn_barotropic_substeps_static: device ordinal %d beyond the 64 this entry point tracks", d);
  if (!addr[d]) {
    void *p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, bt_static_scratch);
    if (e != cudaSuccess || !p) return ocn_check_cuda(e != cudaSuccess ? e : cudaErrorInvalidSymbol, "ocn_barotropic_substeps_static: cudaGetSymbolAddress(bt_static_scratch)");
    addr[d] = p;
  }
  *out = addr[d];
  return OCN_OK;
}

int ocn_barotropic_substeps_static(const ocn_grid *g, double grav, double dt, int N, int M, const double *weights, ocn_barotropic *bt,
                                   const void *FU, const void *FV, void *stream) {
  int rc = check_grid("ocn_barotropic_substeps_static", g);
  if (rc) return rc;
  const size_t esz = g->dtype == OCN_F64 ? 8 : 4, plane = (size_t)g->lay.stride_z * esz;
  if (6 * plane > (size_t)OCN_BT_STATIC_SCRATCH_BYTES)
    return ocn_fail(OCN_ERR_UNSUPPORTED,
                    "ocn_barotropic_substeps_static: six planes of this grid need %zu bytes, the built-in scratch holds %zu "
                    "(OCN_BT_STATIC_SCRATCH_BYTES); use ocn_barotropic_substeps with caller-owned scratch",
                    6 * plane, (size_t)OCN_BT_STATIC_SCRATCH_BYTES);
  void *scratch = nullptr;
  if ((rc = bt_static_scratch_address(&scratch))) return rc;
  // The array still holds whatever the previous call (any grid, any dtype) left in it.  The substep kernels write every interior
  // cell of all six planes before reading it, so only one thing has to start from zero: the three planes of averages (the second
  // half), because they are copied back WHOLE into bt->eta / U / V and their halo and padding elements would otherwise carry the
  // last call's bytes into the caller's planes.
  OCN_CUDA(cudaMemsetAsync((char *)scratch + 3 * plane, 0, 3 * plane, (cudaStream_t)stream));
  return ocn_barotropic_substeps(g, grav, dt, N, M, weights, bt, FU, FV, scratch, stream);
}

int ocn_barotropic_correct(const ocn_grid *g, ocn_fields *state, const ocn_barotropic *bt, void *stream) {
  int rc = check_grid("ocn_barotropic_correct", g);
  if (rc) return rc;
  if (!state || !bt || !state->u || !state->v || !bt->U || !bt->V) return ocn_fail(OCN_ERR_INVALID, "ocn_barotropic_correct: NULL argument");
  dim3 block(64, 2, 1), grid((g->Nx + 63) / 64, (g->Ny + 1) / 2, 2);
  const double rH = 1.0 / column_depth(g);
  cudaStream_t s = (cudaStream_t)stream;
  const Plane2 P = make_plane(g);
  if (g->dtype == OCN_F64) {
    if (g->Nz <= 64) barotropic_correct_kernel<double, 64><<<grid, block, 0, s>>>(g->dev, P, (double *)state->u, (double *)state->v, (const double *)bt->U, (const double *)bt->V, rH);
    else barotropic_correct_kernel<double, 0><<<grid, block, 0, s>>>(g->dev, P, (double *)state->u, (double *)state->v, (const double *)bt->U, (const double *)bt->V, rH);
  } else {
    if (g->Nz <= 64) barotropic_correct_kernel<float, 64><<<grid, block, 0, s>>>(g->dev, P, (float *)state->u, (float *)state->v, (const float *)bt->U, (const float *)bt->V, rH);
    else barotropic_correct_kernel<float, 0><<<grid, block, 0, s>>>(g->dev, P, (float *)state->u, (float *)state->v, (const float *)bt->U, (const float *)bt->V, rH);
  }
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "barotropic_correct_kernel launch");
}

}  // extern "C"
