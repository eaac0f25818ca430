// pressure.cu — SURVEY 8(f) N2: the pressure correction of the NonhydrostaticModel, (A8)-(A12) PAPER.md:829-851.
//
//     rhs = div(u~) / dt                         pressure_rhs_kernel        (A12) right-hand side, (B2) divergence
//     lap p = rhs                                cuFFT R2C (x,y)  ->  poisson_tridiag_kernel (z)  ->  cuFFT C2R
//     u^{m+1} = u~ - dt grad p                   pressure_correct_kernel    (A11)
//
// "an eigenfunction expansion of the discrete second-order Poisson operator evaluated via the fast Fourier transform in
// equispaced directions plus a tridiagonal solve in variably-spaced directions": x and y (Periodic, uniform)
// by FFT — the FFT itself is a library primitive (cuFFT, batched 2-D real-to-complex over the Nz levels, reading / writing
// the interior of the halo-padded field directly through the advanced data layout) — and z (Bounded, possibly stretched) by
// one Thomas solve per horizontal mode, written here.  Readings R21-R23: dt is the caller's interval; wall-normal
// predictor velocity is 0 on wall faces (homogeneous Neumann rows); the singular mean mode is fixed by p^(0,0,k=1) = 0.
//
// All three kernels are HBM-bound streaming passes:
//   rhs      reads u,v,w once, writes rhs                       4 x sizeof per cell
//   tridiag  forward sweep reads r^, writes d' and c'; backward sweep reads d', c', writes p^   (thread per mode, modes
//            contiguous in memory => every level is a fully coalesced row; the recurrence is evaluated in double for
//            both storage types: the low modes have |lambda| ~ (2 pi / N)^2 << 1 next to off-diagonals of O(1/dz^2))
//   correct  reads p (neighbours from L1/L2), reads and writes u,v,w   7 x sizeof per cell
#include <cufft.h>

#include <cmath>
#include <new>

#include "ocn_internal.h"

struct ocn_poisson {
  const ocn_grid *g;      // the solver indexes fields with THIS grid's strides, sizes and dtype; it must not outlive it
  unsigned long long gid; // id of that grid at creation (ocn_grid_alive)
  int Nxh;               // Nx/2 + 1 complex modes along x
  long long nmodes;      // Nxh * Ny
  cufftHandle fwd, inv;
  bool have_plans;
  void *spec;            // DEVICE: nmodes * Nz complex (double2 / float2)
  double *cws;           // DEVICE: nmodes * Nz, the Thomas c' coefficients
  double *zlo, *zup;     // DEVICE: Nz each, 1/(dzf[k] dzc[k]) (0 at k=1), 1/(dzf[k+1] dzc[k]) (0 at k=Nz)
};

namespace {

template <class Real> struct Cplx;
template <> struct Cplx<double> { typedef double2 type; };
template <> struct Cplx<float> { typedef float2 type; };

// ---- (A12) right-hand side: rhs = div(u~)/dt at ccc; face N+1 = face 1 (Periodic) / wall = 0 (Bounded), R22 ----
// A thread owns KC consecutive levels of one column: its KC x 5 loads are issued before the first use (the kernel is a pure HBM
// stream, so what matters is bytes in flight), and the w face between two of its levels is read once.
constexpr int RHS_KC = 8;
template <class Real>
__global__ void __launch_bounds__(256) pressure_rhs_kernel(const GridDev g, const Real *__restrict__ u, const Real *__restrict__ v,
                                                           const Real *__restrict__ w, Real *__restrict__ rhs, const double rdt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1, j = blockIdx.y * blockDim.y + threadIdx.y + 1, k0 = blockIdx.z * RHS_KC + 1;
  if (i > g.Nx || j > g.Ny) return;
  const long long o0 = g.idx(i, j, k0);
  const long long dxo = i == g.Nx ? -(long long)(g.Nx - 1) : 1, dyo = j == g.Ny ? -(long long)(g.Ny - 1) * g.sy : g.sy;   // Periodic wrap
  Real ul[RHS_KC], uh[RHS_KC], vl[RHS_KC], vh[RHS_KC], wf[RHS_KC + 1];
#pragma unroll
  for (int m = 0; m < RHS_KC; ++m) {
    const bool in = k0 + m <= g.Nz;
    const long long o = o0 + m * g.sz;
    ul[m] = in && u ? u[o] : Real(0); uh[m] = in && u ? u[o + dxo] : Real(0);
    vl[m] = in && v ? v[o] : Real(0); vh[m] = in && v ? v[o + dyo] : Real(0);
  }
#pragma unroll
  for (int m = 0; m <= RHS_KC; ++m) {   // z Bounded: faces 1 and Nz+1 are walls (R22)
    const int k = k0 + m;
    wf[m] = (w && k > 1 && k <= g.Nz) ? w[o0 + m * g.sz] : Real(0);
  }
  // arithmetic in the storage type (fp32 grids: ten F2F conversions per cell cost more than the memory traffic, measured)
  const Real rdx = Real(g.rdx), rdy = Real(g.rdy), rdtr = Real(rdt);
#pragma unroll
  for (int m = 0; m < RHS_KC; ++m) {
    if (k0 + m > g.Nz) break;
    Real d = (uh[m] - ul[m]) * rdx;
    d = fma(vh[m] - vl[m], rdy, d);
    if (w) d = fma(wf[m + 1] - wf[m], Real(g.rdzc[g.zi(k0 + m)]), d);
    rhs[o0 + m * g.sz] = d * rdtr;
  }
}

// ---- z: one Thomas solve per horizontal mode (mx,my); thread t owns mode t = my*Nxh + mx, level stride = nmodes ----
//   (lx + ly) p_k + zup[k] (p_{k+1} - p_k) - zlo[k] (p_k - p_{k-1}) = r_k        (no-flux walls: zlo[1] = zup[Nz] = 0)
template <class Real>
__global__ void __launch_bounds__(128) poisson_tridiag_kernel(typename Cplx<Real>::type *__restrict__ spec, double *__restrict__ cws,
                                                              const double *__restrict__ zlo, const double *__restrict__ zup,
                                                              const int Nx, const int Ny, const int Nz, const int Nxh,
                                                              const double dx, const double dy, const double scale) {
  typedef typename Cplx<Real>::type C2;
  const long long nm = (long long)Nxh * Ny;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nm) return;
  const int mx = (int)(t % Nxh), my = (int)(t / Nxh);
  const double sx = sinpi((double)mx / (double)Nx), sy = sinpi((double)my / (double)Ny);
  const double lam = -4.0 * sx * sx / (dx * dx) - 4.0 * sy * sy / (dy * dy);
  const bool mean_mode = t == 0;
  if (Nz == 1) {   // z Flat: p^ = r^ / lambda, mean mode 0 (R23)
    C2 r = spec[t];
    const double s = mean_mode ? 0.0 : scale / lam;
    r.x = Real((double)r.x * s); r.y = Real((double)r.y * s);
    spec[t] = r;
    return;
  }
  // The grid has only Nx/2+1 x Ny threads (C2: 889 per SM), so the bytes in flight must come from each thread: every batch of
  // TB levels is loaded before its recurrence runs and stores (the compiler does not hoist a load above an earlier store).
  constexpr int TB = 8;
  double cp = 0.0, dre = 0.0, dim = 0.0;
  int k = 0;
  for (; k + TB <= Nz; k += TB) {
    C2 r[TB];
    double lo[TB], up[TB];
#pragma unroll
    for (int m = 0; m < TB; ++m) { r[m] = spec[t + (long long)(k + m) * nm]; lo[m] = zlo[k + m]; up[m] = zup[k + m]; }
#pragma unroll
    for (int m = 0; m < TB; ++m) {
      double diag = lam - lo[m] - up[m], rre = (double)r[m].x * scale, rim = (double)r[m].y * scale;
      if (mean_mode && k + m == 0) { up[m] = 0.0; diag = 1.0; rre = 0.0; rim = 0.0; }   // gauge row (R23)
      const double inv = 1.0 / (diag - lo[m] * cp);
      cp = up[m] * inv;
      dre = (rre - lo[m] * dre) * inv;
      dim = (rim - lo[m] * dim) * inv;
      cws[t + (long long)(k + m) * nm] = cp;
      C2 d; d.x = Real(dre); d.y = Real(dim);
      spec[t + (long long)(k + m) * nm] = d;
    }
  }
  for (; k < Nz; ++k) {
    const long long o = t + (long long)k * nm;
    const C2 r = spec[o];
    double lo = zlo[k], up = zup[k], diag = lam - lo - up;
    double rre = (double)r.x * scale, rim = (double)r.y * scale;
    if (mean_mode && k == 0) { up = 0.0; diag = 1.0; rre = 0.0; rim = 0.0; }
    const double inv = 1.0 / (diag - lo * cp);
    cp = up * inv;
    dre = (rre - lo * dre) * inv;
    dim = (rim - lo * dim) * inv;
    cws[o] = cp;
    C2 d; d.x = Real(dre); d.y = Real(dim);
    spec[o] = d;
  }
  // back substitution: p_k = d'_k - c'_k p_{k+1}; level Nz-1 already holds its solution
  double xre = dre, xim = dim;
  k = Nz - 2;
  for (; k - TB + 1 >= 0; k -= TB) {
    C2 d[TB];
    double c[TB];
#pragma unroll
    for (int m = 0; m < TB; ++m) { d[m] = spec[t + (long long)(k - m) * nm]; c[m] = cws[t + (long long)(k - m) * nm]; }
#pragma unroll
    for (int m = 0; m < TB; ++m) {
      xre = (double)d[m].x - c[m] * xre;
      xim = (double)d[m].y - c[m] * xim;
      C2 x; x.x = Real(xre); x.y = Real(xim);
      spec[t + (long long)(k - m) * nm] = x;
    }
  }
  for (; k >= 0; --k) {
    const long long o = t + (long long)k * nm;
    const C2 d = spec[o];
    const double c = cws[o];
    xre = (double)d.x - c * xre;
    xim = (double)d.y - c * xim;
    C2 x; x.x = Real(xre); x.y = Real(xim);
    spec[o] = x;
  }
}

// ---- (A11): u -= dt dx(p)/dx, v -= dt dy(p)/dy, w -= dt dz(p)/dzf on non-wall faces; Periodic wrap of p in x,y ----
// KC levels per thread with every load issued before the first use, as in pressure_rhs_kernel; p between two of the thread's
// levels is read once.
constexpr int COR_KC = 4;
template <class Real>
__global__ void __launch_bounds__(256) pressure_correct_kernel(const GridDev g, Real *__restrict__ u, Real *__restrict__ v,
                                                               Real *__restrict__ w, const Real *__restrict__ p, const double dt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x + 1, j = blockIdx.y * blockDim.y + threadIdx.y + 1, k0 = blockIdx.z * COR_KC + 1;
  if (i > g.Nx || j > g.Ny) return;
  const long long o0 = g.idx(i, j, k0);
  const long long dxo = i == 1 ? (long long)(g.Nx - 1) : -1, dyo = j == 1 ? (long long)(g.Ny - 1) * g.sy : -g.sy;   // Periodic wrap
  Real pc[COR_KC + 1], px[COR_KC], py[COR_KC], uu[COR_KC], vv[COR_KC], ww[COR_KC];
  pc[0] = k0 > 1 ? p[o0 - g.sz] : Real(0);
#pragma unroll
  for (int m = 0; m < COR_KC; ++m) {
    const bool in = k0 + m <= g.Nz;
    const long long o = o0 + m * g.sz;
    pc[m + 1] = in ? p[o] : Real(0);
    px[m] = in && u ? p[o + dxo] : Real(0); py[m] = in && v ? p[o + dyo] : Real(0);
    uu[m] = in && u ? u[o] : Real(0); vv[m] = in && v ? v[o] : Real(0); ww[m] = in && w ? w[o] : Real(0);
  }
  const Real mdt = Real(-dt), rdx = Real(g.rdx), rdy = Real(g.rdy);   // arithmetic in the storage type
#pragma unroll
  for (int m = 0; m < COR_KC; ++m) {
    const int k = k0 + m;
    if (k > g.Nz) break;
    const long long o = o0 + m * g.sz;
    if (u) u[o] = fma(mdt, (pc[m + 1] - px[m]) * rdx, uu[m]);
    if (v) v[o] = fma(mdt, (pc[m + 1] - py[m]) * rdy, vv[m]);
    if (w && k > 1) w[o] = fma(mdt, (pc[m + 1] - pc[m]) * Real(g.rdzf[g.zi(k)]), ww[m]);
  }
}

int check_cufft(cufftResult r, const char *what) {
  if (r == CUFFT_SUCCESS) return OCN_OK;
  return ocn_fail(OCN_ERR_CUDA, "%s: cuFFT error %d", what, (int)r);
}

int supported(const char *who, const ocn_grid *g) {
  if (!g) return ocn_fail(OCN_ERR_INVALID, "%s: grid is NULL", who);
  if (g->topo[0] != OCN_PERIODIC || g->topo[1] != OCN_PERIODIC || g->topo[2] == OCN_PERIODIC)
    return ocn_fail(OCN_ERR_UNSUPPORTED, "%s: the pressure solver covers Periodic x, Periodic y and Bounded or Flat z (the nonhydrostatic configurations)", who);
  if (g->ext_halo[1])   // the y transform would wrap inside the local slab
    return ocn_fail(OCN_ERR_UNSUPPORTED, "%s: the FFT pressure solver is not sharded: this grid is a y-slab (ocn_grid_set_external_halo)", who);
  return OCN_OK;
}

dim3 cell_grid(const ocn_grid *g, dim3 block) { return dim3((g->Nx + block.x - 1) / block.x, (g->Ny + block.y - 1) / block.y, g->Nz); }

}  // namespace

const ocn_grid *ocn_poisson_grid(const ocn_poisson *ps, const char *who) {
  if (!ps) { ocn_fail(OCN_ERR_INVALID, "%s: solver is NULL", who); return nullptr; }
  if (!ocn_grid_alive(ps->g, ps->gid)) { ocn_fail(OCN_ERR_INVALID, "%s: the grid this Poisson solver was created for has been destroyed", who); return nullptr; }
  return ps->g;
}

extern "C" {

int ocn_poisson_create(ocn_poisson **out, const ocn_grid *g) {
  if (!out) return ocn_fail(OCN_ERR_INVALID, "ocn_poisson_create: out is NULL");
  *out = nullptr;
  int rc = supported("ocn_poisson_create", g);
  if (rc) return rc;
  ocn_poisson *ps = new (std::nothrow) ocn_poisson();
  if (!ps) return ocn_fail(OCN_ERR_NOMEM, "ocn_poisson_create: out of host memory");
  ps->g = g; ps->gid = g->id; ps->Nxh = g->Nx / 2 + 1; ps->nmodes = (long long)ps->Nxh * g->Ny;
  ps->have_plans = false; ps->spec = nullptr; ps->cws = nullptr; ps->zlo = nullptr; ps->zup = nullptr;
  const int Nz = g->Nz;
  const size_t csz = g->dtype == OCN_F64 ? sizeof(double2) : sizeof(float2);
  cudaError_t e = cudaMalloc(&ps->spec, csz * ps->nmodes * Nz);
  if (e == cudaSuccess) e = cudaMalloc((void **)&ps->cws, sizeof(double) * ps->nmodes * Nz);
  if (e == cudaSuccess) e = cudaMalloc((void **)&ps->zlo, sizeof(double) * 2 * Nz);
  if (e != cudaSuccess) { ocn_poisson_destroy(ps); return ocn_check_cuda(e, "ocn_poisson_create: cudaMalloc"); }
  ps->zup = ps->zlo + Nz;
  std::vector<double> z(2 * Nz, 0.0);
  for (int k = 1; k <= Nz; ++k) {
    const double dzc = g->h_dzc[k + g->Hz];
    if (k > 1) z[k - 1] = 1.0 / (g->h_dzf[k + g->Hz] * dzc);
    if (k < Nz) z[Nz + k - 1] = 1.0 / (g->h_dzf[k + 1 + g->Hz] * dzc);
  }
  e = cudaMemcpy(ps->zlo, z.data(), sizeof(double) * 2 * Nz, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { ocn_poisson_destroy(ps); return ocn_check_cuda(e, "ocn_poisson_create: cudaMemcpy"); }
  // batched 2-D transforms over the Nz levels straight from / into the interior of the padded field
  int n[2] = {g->Ny, g->Nx};
  int rembed[2] = {(int)g->lay.ny_pad, (int)g->lay.stride_y};
  int cembed[2] = {g->Ny, ps->Nxh};
  const bool f64 = g->dtype == OCN_F64;
  cufftResult r = cufftPlanMany(&ps->fwd, 2, n, rembed, 1, (int)g->lay.stride_z, cembed, 1, (int)ps->nmodes, f64 ? CUFFT_D2Z : CUFFT_R2C, Nz);
  if (r != CUFFT_SUCCESS) { ocn_poisson_destroy(ps); return check_cufft(r, "ocn_poisson_create: cufftPlanMany(forward)"); }
  r = cufftPlanMany(&ps->inv, 2, n, cembed, 1, (int)ps->nmodes, rembed, 1, (int)g->lay.stride_z, f64 ? CUFFT_Z2D : CUFFT_C2R, Nz);
  if (r != CUFFT_SUCCESS) { cufftDestroy(ps->fwd); ocn_poisson_destroy(ps); return check_cufft(r, "ocn_poisson_create: cufftPlanMany(inverse)"); }
  ps->have_plans = true;
  *out = ps;
  return OCN_OK;
}

int ocn_poisson_destroy(ocn_poisson *ps) {
  if (!ps) return OCN_OK;
  if (ps->have_plans) { cufftDestroy(ps->fwd); cufftDestroy(ps->inv); }
  if (ps->spec) cudaFree(ps->spec);
  if (ps->cws) cudaFree(ps->cws);
  if (ps->zlo) cudaFree(ps->zlo);
  delete ps;
  return OCN_OK;
}

int ocn_pressure_rhs(const ocn_grid *g, double dt, const ocn_fields *state, void *rhs, void *stream) {
  int rc = supported("ocn_pressure_rhs", g);
  if (rc) return rc;
  if (!state || !rhs) return ocn_fail(OCN_ERR_INVALID, "ocn_pressure_rhs: NULL argument");
  if (!(dt > 0.0)) return ocn_fail(OCN_ERR_INVALID, "ocn_pressure_rhs: dt must be > 0");
  if (!state->u || !state->v || (g->topo[2] != OCN_FLAT && !state->w)) return ocn_fail(OCN_ERR_INVALID, "ocn_pressure_rhs: a velocity component is NULL");
  const void *w = g->topo[2] == OCN_FLAT ? nullptr : state->w;
  dim3 block(64, 4, 1), grid = cell_grid(g, block);
  grid.z = (g->Nz + RHS_KC - 1) / RHS_KC;
  cudaStream_t s = (cudaStream_t)stream;
  if (g->dtype == OCN_F64) pressure_rhs_kernel<double><<<grid, block, 0, s>>>(g->dev, (const double *)state->u, (const double *)state->v, (const double *)w, (double *)rhs, 1.0 / dt);
  else pressure_rhs_kernel<float><<<grid, block, 0, s>>>(g->dev, (const float *)state->u, (const float *)state->v, (const float *)w, (float *)rhs, 1.0 / dt);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "pressure_rhs_kernel launch");
}

int ocn_poisson_solve(ocn_poisson *ps, const void *rhs, void *p, void *stream) {
  if (!ps || !rhs || !p) return ocn_fail(OCN_ERR_INVALID, "ocn_poisson_solve: NULL argument");
  const ocn_grid *g = ocn_poisson_grid(ps, "ocn_poisson_solve");
  if (!g) return OCN_ERR_INVALID;
  if (int rcs = supported("ocn_poisson_solve", g)) return rcs;
  if (int rca = ocn_check_aligned("ocn_poisson_solve", g, rhs, "rhs")) return rca;
  if (int rca = ocn_check_aligned("ocn_poisson_solve", g, p, "p")) return rca;
  cudaStream_t s = (cudaStream_t)stream;
  int rc;
  if ((rc = check_cufft(cufftSetStream(ps->fwd, s), "cufftSetStream"))) return rc;
  if ((rc = check_cufft(cufftSetStream(ps->inv, s), "cufftSetStream"))) return rc;
  const double scale = 1.0 / ((double)g->Nx * (double)g->Ny);   // cuFFT transforms are unnormalised
  const int threads = 128;
  const unsigned blocks = (unsigned)((ps->nmodes + threads - 1) / threads);
  if (g->dtype == OCN_F64) {
    double *in = (double *)rhs + g->lay.offset0, *outp = (double *)p + g->lay.offset0;
    if ((rc = check_cufft(cufftExecD2Z(ps->fwd, in, (cufftDoubleComplex *)ps->spec), "cufftExecD2Z"))) return rc;
    poisson_tridiag_kernel<double><<<blocks, threads, 0, s>>>((double2 *)ps->spec, ps->cws, ps->zlo, ps->zup, g->Nx, g->Ny, g->Nz, ps->Nxh, g->dx, g->dy, scale);
    OCN_CUDA(cudaGetLastError());
    if ((rc = check_cufft(cufftExecZ2D(ps->inv, (cufftDoubleComplex *)ps->spec, outp), "cufftExecZ2D"))) return rc;
  } else {
    float *in = (float *)rhs + g->lay.offset0, *outp = (float *)p + g->lay.offset0;
    if ((rc = check_cufft(cufftExecR2C(ps->fwd, in, (cufftComplex *)ps->spec), "cufftExecR2C"))) return rc;
    poisson_tridiag_kernel<float><<<blocks, threads, 0, s>>>((float2 *)ps->spec, ps->cws, ps->zlo, ps->zup, g->Nx, g->Ny, g->Nz, ps->Nxh, g->dx, g->dy, scale);
    OCN_CUDA(cudaGetLastError());
    if ((rc = check_cufft(cufftExecC2R(ps->inv, (cufftComplex *)ps->spec, outp), "cufftExecC2R"))) return rc;
  }
  ocn_count_launch();   // the Thomas kernel (cuFFT's own kernels are not counted: they are library launches)
  return OCN_OK;
}

int ocn_pressure_correct(const ocn_grid *g, double dt, ocn_fields *state, const void *p, void *stream) {
  int rc = supported("ocn_pressure_correct", g);
  if (rc) return rc;
  if (!state || !p) return ocn_fail(OCN_ERR_INVALID, "ocn_pressure_correct: NULL argument");
  if (!state->u || !state->v || (g->topo[2] != OCN_FLAT && !state->w)) return ocn_fail(OCN_ERR_INVALID, "ocn_pressure_correct: a velocity component is NULL");
  void *w = g->topo[2] == OCN_FLAT ? nullptr : state->w;
  dim3 block(64, 4, 1), grid = cell_grid(g, block);
  grid.z = (g->Nz + COR_KC - 1) / COR_KC;
  cudaStream_t s = (cudaStream_t)stream;
  if (g->dtype == OCN_F64) pressure_correct_kernel<double><<<grid, block, 0, s>>>(g->dev, (double *)state->u, (double *)state->v, (double *)w, (const double *)p, dt);
  else pressure_correct_kernel<float><<<grid, block, 0, s>>>(g->dev, (float *)state->u, (float *)state->v, (float *)w, (const float *)p, dt);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "pressure_correct_kernel launch");
}

int ocn_pressure_correction(ocn_poisson *ps, double dt, ocn_fields *state, void *p, void *stream) {
  const ocn_grid *g = ocn_poisson_grid(ps, "ocn_pressure_correction");
  if (!g) return OCN_ERR_INVALID;
  int rc = ocn_pressure_rhs(g, dt, state, p, stream);
  if (rc) return rc;
  if ((rc = ocn_poisson_solve(ps, p, p, stream))) return rc;
  return ocn_pressure_correct(g, dt, state, p, stream);
}

}  // extern "C"
