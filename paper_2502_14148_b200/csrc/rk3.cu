// rk3.cu — a11: low-storage RK3 substage, eq. (A4) PAPER.md:797-801:
//     q <- q + dt (gamma^m G^m - zeta^m G^{m-1})     gamma = (8/15, 5/12, 3/4), zeta = (0, 17/60, 5/12)
// on the interior non-wall points of every prognostic field, ALL fields in one launch (blockIdx.y = field).
// Pointwise and HBM-bound (4 x sizeof bytes per field-point, 3 x at stage 1 where zeta = 0 and G^{m-1} is
// not read): rows are walked with 16-byte vector accesses (the library-chosen layout makes every interior
// row start 16-byte aligned), several independent vectors in flight per thread.
#include "ocn_internal.h"

namespace {

struct SubArgs {
  GridDev g;
  int nfields;
  void *q[3 + OCN_MAX_TRACERS];
  const void *G[3 + OCN_MAX_TRACERS];
  const void *Gp[3 + OCN_MAX_TRACERS];
  int i0[3 + OCN_MAX_TRACERS], j0[3 + OCN_MAX_TRACERS], k0[3 + OCN_MAX_TRACERS];   // first prognostic index
  double a, b;   // dt*gamma, dt*zeta
  int use_prev;
};

template <class Real> struct Vec;
template <> struct Vec<double> { typedef double2 T; static constexpr int W = 2; };
template <> struct Vec<float> { typedef float4 T; static constexpr int W = 4; };

template <class Real, bool PREV>
__global__ void __launch_bounds__(256) substage_kernel(const SubArgs s) {
  typedef typename Vec<Real>::T V;
  constexpr int W = Vec<Real>::W;
  const GridDev &g = s.g;
  const int f = blockIdx.y;
  Real *__restrict__ q = (Real *)s.q[f];
  const Real *__restrict__ G = (const Real *)s.G[f];
  const Real *__restrict__ Gp = (const Real *)s.Gp[f];
  const Real a = Real(s.a), b = Real(s.b);
  const int i0 = s.i0[f], j0 = s.j0[f], k0 = s.k0[f];
  const int nvec = (g.Nx + W - 1) / W;                     // vectors per row (last one may be ragged)
  const long long rows = (long long)g.Ny * g.Nz;
  const long long total = rows * nvec;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
    const long long row = t / nvec;
    const int iv = (int)(t - row * nvec);
    const int k = (int)(row / g.Ny) + 1, j = (int)(row % g.Ny) + 1;
    if (k < k0 || j < j0) continue;
    const int i = iv * W + 1;
    const long long o = g.idx(i, j, k);
    if (i + W - 1 <= g.Nx && i >= i0) {
      V vq = *reinterpret_cast<const V *>(q + o);
      const V vg = *reinterpret_cast<const V *>(G + o);
      Real *pq = reinterpret_cast<Real *>(&vq);
      const Real *pg = reinterpret_cast<const Real *>(&vg);
      if (PREV) {
        const V vp = *reinterpret_cast<const V *>(Gp + o);
        const Real *pp = reinterpret_cast<const Real *>(&vp);
#pragma unroll
        for (int e = 0; e < W; ++e) pq[e] = rk3_update(pq[e], pg[e], pp[e], a, b);
      } else {
#pragma unroll
        for (int e = 0; e < W; ++e) pq[e] = rk3_update(pq[e], pg[e], a);
      }
      *reinterpret_cast<V *>(q + o) = vq;
    } else {
      for (int e = 0; e < W; ++e) {
        const int ii = i + e;
        if (ii > g.Nx || ii < i0) continue;
        q[o + e] = PREV ? rk3_update(q[o + e], G[o + e], Gp[o + e], a, b) : rk3_update(q[o + e], G[o + e], a);
      }
    }
  }
}

}  // namespace

int launch_substage(const ocn_grid *g, const ModelDev &m, double gamma, double zeta, double dt, const FieldsDev &st,
                    const FieldsDev &G, const FieldsDev &Gp, cudaStream_t s) {
  SubArgs a;
  a.g = g->dev;
  int n = 0;
  const bool prev = zeta != 0.0;
  auto add = [&](void *q, const void *gg, const void *gp, int fx, int fy, int fz) {
    a.q[n] = q; a.G[n] = gg; a.Gp[n] = gp;
    a.i0[n] = fx ? first_face(g->topo[0]) : 1;
    a.j0[n] = fy ? first_face(g->topo[1]) : 1;
    a.k0[n] = fz ? first_face(g->topo[2]) : 1;
    ++n;
  };
  if (m.momentum) {
    if (st.u) add(st.u, G.u, Gp.u, 1, 0, 0);
    if (st.v) add(st.v, G.v, Gp.v, 0, 1, 0);
    if (st.w && !m.hydrostatic && g->topo[2] != OCN_FLAT) add(st.w, G.w, Gp.w, 0, 0, 1);
  }
  for (int t = 0; t < m.n_tracers; ++t) add(st.c[t], G.c[t], Gp.c[t], 0, 0, 0);
  for (int f = 0; f < n; ++f) {
    if (!a.G[f]) return ocn_fail(OCN_ERR_INVALID, "substage: tendency of prognostic field %d is NULL", f);
    if (prev && !a.Gp[f]) return ocn_fail(OCN_ERR_INVALID, "substage: previous tendency of field %d is NULL but zeta != 0", f);
  }
  a.nfields = n;
  if (n == 0) return OCN_OK;
  a.a = dt * gamma;
  a.b = dt * zeta;
  a.use_prev = prev;
  const int W = g->dtype == OCN_F64 ? 2 : 4;
  const long long total = (long long)g->Ny * g->Nz * ((g->Nx + W - 1) / W);
  long long blocks = (total + 255) / 256;
  if (blocks > 148LL * 16) blocks = 148LL * 16;
  if (blocks < 1) blocks = 1;
  dim3 grid((unsigned)blocks, (unsigned)n, 1);
  if (g->dtype == OCN_F64) {
    if (prev) substage_kernel<double, true><<<grid, 256, 0, s>>>(a);
    else substage_kernel<double, false><<<grid, 256, 0, s>>>(a);
  } else {
    if (prev) substage_kernel<float, true><<<grid, 256, 0, s>>>(a);
    else substage_kernel<float, false><<<grid, 256, 0, s>>>(a);
  }
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "substage_kernel launch");
}
