// tend_fused.cu — OCN_KERNEL_FUSED: the fused tendency kernel for 3-D grids with WENO5 in x,y.
//
// 2.5-D blocking with DIRECTION-SPECIALISED warps.  A block owns a 31 x TY tile of (i,j) columns and marches along z:
//   * a producer warp streams plane after plane of every input field, with a 3-cell halo, into a ring of NBUF
//     shared-memory slots by TMA tiled loads (cp.async.bulk.tensor.3d + mbarrier complete_tx); the ring keeps the six
//     planes k-2..k+3 of the z-stencil live plus two in flight, so NOTHING else is read from global memory and no
//     z-window lives in registers (which is what lets 20 warps fit the register file: the FP64 pipe needs >= 4
//     independent DFMAs in flight per scheduler, measured dependent-issue latency 8.6 cycles, issue interval 2.18);
//   * per tile row three warps work on plane k concurrently: the X warp computes the x-face fluxes of all fields, the
//     Y warp the y-face fluxes, the Z warp the z-face fluxes: 5 WENO reconstructions each, a balanced split;
//   * EVERY FACE FLUX IS COMPUTED ONCE: each thread computes the flux through the LOW x-/y-face (HIGH z-face) of its
//     control volumes; the other face comes from lane+1 (shuffle), from row+1 (shared memory; row TY is a ghost row
//     of Y warps only) or from the previous plane (register carried by the Z warp).  Diffusive fluxes ride along.
//   * who FINALISES (gathers the three directional parts of a field, adds the pointwise terms, applies the substage, stores)
//     depends on the instantiation (constexpr ZMOM in the kernel):
//       - LES (nonhydrostatic, WENO5 along z; C1, C2, C4): the X warp finalises EVERY field — the Z warp carries as many
//         reconstructions as the X warp, so it only publishes its z-divergences;
//       - hydrostatic (Centered(2) along z; C3): the Z warp has a fifth of the X warp's flux work, so the finalisation is
//         SPLIT: the Z warp finalises the MOMENTUM (gathers the x-divergences and y-fluxes, adds Coriolis and the pressure
//         gradient, accumulates the slow barotropic forcing (A19) when asked, applies the substage, stores) and the X warp the
//         TRACERS, both ONE PLANE LATE so that neither waits for the other's current plane (C3: 3.72 -> 2.79 ms); the
//         producer warp also diagnoses w from continuity (eq. 15) plane by plane when the step entry points ask for it.
//     All hand-offs go through shared memory with mbarrier publish/consume (no __syncthreads in the plane loop);
//   * tracers use the cancellation-free form (H1): flux anomalies relative to the cell's own value plus
//     c * div(u) with div(u) accumulated in double-double.
// Operators and citations are those of tend_percell.cu: (B2),(B3),(B8),(B9),(B21), eq. 6/8/9/17.
#include <cuda.h>
#include <cudaTypedefs.h>

#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <utility>

#include "ocn_internal.h"
#include "recon.cuh"

namespace {

using namespace ocn;

constexpr int NBUF = 8;          // TMA ring depth: planes k-2..k+3 live + two in flight (power of two)
constexpr int NXB = 3;           // depth of the flux-exchange ring between the Y / Z warps and the X (combiner) warps
constexpr int MAXF = 3 + 3;      // u, v, w + up to 3 tracers in the fused instantiations

template <class Real>
struct FusedArgs {
  CUtensorMap tmap[MAXF];        // one 3-D tiled map per input field: dims (pitch, ny_pad, nz_pad), box (TW, TY+6, 1)
  GridDev g;
  ModelDev m;
  const Real *phy;
  Real *G[MAXF];
  // fused substage (A4) (FUSE_RK3 instantiations): q_new = q + (rk_a G - rk_b G_prev), rk_a = dt gamma, rk_b = dt zeta
  const Real *Gp[MAXF];          // previous-stage tendencies (read iff use_prev)
  Real *Qn[MAXF];                // the OTHER state buffer of the ping-pong pair (written on interior points)
  Real rk_a, rk_b;
  int xa_off, ya_off, za_off;    // array coordinates of logical (i,j,k) = (i + xa_off, j + ya_off, k + za_off)
  int kchunk;                    // planes per block along z
  int diag_w;                    // hydrostatic: w is NOT loaded; the producer warp diagnoses it from continuity, eq. (15), plane by plane
  // hydrostatic + fused substage: the slow barotropic forcing (A19) F = sum_k dz_c (f_a G - f_b G_prev) of u, v accumulated by the warps
  // that finalise the momentum (one z-chunk) and written to these planes; NULL: not wanted
  Real *FUo, *FVo;
  double f_a, f_b;
};

// ---- mbarrier / TMA primitives (PTX; SASS: SYNCS.*, UTMALDG) ------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint64_t *bar, uint32_t parity) {
  // try_wait with a suspend-time hint: the hardware parks the thread (no issue slots burnt) until the phase
  // completes or the hint (ns) elapses
  uint32_t done;
  asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\nselp.u32 %0, 1, 0, p;\n}\n"
               : "=r"(done) : "r"(smem_u32(bar)), "r"(parity), "r"(20000u) : "memory");
  return done != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  while (!mbar_try(bar, parity)) {}
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int x, int y, int z, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
      : "memory");
}

// per-thread asynchronous global -> shared copy of one element (SASS: LDGSTS), no register staging
__device__ __forceinline__ void cp_async_elem(double *dst, const double *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_elem(float *dst, const float *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void st_global(unsigned long long addr, double v) { asm volatile("st.global.f64 [%0], %1;" ::"l"(addr), "d"(v) : "memory"); }
__device__ __forceinline__ void st_global(unsigned long long addr, float v) { asm volatile("st.global.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ double shfl_down1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_down1(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// vel > 0 for the upwind selection.  For doubles the test is made on the high word in the integer pipe (a DSETP holds the
// FP64 pipe for two cycles, ocn_alu_probe): identical to `vel > 0` for +-0 and every normal number; a positive subnormal
// (< 2.3e-308) counts as not positive, which moves the flux vel * (...) by less than 1e-300; a NaN velocity gives a NaN flux
// on either side.
__device__ __forceinline__ bool is_pos(double v) { return __double2hiint(v) > 0; }
__device__ __forceinline__ bool is_pos(float v) { return v > 0.0f; }

template <class Real> struct TileGeom {
  static constexpr int TW = sizeof(Real) == 8 ? 38 : 40;   // box row: 37 columns (i0-3 .. i0+33) + start alignment slack; bytes % 16 == 0
};

template <class Real, int NT, int TY>
struct SmemLayout {
  static constexpr int NF = 3 + NT;
  static constexpr int TW = TileGeom<Real>::TW;
  static constexpr int TH = TY + 6;
  static constexpr int FS = ((TW * TH * (int)sizeof(Real) + 127) / 128) * 128 / (int)sizeof(Real);   // field stride (elements)
  static constexpr int PS = NF * FS;                                    // plane (slot) stride
  static constexpr int TILE_ELEMS = NBUF * PS;
  static constexpr int NY = NF + NT;                                    // y-published values per thread: momentum F; tracers F_hi, F_lo
  static constexpr int FY_SLOT = NY * (TY + 1) * 32;
  static constexpr int PZ_SLOT = NF * TY * 32;                          // [0..2]: momentum x-divergences (X -> Z); [3..]: tracer z-divergences (Z -> X)
  static constexpr int NBAR = 2 * NBUF + 4 * NXB;                       // full, empty; ypub, zpub, xpub, cons
  static constexpr size_t BYTES = (size_t)(TILE_ELEMS + NXB * (FY_SLOT + PZ_SLOT)) * sizeof(Real) + NBAR * sizeof(uint64_t) + 3 * MAXF * sizeof(unsigned long long);
  static constexpr uint32_t PLANE_BYTES = (uint32_t)(NF * TW * TH * sizeof(Real));
  static constexpr int PH_ELEMS = 3 * TY * 32;                          // hydrostatic: per-thread staging of p_hy(i,j), (i-1,j), (i,j-1) (cp.async)
  static constexpr int GP_ELEMS = NF * TY * 32;                         // FUSE_RK3: per-thread staging of G_prev (cp.async)
  static constexpr size_t bytes(bool hydro, bool fuse) {
    return BYTES + (size_t)((hydro ? PH_ELEMS : 0) + (fuse ? GP_ELEMS : 0)) * sizeof(Real);
  }
};

// Upwind-selected five-point stencils of N fields by ADDRESS selection (no value selects).  hi[n] is the offset (in
// `base`) of the element on the high side of the face (index m), step the element stride along the flux direction.
// Left-biased (vel > 0): (a..e) = q[m-3 .. m+1]; right-biased: the mirror image q[m+2 .. m-2]  (reading R3).
template <class Real, int N>
__device__ __forceinline__ void upwind_diffs(const Real *base, const int (&hi)[N], int step, const Real (&vel)[N], Real (&d1)[N],
                                             Real (&d2)[N], Real (&d3)[N], Real (&d4)[N], Real (&cc)[N]) {
#pragma unroll
  for (int n = 0; n < N; ++n) {
    const bool pos = is_pos(vel[n]);
    const int s = pos ? step : -step;
    const Real *c = base + (pos ? hi[n] - step : hi[n]);
    const Real qa = c[-2 * s], qb = c[-s], qc = c[0], qd = c[s], qe = c[2 * s];
    d1[n] = qb - qa; d2[n] = qc - qb; d3[n] = qd - qc; d4[n] = qe - qd;
    cc[n] = qc;
  }
}
// the same for N fields advected by ONE velocity (tracers): fields are `fs` elements apart
template <class Real, int N>
__device__ __forceinline__ void upwind_diffs_shared(const Real *hi0, int fs, int step, Real vel, Real (&d1)[N], Real (&d2)[N],
                                                    Real (&d3)[N], Real (&d4)[N], Real (&cc)[N]) {
  const bool pos = is_pos(vel);
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
// along z: po[0..5] are the offsets of this thread's element in the planes m-3 .. m+2 of the ring
template <class Real, int N>
__device__ __forceinline__ void upwind_diffs_z(const Real *base, const int (&po)[6], const int (&fo)[N], const Real (&vel)[N],
                                               Real (&d1)[N], Real (&d2)[N], Real (&d3)[N], Real (&d4)[N], Real (&cc)[N]) {
#pragma unroll
  for (int n = 0; n < N; ++n) {
    const bool pos = is_pos(vel[n]);
    const Real *b = base + fo[n];
    const Real qa = b[pos ? po[0] : po[5]], qb = b[pos ? po[1] : po[4]], qc = b[pos ? po[2] : po[3]];
    const Real qd = b[pos ? po[3] : po[2]], qe = b[pos ? po[4] : po[1]];
    d1[n] = qb - qa; d2[n] = qc - qb; d3[n] = qd - qc; d4[n] = qe - qd;
    cc[n] = qc;
  }
}
template <class Real, int N>
__device__ __forceinline__ void upwind_diffs_z_shared(const Real *base, const int (&po)[6], int fs, Real vel, Real (&d1)[N],
                                                      Real (&d2)[N], Real (&d3)[N], Real (&d4)[N], Real (&cc)[N]) {
  const bool pos = is_pos(vel);
  const int ia = pos ? po[0] : po[5], ib = pos ? po[1] : po[4], ic = pos ? po[2] : po[3], id = pos ? po[3] : po[2], ie = pos ? po[4] : po[1];
#pragma unroll
  for (int n = 0; n < N; ++n) {
    const Real *b = base + n * fs;
    const Real qa = b[ia], qb = b[ib], qc = b[ic], qd = b[id], qe = b[ie];
    d1[n] = qb - qa; d2[n] = qc - qb; d3[n] = qd - qc; d4[n] = qe - qd;
    cc[n] = qc;
  }
}

// fp32 instantiations: upwind-selected five-point stencils by PREDICATED LOADS.  Left-biased (vel > 0): (a..e) = q[m-3 .. m+1]; right-biased: the mirror
// image q[m+2 .. m-2] (reading R3), m the element on the high side of the face.  Every value is a pair of shared-memory loads at
// IMMEDIATE offsets from one base register, one predicated on the sign of the advecting velocity and the other on its negation
// (SASS: @P LDS / @!P LDS; the nullified one makes no shared-memory access).  The first version selected the stencil by ADDRESS
// (base and stride flip with the sign): ~22 integer instructions per momentum reconstruction (SEL, IADD3, IMAD.IADD: ncu source
// view).  Used by the fp32 instantiations only (C4 9.43 -> 9.24 ms); in fp64 the ten 64-bit loads per reconstruction are not free
// beside FP64 work and the blocks cost spills (C2 6.09 -> 8.00 ms), so fp64 keeps the address-selected loads above.
//   a_lo: shared-memory byte address of element m-3 (x, y: along the stencil) of the FIRST field; OFF: element offset of the field.
template <int B0, int B1, int B2, int B3, int B4, int B5>
__device__ __forceinline__ void lds_upwind5(uint32_t a_lo, bool pos, double &qa, double &qb, double &qc, double &qd, double &qe) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.s32 p, %6, 0;\n"
      "@p ld.shared.f64 %0, [%5+%7];\n@!p ld.shared.f64 %0, [%5+%12];\n"
      "@p ld.shared.f64 %1, [%5+%8];\n@!p ld.shared.f64 %1, [%5+%11];\n"
      "@p ld.shared.f64 %2, [%5+%9];\n@!p ld.shared.f64 %2, [%5+%10];\n"
      "@p ld.shared.f64 %3, [%5+%10];\n@!p ld.shared.f64 %3, [%5+%9];\n"
      "@p ld.shared.f64 %4, [%5+%11];\n@!p ld.shared.f64 %4, [%5+%8];\n}\n"
      : "=d"(qa), "=d"(qb), "=d"(qc), "=d"(qd), "=d"(qe)
      : "r"(a_lo), "r"((int)pos), "n"(B0), "n"(B1), "n"(B2), "n"(B3), "n"(B4), "n"(B5)
      : "memory");
}
template <int B0, int B1, int B2, int B3, int B4, int B5>
__device__ __forceinline__ void lds_upwind5(uint32_t a_lo, bool pos, float &qa, float &qb, float &qc, float &qd, float &qe) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.s32 p, %6, 0;\n"
      "@p ld.shared.f32 %0, [%5+%7];\n@!p ld.shared.f32 %0, [%5+%12];\n"
      "@p ld.shared.f32 %1, [%5+%8];\n@!p ld.shared.f32 %1, [%5+%11];\n"
      "@p ld.shared.f32 %2, [%5+%9];\n@!p ld.shared.f32 %2, [%5+%10];\n"
      "@p ld.shared.f32 %3, [%5+%10];\n@!p ld.shared.f32 %3, [%5+%9];\n"
      "@p ld.shared.f32 %4, [%5+%11];\n@!p ld.shared.f32 %4, [%5+%8];\n}\n"
      : "=f"(qa), "=f"(qb), "=f"(qc), "=f"(qd), "=f"(qe)
      : "r"(a_lo), "r"((int)pos), "n"(B0), "n"(B1), "n"(B2), "n"(B3), "n"(B4), "n"(B5)
      : "memory");
}
// along z the six planes m-3 .. m+2 of the ring have runtime addresses a[0..5]; B: byte offset of the field
template <int B>
__device__ __forceinline__ void lds_upwind5_z(const uint32_t (&a)[6], bool pos, double &qa, double &qb, double &qc, double &qd, double &qe) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.s32 p, %11, 0;\n"
      "@p ld.shared.f64 %0, [%5+%12];\n@!p ld.shared.f64 %0, [%10+%12];\n"
      "@p ld.shared.f64 %1, [%6+%12];\n@!p ld.shared.f64 %1, [%9+%12];\n"
      "@p ld.shared.f64 %2, [%7+%12];\n@!p ld.shared.f64 %2, [%8+%12];\n"
      "@p ld.shared.f64 %3, [%8+%12];\n@!p ld.shared.f64 %3, [%7+%12];\n"
      "@p ld.shared.f64 %4, [%9+%12];\n@!p ld.shared.f64 %4, [%6+%12];\n}\n"
      : "=d"(qa), "=d"(qb), "=d"(qc), "=d"(qd), "=d"(qe)
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"((int)pos), "n"(B)
      : "memory");
}
template <int B>
__device__ __forceinline__ void lds_upwind5_z(const uint32_t (&a)[6], bool pos, float &qa, float &qb, float &qc, float &qd, float &qe) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.s32 p, %11, 0;\n"
      "@p ld.shared.f32 %0, [%5+%12];\n@!p ld.shared.f32 %0, [%10+%12];\n"
      "@p ld.shared.f32 %1, [%6+%12];\n@!p ld.shared.f32 %1, [%9+%12];\n"
      "@p ld.shared.f32 %2, [%7+%12];\n@!p ld.shared.f32 %2, [%8+%12];\n"
      "@p ld.shared.f32 %3, [%8+%12];\n@!p ld.shared.f32 %3, [%7+%12];\n"
      "@p ld.shared.f32 %4, [%9+%12];\n@!p ld.shared.f32 %4, [%6+%12];\n}\n"
      : "=f"(qa), "=f"(qb), "=f"(qc), "=f"(qd), "=f"(qe)
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"((int)pos), "n"(B)
      : "memory");
}

// field n (n = 0 .. N-1, FS elements apart, the first one at T0) advected by vel[n] along a direction of element stride S;
// T0 points at the element on the high side of the face (index m)
template <class Real, int B0, int S>
__device__ __forceinline__ void upwind_diffs_one_pl(uint32_t a_lo, Real vel, Real &d1, Real &d2, Real &d3, Real &d4, Real &cc) {
  constexpr int E = (int)sizeof(Real);
  Real qa, qb, qc, qd, qe;
  lds_upwind5<B0 * E, (B0 + S) * E, (B0 + 2 * S) * E, (B0 + 3 * S) * E, (B0 + 4 * S) * E, (B0 + 5 * S) * E>(a_lo, is_pos(vel), qa, qb, qc, qd, qe);
  d1 = qb - qa; d2 = qc - qb; d3 = qd - qc; d4 = qe - qd;
  cc = qc;
}
template <class Real, int N, int FS, int S, int... Is>
__device__ __forceinline__ void upwind_diffs_impl_pl(const Real *T0, const Real (&vel)[N], Real (&d1)[N], Real (&d2)[N], Real (&d3)[N],
                                                  Real (&d4)[N], Real (&cc)[N], std::integer_sequence<int, Is...>) {
  const uint32_t a_lo = smem_u32(T0 - 3 * S);
  (upwind_diffs_one_pl<Real, Is * FS, S>(a_lo, vel[Is], d1[Is], d2[Is], d3[Is], d4[Is], cc[Is]), ...);
}
template <class Real, int N, int FS, int S>
__device__ __forceinline__ void upwind_diffs_pl(const Real *T0, const Real (&vel)[N], Real (&d1)[N], Real (&d2)[N], Real (&d3)[N],
                                             Real (&d4)[N], Real (&cc)[N]) {
  upwind_diffs_impl_pl<Real, N, FS, S>(T0, vel, d1, d2, d3, d4, cc, std::make_integer_sequence<int, N>{});
}
// the same for N fields advected by ONE velocity (tracers)
template <class Real, int N, int FS, int S>
__device__ __forceinline__ void upwind_diffs_shared_pl(const Real *T0, Real vel, Real (&d1)[N], Real (&d2)[N], Real (&d3)[N], Real (&d4)[N],
                                                    Real (&cc)[N]) {
  Real v[N];
#pragma unroll
  for (int n = 0; n < N; ++n) v[n] = vel;
  upwind_diffs_impl_pl<Real, N, FS, S>(T0, v, d1, d2, d3, d4, cc, std::make_integer_sequence<int, N>{});
}
// along z: az[0..5] are the shared-memory byte addresses of this thread's element of field 0 in the planes m-3 .. m+2 of the ring;
// field n lies F0 + n FS elements further
template <class Real, int B>
__device__ __forceinline__ void upwind_diffs_z_one_pl(const uint32_t (&az)[6], Real vel, Real &d1, Real &d2, Real &d3, Real &d4, Real &cc) {
  Real qa, qb, qc, qd, qe;
  lds_upwind5_z<B * (int)sizeof(Real)>(az, is_pos(vel), qa, qb, qc, qd, qe);
  d1 = qb - qa; d2 = qc - qb; d3 = qd - qc; d4 = qe - qd;
  cc = qc;
}
template <class Real, int N, int FS, int F0, int... Is>
__device__ __forceinline__ void upwind_diffs_z_impl_pl(const uint32_t (&az)[6], const Real (&vel)[N], Real (&d1)[N], Real (&d2)[N],
                                                    Real (&d3)[N], Real (&d4)[N], Real (&cc)[N], std::integer_sequence<int, Is...>) {
  (upwind_diffs_z_one_pl<Real, F0 + Is * FS>(az, vel[Is], d1[Is], d2[Is], d3[Is], d4[Is], cc[Is]), ...);
}
template <class Real, int N, int FS, int F0>
__device__ __forceinline__ void upwind_diffs_z_pl(const uint32_t (&az)[6], const Real (&vel)[N], Real (&d1)[N], Real (&d2)[N], Real (&d3)[N],
                                               Real (&d4)[N], Real (&cc)[N]) {
  upwind_diffs_z_impl_pl<Real, N, FS, F0>(az, vel, d1, d2, d3, d4, cc, std::make_integer_sequence<int, N>{});
}
template <class Real, int N, int FS, int F0>
__device__ __forceinline__ void upwind_diffs_z_shared_pl(const uint32_t (&az)[6], Real vel, Real (&d1)[N], Real (&d2)[N], Real (&d3)[N],
                                                      Real (&d4)[N], Real (&cc)[N]) {
  Real v[N];
#pragma unroll
  for (int n = 0; n < N; ++n) v[n] = vel;
  upwind_diffs_z_impl_pl<Real, N, FS, F0>(az, v, d1, d2, d3, d4, cc, std::make_integer_sequence<int, N>{});
}

// Warps of a block: warp w < 3TY serves tile row w/3 in role w%3 (0: X + combine + store, 1: Y, 2: Z);
//                    warp 3TY is the ghost row of the Y role; warp 3TY+1 the TMA producer.
// Barriers: full[slot]/empty[slot] for the plane ring; ypub[s]/zpub[s]/xpub[s] "the Y / Z / X warps have published into
// exchange slot s", cons[s] "the X and the Z warps have consumed exchange slot s" (2 TY arrivals).
template <class Real, int NT, int SZ, bool HYDRO, int TY, int RK>
__global__ void __launch_bounds__(32 * (3 * TY + 2), 1) tend_fused_kernel(const __grid_constant__ FusedArgs<Real> a) {
  using SL = SmemLayout<Real, NT, TY>;
  constexpr int NF = SL::NF, TW = SL::TW, FS = SL::FS, PS = SL::PS;
  constexpr int FU = 0, FV = 1, FW = 2, FC = 3;
  constexpr int N = NT > 0 ? NT : 1;
  constexpr int NM = HYDRO ? 2 : 3;                      // momentum components that carry a tendency
  constexpr int IA = SZ == 5 ? S_WENO5 : S_CENTERED2;   // interpolation order of the velocity advecting through z-faces (R4)
  constexpr int ZLO = SZ == 5 ? 2 : 0, ZHI = SZ == 5 ? 3 : 1;   // planes k-ZLO .. k+ZHI are live while plane k is computed
  constexpr int XHI = (SZ == 5 && !HYDRO) ? 1 : 0;      // X / Y warps read up to plane k+1 (Centered(4) of u, v along z)
  constexpr int NR = TY + 1;
  constexpr bool FUSE_RK3 = RK != 0;                      // RK: 0 tendencies only, 1 fused substage without G_prev (zeta = 0), 2 with G_prev
  constexpr bool USE_PREV = RK == 2;
  // Who finalises the momentum tendencies (gathers the three directional parts, adds the pointwise terms, applies the
  // substage and stores)?  LES (WENO5 along z): the X warp finalises every field (the Z warp is as loaded as the X warp).
  // Hydrostatic (Centered(2) along z: the Z warp has a fifth of the X warp's work): the Z warp finalises u, v and the X
  // warp only the tracers, both ONE PLANE LATE so that neither waits for the other's current plane (C3: 3.72 -> 2.79 ms).
  constexpr bool ZMOM = HYDRO;
  constexpr int ZREL = ZMOM ? (ZLO > 1 ? ZLO : 1) : ZLO;  // the Z warps release plane k-ZREL after iteration k

  extern __shared__ __align__(1024) unsigned char smem_raw[];
  Real *tile = reinterpret_cast<Real *>(smem_raw);
  Real *fyb = tile + SL::TILE_ELEMS;                     // [NXB][NY][NR][32]
  Real *pzb = fyb + NXB * SL::FY_SLOT;                   // [NXB][NF][TY][32]
  uint64_t *full = reinterpret_cast<uint64_t *>(pzb + NXB * SL::PZ_SLOT);
  uint64_t *empty = full + NBUF;
  uint64_t *ypub = empty + NBUF, *zpub = ypub + NXB, *xpub = zpub + NXB, *cons = xpub + NXB;
  // output / G_prev base addresses, [field][G, Qn, Gp]: read with broadcast LDS in the store blocks.  (From the kernel
  // parameters every use costs an LDCU into a scarce uniform register plus its ~20-cycle latency on the in-order path of the
  // finalising warp: ncu showed the store block at 29 % of that warp's time.)
  unsigned long long *ptab = reinterpret_cast<unsigned long long *>(cons + NXB);
  Real *phb = reinterpret_cast<Real *>(ptab + 3 * MAXF);   // [3][TY][32], HYDRO only
  Real *gpb = phb + (HYDRO ? SL::PH_ELEMS : 0);            // [NF][TY][32], FUSE_RK3 only

  const GridDev &g = a.g;
  const ModelDev &m = a.m;
  const int lane = threadIdx.x, wid = threadIdx.y;
  const int i0 = blockIdx.x * 31 + 1, j0 = blockIdx.y * TY + 1;
  const int kc0 = 1 + blockIdx.z * a.kchunk;
  const int kc1 = min(kc0 + a.kchunk, g.Nz + 1);          // cell planes kc0 .. kc1-1
  const int pstart = kc0 - 1 - ZLO, pend = kc1 - 1 + ZHI; // planes streamed through the ring

  if (lane == 0 && wid == 0) {
    // full[b]: the producer's expect_tx arrival (+ the TMA bytes) and, when it also diagnoses w, its arrival after writing w's plane
    for (int b = 0; b < NBUF; ++b) { mbar_init(&full[b], (HYDRO && a.diag_w) ? 2 : 1); mbar_init(&empty[b], 3 * TY + 1); }
    for (int s = 0; s < NXB; ++s) { mbar_init(&ypub[s], NR); mbar_init(&zpub[s], TY); mbar_init(&xpub[s], TY); mbar_init(&cons[s], ZMOM ? 2 * TY : TY); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int f = 0; f < NF; ++f) {
      ptab[2 * f] = (unsigned long long)a.G[f];
      ptab[2 * f + 1] = (unsigned long long)a.Qn[f];
      ptab[2 * MAXF + f] = (unsigned long long)a.Gp[f];
    }
  }
  __syncthreads();

  constexpr int XA = 16 / (int)sizeof(Real);
  if (wid == 3 * TY + 1) {
    // ------------------------------------------------ producer warp: one lane feeds the TMA ring
    if constexpr (HYDRO) {
      if (a.diag_w) {
        // w FROM CONTINUITY INSIDE THE KERNEL (a2, eq. (15)): w[1] = 0, w[k+1] = w[k] - dz_c[k] (dx^-1 dx(u) + dy^-1 dy(v)),
        // the statements of compute_w_kernel (scan.cu) so that the values are bit-identical.  The block marches upwards and every
        // plane's u, v boxes pass through this warp's ring anyway, so the warp that otherwise only issues the TMA loads writes w's plane
        // of slot b itself — on the 32 x 7 columns the consumers read (their own cells, one to the left, one below) — and arrives on
        // full[b] a second time; the consumers are unchanged.  The launch is one z-chunk (the recurrence starts at the bottom); it
        // saves the separate scan (1.2 GB of traffic per substage at C3) and w's TMA load.
        const int tx0 = ((i0 - 3 + a.xa_off) / XA) * XA, ty0 = j0 - 3 + a.ya_off;
        const int xs_ = (i0 - 3 + a.xa_off) % XA;
        const Real rdx_ = Real(g.rdx), rdy_ = Real(g.rdy);
        // columns lane-1 = -1 .. 30 (one per lane) x rows -1 .. TY-1: what the cells that are stored (lanes 0 .. 30) read
        constexpr int WX = 32, WY = TY + 1, WN = WX * WY, WM = WY;
        for (int p = pstart, n = 0; p <= pend; ++p, ++n) {
          const int b = n & (NBUF - 1);
          if (n >= NBUF) mbar_wait(&empty[b], (uint32_t)(((n / NBUF) - 1) & 1));
          if (lane == 0) {
            mbar_expect_tx(&full[b], (uint32_t)((NF - 1) * TW * SL::TH * sizeof(Real)));
#pragma unroll
            for (int f = 0; f < NF; ++f)
              if (f != FW) tma_load_3d(tile + b * PS + f * FS, &a.tmap[f], tx0, ty0, p + a.za_off, &full[b]);
          }
          Real *wp = tile + b * PS + FW * FS;
          if (p <= 1) {                                   // w[1] = 0 at the bottom; the plane below is never read
#pragma unroll
            for (int m_ = 0; m_ < WM; ++m_) {
              const int t = lane + 32 * m_;
              if (t < WN) wp[(t / WX + 2) * TW + t % WX + 2 + xs_] = Real(0);
            }
          } else {
            const int bm = (n - 1) & (NBUF - 1);          // plane p-1: its u, v have landed once full[bm] completes (w[p-1] is ours)
            mbar_wait(&full[bm], (uint32_t)(((n - 1) / NBUF) & 1));
            const Real *um = tile + bm * PS + FU * FS, *vm = tile + bm * PS + FV * FS, *wm = tile + bm * PS + FW * FS;
            const Real dz = Real(g.dzc[g.zi(p - 1)]);
#pragma unroll
            for (int m_ = 0; m_ < WM; ++m_) {
              const int t = lane + 32 * m_;
              if (t < WN) {
                const int o = (t / WX + 2) * TW + t % WX + 2 + xs_;
                Real d = Real(0);
                d = ocn_fma(um[o + 1] - um[o], rdx_, d);
                d = ocn_fma(vm[o + TW] - vm[o], rdy_, d);
                wp[o] = ocn_fma(-dz, d, wm[o]);
              }
            }
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(&full[b]);
        }
        return;
      }
    }
    if (lane == 0) {
      // TMA needs the innermost start coordinate on a 16-byte boundary (measured: an odd fp64 x raises "illegal
      // instruction" on sm_100a): start the box at the aligned column at or left of i0-3; the readers shift by xs.
      const int tx0 = ((i0 - 3 + a.xa_off) / XA) * XA, ty0 = j0 - 3 + a.ya_off;
      for (int p = pstart, n = 0; p <= pend; ++p, ++n) {
        const int b = n & (NBUF - 1);
        if (n >= NBUF) mbar_wait(&empty[b], (uint32_t)(((n / NBUF) - 1) & 1));
        mbar_expect_tx(&full[b], SL::PLANE_BYTES);
#pragma unroll
        for (int f = 0; f < NF; ++f) tma_load_3d(tile + b * PS + f * FS, &a.tmap[f], tx0, ty0, p + a.za_off, &full[b]);
      }
    }
    return;
  }

  const int xs = (i0 - 3 + a.xa_off) % XA;
  const Real eps4 = Real(4.0 * m.weno_eps);
  const Real nu = Real(m.nu);
  const Real nuz = Real(m.nu_z);   // N3: the vertical part is treated implicitly (A2),(A8)
  // -kappa per tracer.  fp32 grids: converted ONCE (an F2F.F32.F64 per use and plane is a quarter-rate instruction on the
  // path of every role); fp64: the constant-bank operand is free, a register copy would only add pressure.
  Real nkap_h[N], nkap_z[N];
  if constexpr (sizeof(Real) == 4) {
#pragma unroll
    for (int t = 0; t < N; ++t) { nkap_h[t] = Real(-m.kappa[t]); nkap_z[t] = Real(-m.kappa_z[t]); }
  }
  auto NKH = [&](int t) -> Real { if constexpr (sizeof(Real) == 4) return nkap_h[t]; else return Real(-m.kappa[t]); };
  auto NKZ = [&](int t) -> Real { if constexpr (sizeof(Real) == 4) return nkap_z[t]; else return Real(-m.kappa_z[t]); };
  // store G (and the new state) of field f at byte offset ob: one 16-byte broadcast LDS for the two base addresses
  auto store_G = [&](int f, unsigned long long ob, Real Gf) {
    const ulonglong2 b = *reinterpret_cast<const ulonglong2 *>(ptab + 2 * f);
    st_global(b.x + ob, Gf);
  };
  auto store_GQ = [&](int f, unsigned long long ob, Real Gf, Real qn) {
    const ulonglong2 b = *reinterpret_cast<const ulonglong2 *>(ptab + 2 * f);
    st_global(b.x + ob, Gf);
    st_global(b.y + ob, qn);
  };
  auto PP = [&](int f, unsigned long long ob) { return reinterpret_cast<const Real *>(ptab[2 * MAXF + f] + ob); };   // Gp[f] + o
  auto PB = [&](int p) { return ((p - pstart) & (NBUF - 1)) * PS; };                     // ring offset of plane p
  auto wait_plane = [&](int p) { mbar_wait(&full[(p - pstart) & (NBUF - 1)], (uint32_t)(((p - pstart) / NBUF) & 1)); };
  auto release_plane = [&](int p) { if (lane == 0) mbar_arrive(&empty[(p - pstart) & (NBUF - 1)]); };

  // Warp -> (role, row).  The kernel is ISSUE-bound (a DFMA holds a scheduler's issue port for 2.18 cycles,
  // anything else for 1), so a plane takes as long as the most loaded of the four schedulers (warp % 4) needs to issue
  // its warps' instructions.  The X role is the heaviest (it also combines, stores and applies the substage), and
  // scheduler 3 hosts only four compute warps beside the idle producer: with TY = 6 it gets four X warps, schedulers
  // 0 and 1 get {X, Y, Y, Z, Z} and scheduler 2 {Y, Y, Y, Z, Z}.  Other TY: roles interleaved over the warp index.
  int role, wrow;                                      // role 0 = X, 1 = Y (row TY = ghost row), 2 = Z
  if constexpr (TY == 6) {
    //                  wid:  0  1  2  3  4  5  6  7  8  9 10 11 12 13 14 15 16 17 18
    constexpr int R[19] = {0, 0, 1, 0, 1, 1, 1, 0, 1, 1, 1, 0, 2, 2, 2, 0, 2, 2, 2};
    constexpr int W[19] = {4, 5, 0, 0, 1, 2, 3, 1, 4, 5, 6, 2, 0, 1, 2, 3, 3, 4, 5};
    role = 0; wrow = 0;
#pragma unroll
    for (int t = 0; t < 19; ++t)
      if (wid == t) { role = R[t]; wrow = W[t]; }
  } else {
    role = wid == 3 * TY ? 1 : wid % 3;
    wrow = wid == 3 * TY ? TY : wid / 3;
  }
  if (role == 0) {
    // =============================================================================== X warps: x-fluxes + combine
    const int row = wrow, i = i0 + lane, j = j0 + row;
    const int pos0 = (row + 3) * TW + lane + 3 + xs;
    const bool can_store = lane < 31 && i <= g.Nx && j <= g.Ny;
    const Real rdx = Real(g.rdx), rdy = Real(g.rdy);
    if constexpr (ZMOM) {
      long long o = g.idx(min(i, g.Nx), min(j, g.Ny), kc0);
      Real um2 = Real(0), um1 = Real(0);                 // u(k-2), u(k-1) of this column (Centered(4) along z), carried
      Real accp[N];                                      // x-divergences of the tracers of the PREVIOUS plane (deferred finalisation)
  #pragma unroll
      for (int t = 0; t < N; ++t) accp[t] = Real(0);
      // Finalise the tracers of plane kp (iteration np, element offset op): x-part (carried) + z-part (published by the Z warp)
      // - y-difference (published by the Y warps), substage, store.  It runs ONE PLANE LATE, after the x-fluxes of the next
      // plane have been published, so that the X and the Z warps never wait for each other's current plane.
      auto finalize_tracers = [&](int kp, int np, long long op) {
        const int sp = np % NXB;
        const uint32_t php = (uint32_t)((np / NXB) & 1);
        mbar_wait(&ypub[sp], php);
        mbar_wait(&zpub[sp], php);
        const Real *fy = fyb + sp * SL::FY_SLOT + row * 32 + lane;
        const Real *pz = pzb + sp * SL::PZ_SLOT + row * 32 + lane;
        Real Gt[N];
  #pragma unroll
        for (int t = 0; t < NT; ++t)
          Gt[t] = accp[t] + (pz[(FC + t) * TY * 32] - (fy[(3 + 2 * t) * NR * 32 + 32] - fy[(3 + 2 * t + 1) * NR * 32]) * rdy);
        __syncwarp();
        if (lane == 0) mbar_arrive(&cons[sp]);
        if constexpr (FUSE_RK3) cp_async_wait_all();
        if (can_store) {
          const Real *Tp = tile + PB(kp) + pos0;
          const unsigned long long ob = (unsigned long long)op * sizeof(Real);
  #pragma unroll
          for (int t = 0; t < NT; ++t) {
            const int f = FC + t;
            if constexpr (FUSE_RK3) {
              const Real q = Tp[f * FS];
              store_GQ(f, ob, Gt[t], USE_PREV ? rk3_update(q, Gt[t], gpb[(f * TY + row) * 32 + lane], a.rk_a, a.rk_b) : rk3_update(q, Gt[t], a.rk_a));
            } else {
              store_G(f, ob, Gt[t]);
            }
          }
        }
        __syncwarp();
        release_plane(kp);
      };
      for (int k = kc0, n = 0; k < kc1; ++k, ++n, o += g.sz) {
        const int sx = n % NXB;
        if constexpr (FUSE_RK3 && NT > 0) {
          // fused substage: start fetching the previous-stage TRACER tendencies of the plane that is finalised at the end of
          // this iteration (global -> this thread's own shared-memory slots, no registers held)
          if (n > 0 && USE_PREV && can_store) {
  #pragma unroll
            for (int t = 0; t < NT; ++t) cp_async_elem(gpb + ((FC + t) * TY + row) * 32 + lane, PP(FC + t, (unsigned long long)(o - g.sz) * sizeof(Real)));
          }
        }
        for (int p = (n == 0 ? pstart : k + XHI); p <= k + XHI; ++p) wait_plane(p);
        if (n == 0) {
          if constexpr (XHI) { um2 = tile[PB(k - 2) + pos0 + FU * FS]; um1 = tile[PB(k - 1) + pos0 + FU * FS]; }
          __syncwarp();
          for (int p = pstart; p < kc0; ++p) release_plane(p);     // the planes below kc0 only served the carried values
        }
        const int pb = PB(k);
        const Real *T0 = tile + pb + pos0;
        const Real ui = T0[FU * FS];
        Real acc[NF];
        if constexpr (HYDRO) acc[FW] = Real(0);
        if constexpr (NT > 0) {
          // tracers: face velocity u(i,j,k) used directly (B3); anomalies relative to c(i-1) [for the cell on the left]
          // and to c(i) [for this cell] (H1); the diffusive flux -kappa dc/dx rides along
          Real d1[N], d2[N], d3[N], d4[N], cc[N], r[N];
          if constexpr (sizeof(Real) == 4) upwind_diffs_shared_pl<Real, N, FS, 1>(T0 + FC * FS, ui, d1, d2, d3, d4, cc);
          else upwind_diffs_shared<Real, N>(T0 + FC * FS, FS, 1, ui, d1, d2, d3, d4, cc);
          weno5z_anom_v<N>(d1, d2, d3, d4, eps4, r);
  #pragma unroll
          for (int t = 0; t < NT; ++t) {
            const Real cm = T0[(FC + t) * FS - 1], c0 = T0[(FC + t) * FS];
            const Real Fd = NKH(t) * (c0 - cm) * rdx;
            const Real Fhi = ui * (r[t] + (cc[t] - cm)) + Fd, Flo = ui * (r[t] + (cc[t] - c0)) + Fd;
            acc[FC + t] = -(shfl_down1(Fhi) - Flo) * rdx;
          }
        }
        {
          int hi[NM];
          Real vl[NM], d1[NM], d2[NM], d3[NM], d4[NM], cc[NM], r[NM];
          hi[FU] = pb + pos0 + FU * FS;                                                                   // u at the centre i-1 (m = i)
          vl[FU] = interp_adv<Real>(S_WENO5, T0[FU * FS - 2], T0[FU * FS - 1], ui, T0[FU * FS + 1]);
          hi[FV] = pb + pos0 + FV * FS;                                                                   // v along x at (i-1/2, j-1/2)
          vl[FV] = interp_adv<Real>(S_WENO5, T0[FU * FS - 2 * TW], T0[FU * FS - TW], ui, T0[FU * FS + TW]);   // u~ along y  (B21)
          if constexpr (!HYDRO) {
            hi[FW] = pb + pos0 + FW * FS;                                                                 // w along x at (i-1/2, k-1/2)
            vl[FW] = interp_adv<Real>(S_WENO5, um2, um1, ui, tile[PB(k + 1) + pos0 + FU * FS]);              // u~ along z
          }
          if constexpr (sizeof(Real) == 4) upwind_diffs_pl<Real, NM, FS, 1>(T0, vl, d1, d2, d3, d4, cc);
          else upwind_diffs<Real, NM>(tile, hi, 1, vl, d1, d2, d3, d4, cc);
          weno5z_anom_v<NM>(d1, d2, d3, d4, eps4, r);
  #pragma unroll
          for (int t = 0; t < NM; ++t) {
            const Real F = vl[t] * (r[t] + cc[t]) - nu * (T0[t * FS] - T0[t * FS - 1]) * rdx;
            acc[t] = -(shfl_down1(F) - F) * rdx;
          }
        }
        // ---- publish the momentum x-divergences for the Z warp of this row (exchange slot sx must have been consumed)
        if (n >= NXB) mbar_wait(&cons[sx], (uint32_t)(((n / NXB) - 1) & 1));
        Real *px = pzb + sx * SL::PZ_SLOT + row * 32 + lane;
  #pragma unroll
        for (int t = 0; t < NM; ++t) px[t * TY * 32] = acc[t];
        __syncwarp();
        if (lane == 0) mbar_arrive(&xpub[sx]);
        // ---- finalise the tracers of the previous plane, then carry this plane's x-parts
        if (n > 0) finalize_tracers(k - 1, n - 1, o - g.sz);
  #pragma unroll
        for (int t = 0; t < NT; ++t) accp[t] = acc[FC + t];
        um2 = um1; um1 = ui;
      }
      if (kc1 > kc0) {
        if constexpr (FUSE_RK3 && NT > 0) {
          if (kc1 - kc0 > 0 && USE_PREV && can_store) {
  #pragma unroll
            for (int t = 0; t < NT; ++t) cp_async_elem(gpb + ((FC + t) * TY + row) * 32 + lane, PP(FC + t, (unsigned long long)(o - g.sz) * sizeof(Real)));
          }
        }
        finalize_tracers(kc1 - 1, kc1 - 1 - kc0, o - g.sz);
      }
    } else {
      const Real fu = Real(m.f0 + m.beta * ((j - 0.5) * g.dy - m.y0));      // f at the u point (y_c[j]), R8
      const Real fv = Real(m.f0 + m.beta * ((j - 1.0) * g.dy - m.y0));      // f at the v point (y_f[j])
      const bool wall_u = g.topo[0] == OCN_BOUNDED && i == 1;
      const bool wall_v = g.topo[1] == OCN_BOUNDED && j == 1;
      long long o = g.idx(min(i, g.Nx), min(j, g.Ny), kc0);
      Real um2 = Real(0), um1 = Real(0);                 // u(k-2), u(k-1) of this column (Centered(4) along z), carried
      for (int k = kc0, n = 0; k < kc1; ++k, ++n, o += g.sz) {
        const int sx = n % NXB;
        const uint32_t phx = (uint32_t)((n / NXB) & 1);
        if constexpr (FUSE_RK3) {
          // fused substage: start fetching this plane's previous-stage tendencies now (global -> this thread's own
          // shared-memory slots, no registers held); they are read back after the flux work, ~one plane-time later
          if (USE_PREV && can_store) {
  #pragma unroll
            for (int f = 0; f < NF; ++f) {
              if (HYDRO && f == FW) continue;
              cp_async_elem(gpb + (f * TY + row) * 32 + lane, PP(f, (unsigned long long)o * sizeof(Real)));
            }
          }
        }
        for (int p = (n == 0 ? pstart : k + XHI); p <= k + XHI; ++p) wait_plane(p);
        if (n == 0) {
          if constexpr (XHI) { um2 = tile[PB(k - 2) + pos0 + FU * FS]; um1 = tile[PB(k - 1) + pos0 + FU * FS]; }
          __syncwarp();
          for (int p = pstart; p < kc0; ++p) release_plane(p);     // the planes below kc0 only served the carried values
        }
        const int pb = PB(k);
        const Real *T0 = tile + pb + pos0;
        const Real ui = T0[FU * FS], vj = T0[FV * FS];
        Real acc[NF];
        if constexpr (HYDRO) acc[FW] = Real(0);
        if constexpr (NT > 0) {
          // tracers: face velocity u(i,j,k) used directly (B3); anomalies relative to c(i-1) [for the cell on the left]
          // and to c(i) [for this cell] (H1); the diffusive flux -kappa dc/dx rides along
          Real d1[N], d2[N], d3[N], d4[N], cc[N], r[N];
          if constexpr (sizeof(Real) == 4) upwind_diffs_shared_pl<Real, N, FS, 1>(T0 + FC * FS, ui, d1, d2, d3, d4, cc);
          else upwind_diffs_shared<Real, N>(T0 + FC * FS, FS, 1, ui, d1, d2, d3, d4, cc);
          weno5z_anom_v<N>(d1, d2, d3, d4, eps4, r);
  #pragma unroll
          for (int t = 0; t < NT; ++t) {
            const Real cm = T0[(FC + t) * FS - 1], c0 = T0[(FC + t) * FS];
            const Real Fd = NKH(t) * (c0 - cm) * rdx;
            const Real Fhi = ui * (r[t] + (cc[t] - cm)) + Fd, Flo = ui * (r[t] + (cc[t] - c0)) + Fd;
            acc[FC + t] = -(shfl_down1(Fhi) - Flo) * rdx;
          }
        }
        {
          int hi[NM];
          Real vl[NM], d1[NM], d2[NM], d3[NM], d4[NM], cc[NM], r[NM];
          hi[FU] = pb + pos0 + FU * FS;                                                                   // u at the centre i-1 (m = i)
          vl[FU] = interp_adv<Real>(S_WENO5, T0[FU * FS - 2], T0[FU * FS - 1], ui, T0[FU * FS + 1]);
          hi[FV] = pb + pos0 + FV * FS;                                                                   // v along x at (i-1/2, j-1/2)
          vl[FV] = interp_adv<Real>(S_WENO5, T0[FU * FS - 2 * TW], T0[FU * FS - TW], ui, T0[FU * FS + TW]);   // u~ along y  (B21)
          if constexpr (!HYDRO) {
            hi[FW] = pb + pos0 + FW * FS;                                                                 // w along x at (i-1/2, k-1/2)
            vl[FW] = interp_adv<Real>(S_WENO5, um2, um1, ui, tile[PB(k + 1) + pos0 + FU * FS]);              // u~ along z
          }
          if constexpr (sizeof(Real) == 4) upwind_diffs_pl<Real, NM, FS, 1>(T0, vl, d1, d2, d3, d4, cc);
          else upwind_diffs<Real, NM>(tile, hi, 1, vl, d1, d2, d3, d4, cc);
          weno5z_anom_v<NM>(d1, d2, d3, d4, eps4, r);
  #pragma unroll
          for (int t = 0; t < NM; ++t) {
            const Real F = vl[t] * (r[t] + cc[t]) - nu * (T0[t * FS] - T0[t * FS - 1]) * rdx;
            acc[t] = -(shfl_down1(F) - F) * rdx;
          }
        }
        // Coriolis rides on the z-divergences published by the Z warp (balance: the X warp is the longest role)
        if (HYDRO && a.phy != nullptr) {
          const Real p0 = __ldg(a.phy + o);
          acc[FU] -= (p0 - __ldg(a.phy + o - 1)) * rdx;
          acc[FV] -= (p0 - __ldg(a.phy + o - g.sy)) * rdy;
        }
        // ---- gather the y-fluxes (rows r and r+1) and the z-divergences published by the Y and Z warps
        mbar_wait(&ypub[sx], phx);
        mbar_wait(&zpub[sx], phx);
        const Real *fy = fyb + sx * SL::FY_SLOT + row * 32 + lane;
        const Real *pz = pzb + sx * SL::PZ_SLOT + row * 32 + lane;
  #pragma unroll
        for (int t = 0; t < NM; ++t) acc[t] += pz[t * TY * 32] - (fy[t * NR * 32 + 32] - fy[t * NR * 32]) * rdy;
  #pragma unroll
        for (int t = 0; t < NT; ++t)
          acc[FC + t] += pz[(FC + t) * TY * 32] - (fy[(3 + 2 * t) * NR * 32 + 32] - fy[(3 + 2 * t + 1) * NR * 32]) * rdy;
        __syncwarp();
        if (lane == 0) mbar_arrive(&cons[sx]);
        if constexpr (FUSE_RK3) cp_async_wait_all();
        if (can_store) {
          const unsigned long long ob = (unsigned long long)o * sizeof(Real);
          const bool wall[3] = {wall_u, wall_v, g.topo[2] == OCN_BOUNDED && k == 1};
  #pragma unroll
          for (int f = 0; f < NF; ++f) {
            if (HYDRO && f == FW) continue;
            const bool wl = f < 3 && wall[f < 3 ? f : 0];
            const Real Gf = wl ? Real(0) : acc[f];            // wall faces of wall-normal velocities: G = 0, q untouched
            if constexpr (FUSE_RK3) {
              const Real q = T0[f * FS];
              const Real qn = USE_PREV ? rk3_update(q, Gf, gpb[(f * TY + row) * 32 + lane], a.rk_a, a.rk_b) : rk3_update(q, Gf, a.rk_a);
              store_GQ(f, ob, Gf, wl ? q : qn);
            } else {
              store_G(f, ob, Gf);
            }
          }
        }
        um2 = um1; um1 = ui;
        __syncwarp();
        release_plane(k);
      }
    }
  } else if (role == 1) {
    // =============================================================================== Y warps: y-fluxes
    const int row = wrow;                              // 0 .. TY (TY = ghost row: supplies the high face of row TY-1)
    const int pos0 = (row + 3) * TW + lane + 3 + xs;
    const Real rdy = Real(g.rdy), dyr = Real(g.dy);
    Real vm2 = Real(0), vm1 = Real(0);                 // v(k-2), v(k-1) of this column, carried
    for (int k = kc0, n = 0; k < kc1; ++k, ++n) {
      const int sy = n % NXB;
      for (int p = (n == 0 ? pstart : k + 1); p <= k + 1; ++p) wait_plane(p);   // plane k+1: w(k+1) of div(u), v~ along z
      if (n == 0) {
        if constexpr (XHI) { vm2 = tile[PB(k - 2) + pos0 + FV * FS]; vm1 = tile[PB(k - 1) + pos0 + FV * FS]; }
        __syncwarp();
        for (int p = pstart; p < kc0; ++p) release_plane(p);
      }
      if (n >= NXB) mbar_wait(&cons[sy], (uint32_t)(((n / NXB) - 1) & 1));
      const int pb = PB(k);
      const Real *T0 = tile + pb + pos0;
      Real *fy = fyb + sy * SL::FY_SLOT + row * 32 + lane;
      const Real vj = T0[FV * FS];
      if constexpr (NT > 0) {
        Real d1[N], d2[N], d3[N], d4[N], cc[N], r[N];
        if constexpr (sizeof(Real) == 4) upwind_diffs_shared_pl<Real, N, FS, TW>(T0 + FC * FS, vj, d1, d2, d3, d4, cc);
        else upwind_diffs_shared<Real, N>(T0 + FC * FS, FS, TW, vj, d1, d2, d3, d4, cc);
        weno5z_anom_v<N>(d1, d2, d3, d4, eps4, r);
        // div(u) of cell (i,j,k) in double-double: a rounding-level quantity that multiplies the large tracer mean (H1).
        // c * div(u) * dy rides on the published low-face flux (the X warp multiplies the y-difference by 1/dy).
        double Dsum = 0.0;
        if (row < TY) {
          const int zk = g.zi(k);
          const double rz = g.uniform_z ? g.rdz : g.rdzc[zk], rz_lo = g.uniform_z ? g.rdz_lo : g.rdzc_lo[zk];
          if constexpr (sizeof(Real) == 8) {
            double D = 0.0, Dlo = 0.0;
            dd_add_diff_scaled((double)T0[FU * FS + 1], (double)T0[FU * FS], g.rdx, g.rdx_lo, D, Dlo);
            dd_add_diff_scaled((double)T0[FV * FS + TW], (double)vj, g.rdy, g.rdy_lo, D, Dlo);
            dd_add_diff_scaled((double)tile[PB(k + 1) + pos0 + FW * FS], (double)T0[FW * FS], rz, rz_lo, D, Dlo);
            Dsum = D + Dlo;
          } else {
            // fp32 storage: the differences of two floats are exact in double and the sum of the three terms carries 29 guard
            // bits, so plain double already resolves div(u) far below the 2e-5 tolerance (57 -> 6 FP64 instructions)
            (void)rz_lo;
            const double dux = (double)T0[FU * FS + 1] - (double)T0[FU * FS], dvy = (double)T0[FV * FS + TW] - (double)vj;
            const double dwz = (double)tile[PB(k + 1) + pos0 + FW * FS] - (double)T0[FW * FS];
            Dsum = fma(dwz, rz, fma(dvy, g.rdy, dux * g.rdx));
          }
        }
#pragma unroll
        for (int t = 0; t < NT; ++t) {
          const Real cm = T0[(FC + t) * FS - TW], c0 = T0[(FC + t) * FS];
          const Real Fd = NKH(t) * (c0 - cm) * rdy;
          fy[(3 + 2 * t) * NR * 32] = vj * (r[t] + (cc[t] - cm)) + Fd;        // as the HIGH face of the cell below
          fy[(3 + 2 * t + 1) * NR * 32] = (vj * (r[t] + (cc[t] - c0)) + Fd) - Real((double)c0 * Dsum) * dyr;   // LOW face of this cell
        }
      }
      {
        int hi[NM];
        Real vl[NM], d1[NM], d2[NM], d3[NM], d4[NM], cc[NM], r[NM];
        hi[FU] = pb + pos0 + FU * FS;                                                                   // u along y at (i-1/2, j-1/2)
        vl[FU] = interp_adv<Real>(S_WENO5, T0[FV * FS - 2], T0[FV * FS - 1], vj, T0[FV * FS + 1]);      // v~ along x  (B21)
        hi[FV] = pb + pos0 + FV * FS;                                                                   // v at the centre j-1 (m = j)
        vl[FV] = interp_adv<Real>(S_WENO5, T0[FV * FS - 2 * TW], T0[FV * FS - TW], vj, T0[FV * FS + TW]);
        if constexpr (!HYDRO) {
          hi[FW] = pb + pos0 + FW * FS;                                                                 // w along y at (j-1/2, k-1/2)
          vl[FW] = interp_adv<Real>(S_WENO5, vm2, vm1, vj, tile[PB(k + 1) + FV * FS + pos0]);          // v~ along z
        }
        if constexpr (sizeof(Real) == 4) upwind_diffs_pl<Real, NM, FS, TW>(T0, vl, d1, d2, d3, d4, cc);
        else upwind_diffs<Real, NM>(tile, hi, TW, vl, d1, d2, d3, d4, cc);
        weno5z_anom_v<NM>(d1, d2, d3, d4, eps4, r);
#pragma unroll
        for (int t = 0; t < NM; ++t) fy[t * NR * 32] = vl[t] * (r[t] + cc[t]) - nu * (T0[t * FS] - T0[t * FS - TW]) * rdy;
      }
      vm2 = vm1; vm1 = vj;
      __syncwarp();
      if (lane == 0) mbar_arrive(&ypub[sy]);
      release_plane(k);
    }
  } else {
    // =============================================================================== Z warps: z-fluxes, c div(u), buoyancy
    const int row = wrow, i = i0 + lane, j = j0 + row;
    const int pos0 = (row + 3) * TW + lane + 3 + xs;
    const bool can_store = lane < 31 && i <= g.Nx && j <= g.Ny;
    const Real rdx = Real(g.rdx), rdy = Real(g.rdy);
    const Real fu = Real(m.f0 + m.beta * ((j - 0.5) * g.dy - m.y0));      // f at the u point (y_c[j]), R8
    const Real fv = Real(m.f0 + m.beta * ((j - 1.0) * g.dy - m.y0));      // f at the v point (y_f[j])
    const bool wall_u = g.topo[0] == OCN_BOUNDED && i == 1;
    const bool wall_v = g.topo[1] == OCN_BOUNDED && j == 1;
    long long o = g.idx(min(i, g.Nx), min(j, g.Ny), kc0);
    Real Fm[NM], Rp[N], Fdp[N], cp[N];                 // carried: fluxes through the low z-face of the next plane
#pragma unroll
    for (int t = 0; t < NM; ++t) Fm[t] = Real(0);
#pragma unroll
    for (int t = 0; t < N; ++t) { Rp[t] = Real(0); Fdp[t] = Real(0); cp[t] = Real(0); }
    Real wlo = Real(0);
    double bprev = 0.0;
    double Facc[2] = {0.0, 0.0};                       // (A19): column integrals of the slow forcing of u, v (a.FUo != NULL)
    Real outp[NM];                                     // z-parts of the momentum tendencies of the PREVIOUS plane (deferred finalisation)
#pragma unroll
    for (int t = 0; t < NM; ++t) outp[t] = Real(0);
    // Finalise the momentum of plane kp (iteration np, element offset op), one plane late (see the X warp):
    // x-divergence (published by the X warp) + Coriolis / pressure gradient + z-part (carried) - y-difference, substage, store.
    auto finalize_momentum = [&](int kp, int np, long long op) {
      const int sp = np % NXB;
      const uint32_t php = (uint32_t)((np / NXB) & 1);
      const Real *Tp = tile + PB(kp) + pos0;
      Real cor[2] = {Real(0), Real(0)};
      if (m.coriolis) {
        const Real vj = Tp[FV * FS], ui = Tp[FU * FS];
        cor[0] = fu * (Real(0.25) * ((Tp[FV * FS - 1] + vj) + (Tp[FV * FS + TW - 1] + Tp[FV * FS + TW])));
        cor[1] = -(fv * (Real(0.25) * ((Tp[FU * FS - TW] + Tp[FU * FS - TW + 1]) + (ui + Tp[FU * FS + 1]))));
      }
      if (HYDRO && a.phy != nullptr) {
        cp_async_wait_all();                                 // issued one iteration ago (also covers the G_prev staging)
        const Real p0 = phb[(0 * TY + row) * 32 + lane];
        if (can_store) {
          cor[0] -= (p0 - phb[(1 * TY + row) * 32 + lane]) * rdx;
          cor[1] -= (p0 - phb[(2 * TY + row) * 32 + lane]) * rdy;
        }
      }
      mbar_wait(&xpub[sp], php);
      mbar_wait(&ypub[sp], php);
      const Real *fy = fyb + sp * SL::FY_SLOT + row * 32 + lane;
      const Real *px = pzb + sp * SL::PZ_SLOT + row * 32 + lane;
      Real Gm[NM];
#pragma unroll
      for (int t = 0; t < NM; ++t) {
        Real v = px[t * TY * 32];
        if (t < 2) v += cor[t < 2 ? t : 0];
        Gm[t] = v + (outp[t] - (fy[t * NR * 32 + 32] - fy[t * NR * 32]) * rdy);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&cons[sp]);
      if constexpr (FUSE_RK3) cp_async_wait_all();
      if (can_store) {
        const unsigned long long ob = (unsigned long long)op * sizeof(Real);
        const bool wall[3] = {wall_u, wall_v, g.topo[2] == OCN_BOUNDED && kp == 1};
#pragma unroll
        for (int f = 0; f < NM; ++f) {
          const bool wl = wall[f];
          const Real Gf = wl ? Real(0) : Gm[f];            // wall faces of wall-normal velocities: G = 0, q untouched
          if constexpr (FUSE_RK3) {
            const Real q = Tp[f * FS];
            const Real qn = USE_PREV ? rk3_update(q, Gf, gpb[(f * TY + row) * 32 + lane], a.rk_a, a.rk_b) : rk3_update(q, Gf, a.rk_a);
            store_GQ(f, ob, Gf, wl ? q : qn);
            if constexpr (HYDRO) {
              if (a.FUo != nullptr && f < 2) {          // the statements of column_integral_kernel (barotropic.cu): bit-identical sums
                double qf = __dmul_rn(a.f_a, (double)Gf);
                if (USE_PREV) qf = __fma_rn(-a.f_b, (double)gpb[(f * TY + row) * 32 + lane], qf);
                Facc[f] = __fma_rn(g.dzc[g.zi(kp)], qf, Facc[f]);
              }
            }
          } else {
            store_G(f, ob, Gf);
          }
        }
      }
    };
    for (int kz = kc0 - 1; kz < kc1; ++kz) {
      const int n = kz - kc0;                          // -1 on the priming iteration (computes the fluxes through face kc0 only)
      if constexpr (ZMOM) {
        // prefetch what the finalisation of plane kz-1 (later in this iteration) reads from global memory, straight into this
        // thread's shared-memory slots: the hydrostatic pressure at (i,j), (i-1,j), (i,j-1) (ncu: the three __ldg sat on the Z
        // warp's in-order path, long scoreboard 2.3 per issue) and, with the fused substage, the previous-stage tendencies
        if (n >= 1 && can_store) {
          if (HYDRO && a.phy != nullptr) {
            const Real *ph = a.phy + (o - g.sz);
            cp_async_elem(phb + (0 * TY + row) * 32 + lane, ph);
            cp_async_elem(phb + (1 * TY + row) * 32 + lane, ph - 1);
            cp_async_elem(phb + (2 * TY + row) * 32 + lane, ph - g.sy);
          }
          if constexpr (FUSE_RK3) {
            if (USE_PREV) {
#pragma unroll
              for (int f = 0; f < NM; ++f) cp_async_elem(gpb + (f * TY + row) * 32 + lane, PP(f, (unsigned long long)(o - g.sz) * sizeof(Real)));
            }
          }
        }
      }
      for (int p = (kz == kc0 - 1 ? pstart : kz + ZHI); p <= kz + ZHI; ++p) wait_plane(p);
      const int zk = g.zi(kz);
      Real rdzc_k, rdzf_k, rdzf_kp;                    // 1/dz_c[k], 1/dz_f[k], 1/dz_f[k+1]
      if (g.uniform_z) { rdzc_k = rdzf_k = rdzf_kp = Real(g.rdz); }
      else { rdzc_k = Real(g.rdzc[zk]); rdzf_k = Real(g.rdzf[zk]); rdzf_kp = Real(g.rdzf[zk + 1]); }
      const Real *Tk = tile + PB(kz) + pos0, *Tk1 = tile + PB(kz + 1) + pos0;
      const Real wk1 = Tk1[FW * FS];                   // w at face kz+1
      int po[6];
      uint32_t az[6];                                  // fp32: shared-memory byte addresses of the six planes (predicated loads)
      if constexpr (SZ == 5) {
#pragma unroll
        for (int t = 0; t < 6; ++t) { po[t] = PB(kz - 2 + t) + pos0; az[t] = smem_u32(tile + po[t]); }
      }
      Real out[NF];
      // ---- tracers
      if constexpr (NT > 0) {
        Real Rhi[N];
        if constexpr (SZ == 5) {
          Real d1[N], d2[N], d3[N], d4[N], cc[N], r[N];
          if constexpr (sizeof(Real) == 4) upwind_diffs_z_shared_pl<Real, N, FS, FC * FS>(az, wk1, d1, d2, d3, d4, cc);
          else upwind_diffs_z_shared<Real, N>(tile + FC * FS, po, FS, wk1, d1, d2, d3, d4, cc);
          weno5z_anom_v<N>(d1, d2, d3, d4, eps4, r);
#pragma unroll
          for (int t = 0; t < NT; ++t) Rhi[t] = r[t] + (cc[t] - Tk[(FC + t) * FS]);
        } else {
#pragma unroll
          for (int t = 0; t < NT; ++t) Rhi[t] = Real(0.5) * (Tk1[(FC + t) * FS] - Tk[(FC + t) * FS]);     // Centered(2) (B4) minus c(k)
        }
#pragma unroll
        for (int t = 0; t < NT; ++t) {
          const Real ck = Tk[(FC + t) * FS], ck1 = Tk1[(FC + t) * FS];
          const Real Fd = NKZ(t) * (ck1 - ck) * rdzf_kp;
          const Real Fhi = wk1 * Rhi[t] + Fd;                                              // relative to c(k): high face of cell k
          const Real Flo = wlo * (Rp[t] + (cp[t] - ck)) + Fdp[t];                          // the carried face, re-based to c(k)
          out[FC + t] = -(Fhi - Flo) * rdzc_k;                                             // c div(u): added by the Y warp
          Rp[t] = Rhi[t]; Fdp[t] = Fd; cp[t] = ck;
        }
      }
      // ---- momentum
      {
        Real vl[NM], F[NM];
        vl[FU] = interp_adv<Real>(IA, Tk1[FW * FS - 2], Tk1[FW * FS - 1], wk1, Tk1[FW * FS + 1]);              // w~ along x at (i-1/2, k+1/2)
        vl[FV] = interp_adv<Real>(IA, Tk1[FW * FS - 2 * TW], Tk1[FW * FS - TW], wk1, Tk1[FW * FS + TW]);       // w~ along y at (j-1/2, k+1/2)
        if constexpr (SZ == 5) {
          if constexpr (!HYDRO) vl[FW] = interp_adv<Real>(IA, tile[po[1] + FW * FS], tile[po[2] + FW * FS], wk1, tile[po[4] + FW * FS]);   // centre k
          int fo[NM];
          Real d1[NM], d2[NM], d3[NM], d4[NM], cc[NM], r[NM];
#pragma unroll
          for (int t = 0; t < NM; ++t) fo[t] = t * FS;
          if constexpr (sizeof(Real) == 4) upwind_diffs_z_pl<Real, NM, FS, 0>(az, vl, d1, d2, d3, d4, cc);
          else upwind_diffs_z<Real, NM>(tile, po, fo, vl, d1, d2, d3, d4, cc);
          weno5z_anom_v<NM>(d1, d2, d3, d4, eps4, r);
#pragma unroll
          for (int t = 0; t < NM; ++t) F[t] = vl[t] * (r[t] + cc[t]);
        } else {
          F[FU] = vl[FU] * (Real(0.5) * (Tk[FU * FS] + Tk1[FU * FS]));
          F[FV] = vl[FV] * (Real(0.5) * (Tk[FV * FS] + Tk1[FV * FS]));
          if constexpr (!HYDRO) { const Real wz = Real(0.5) * (Tk[FW * FS] + wk1); F[FW] = wz * wz; }
        }
        F[FU] -= nuz * (Tk1[FU * FS] - Tk[FU * FS]) * rdzf_kp;
        F[FV] -= nuz * (Tk1[FV * FS] - Tk[FV * FS]) * rdzf_kp;
        out[FU] = -(F[FU] - Fm[FU]) * rdzc_k;
        out[FV] = -(F[FV] - Fm[FV]) * rdzc_k;
        if constexpr (!HYDRO) {
          F[FW] -= nuz * (wk1 - Tk[FW * FS]) * rdzc_k;                                      // w faces k, k+1 are dz_c[k] apart
          double bk = 0.0;
          if (m.buoyancy) {
            // b = g [alpha (T - Tref) - beta (S - Sref)]  (reading R9); T, S are tracers 0, 1 (fused_applicable)
            const double Ta = m.idx_T >= 0 ? (double)Tk[FC * FS] - g.Tref[zk] : 0.0;
            const double Sa = m.idx_S >= 0 ? (double)Tk[(FC + (NT > 1 ? 1 : 0)) * FS] - g.Sref[zk] : 0.0;
            bk = m.g * (m.alpha_T * Ta - m.beta_S * Sa);
          }
          out[FW] = -(F[FW] - Fm[FW]) * rdzf_k + Real(0.5 * (bprev + bk));                 // w control volume k is dz_f[k] thick
          bprev = bk;
        } else {
          out[FW] = Real(0);
        }
#pragma unroll
        for (int t = 0; t < NM; ++t) Fm[t] = F[t];
      }
      wlo = wk1;
      if (n >= 0) {
        const int sz_ = n % NXB;
        if constexpr (ZMOM) {
          // ---- publish the tracer z-divergences for the X warp of this row
          if (n >= NXB) mbar_wait(&cons[sz_], (uint32_t)(((n / NXB) - 1) & 1));
          Real *pz = pzb + sz_ * SL::PZ_SLOT + row * 32 + lane;
  #pragma unroll
          for (int t = 0; t < NT; ++t) pz[(FC + t) * TY * 32] = out[FC + t];
          __syncwarp();
          if (lane == 0) mbar_arrive(&zpub[sz_]);
          // ---- finalise the momentum of the previous plane, then carry this plane's z-parts
          if (n >= 1) finalize_momentum(kz - 1, n - 1, o - g.sz);
  #pragma unroll
          for (int t = 0; t < NM; ++t) outp[t] = out[t];
        } else {
          if (m.coriolis) {       // pointwise terms ride on the published z-parts
            const Real vj = Tk[FV * FS], ui = Tk[FU * FS];
            out[FU] += fu * (Real(0.25) * ((Tk[FV * FS - 1] + vj) + (Tk[FV * FS + TW - 1] + Tk[FV * FS + TW])));
            out[FV] -= fv * (Real(0.25) * ((Tk[FU * FS - TW] + Tk[FU * FS - TW + 1]) + (ui + Tk[FU * FS + 1])));
          }
          if (n >= NXB) mbar_wait(&cons[sz_], (uint32_t)(((n / NXB) - 1) & 1));
          Real *pz = pzb + sz_ * SL::PZ_SLOT + row * 32 + lane;
  #pragma unroll
          for (int f = 0; f < NF; ++f) {
            if (HYDRO && f == FW) continue;
            pz[f * TY * 32] = out[f];
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(&zpub[sz_]);
        }
        o += g.sz;
      }
      __syncwarp();
      // plane kz-1 stays live for the deferred finalisation (its state values and Coriolis neighbours are read there)
      if (kz - ZREL >= pstart) release_plane(kz - ZREL);
    }
    if (ZMOM && kc1 > kc0) {
      if (can_store) {
        if (HYDRO && a.phy != nullptr) {
          const Real *ph = a.phy + (o - g.sz);
          cp_async_elem(phb + (0 * TY + row) * 32 + lane, ph);
          cp_async_elem(phb + (1 * TY + row) * 32 + lane, ph - 1);
          cp_async_elem(phb + (2 * TY + row) * 32 + lane, ph - g.sy);
        }
        if constexpr (FUSE_RK3) {
          if (USE_PREV) {
#pragma unroll
            for (int f = 0; f < NM; ++f) cp_async_elem(gpb + (f * TY + row) * 32 + lane, PP(f, (unsigned long long)(o - g.sz) * sizeof(Real)));
          }
        }
      }
      finalize_momentum(kc1 - 1, kc1 - 1 - kc0, o - g.sz);
      if constexpr (HYDRO && FUSE_RK3) {
        if (a.FUo != nullptr && can_store) {               // one z-chunk: this thread has seen its whole column
          const long long op = g.idx(i, j, 1 - g.Hz);      // the 2-D plane of the grid layout
          a.FUo[op] = Real(Facc[0]);
          a.FVo[op] = Real(Facc[1]);
        }
      }
    }
  }
}

// ---- host side --------------------------------------------------------------------------------------------
PFN_cuTensorMapEncodeTiled_v12000 get_encode() { return reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(ocn_tensormap_encoder()); }

PFN_cuTensorMapEncodeTiled_v12000 get_encode_impl() {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(p);
  }
  return fn;
}

template <class Real, int NT, int SZ, bool HYDRO, int TY, int RK>
int launch_fused_t(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G,
                   const Rk3Fuse *rk, cudaStream_t s) {
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
  constexpr bool FUSE_RK3 = RK != 0;
  if (FUSE_RK3) {
    const void *gp[MAXF] = {rk->Gp.u, rk->Gp.v, rk->Gp.w, rk->Gp.c[0], rk->Gp.c[1], rk->Gp.c[2]};
    void *qn[MAXF] = {rk->Qn.u, rk->Qn.v, rk->Qn.w, rk->Qn.c[0], rk->Qn.c[1], rk->Qn.c[2]};
    for (int f = 0; f < 3 + NT; ++f) { a.Gp[f] = (const Real *)gp[f]; a.Qn[f] = (Real *)qn[f]; }
    a.rk_a = Real(rk->a); a.rk_b = Real(rk->b);
  }
  for (int f = 0; f < 3 + NT; ++f) {
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
  // z-chunks: one block per SM at a time, so the launch takes ceil(blocks / SMs) waves of (kchunk + priming) plane-times;
  // pick the chunk count that minimises that product (C1: 110 tiles -> 4 chunks of 16 planes = 2.97 waves instead of 3 chunks
  // = 2.23 waves rounded up to 3; C2-C4: thousands of tiles, 1 chunk).  Chunks of at least 8 planes: each one re-primes the
  // plane ring and the carried z-fluxes (~1.5 plane-times).
  int sms = 148;
  {
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (sms < 1) sms = 148;
  }
  int nch = 1;
  {
    const int tiles = nbx * nby, maxch = std::max(1, (g->Nz + 7) / 8);
    double best = 1e300;
    for (int c = 1; c <= maxch; ++c) {
      const int kc = (g->Nz + c - 1) / c, cc = (g->Nz + kc - 1) / kc;
      const double waves = (double)(((long long)tiles * cc + sms - 1) / sms);
      const double cost = waves * (kc + 1.5);
      if (cost < best * 0.999) { best = cost; nch = cc; }
    }
  }
  a.diag_w = (HYDRO && rk && rk->diag_w) ? 1 : 0;
  if (HYDRO && FUSE_RK3 && rk && rk->FU && rk->FV) { a.FUo = (Real *)rk->FU; a.FVo = (Real *)rk->FV; a.f_a = rk->f_a; a.f_b = rk->f_b; }
  if (a.diag_w || a.FUo) nch = 1;                 // the continuity recurrence / the column integrals span the column: one z-chunk
  a.kchunk = (g->Nz + nch - 1) / nch;
  nch = (g->Nz + a.kchunk - 1) / a.kchunk;
  auto kern = tend_fused_kernel<Real, NT, SZ, HYDRO, TY, RK>;
  constexpr size_t SMEM = SL::bytes(HYDRO, FUSE_RK3);
  static OcnPerDeviceOnce attr_once;
  if (attr_once.first()) {
    OCN_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM));
  }
  dim3 block(32, 3 * TY + 2, 1), grid(nbx, nby, nch);
  kern<<<grid, block, SMEM, s>>>(a);
  ocn_count_launch();
  return ocn_check_cuda(cudaGetLastError(), "tend_fused_kernel launch");
}

constexpr int TYD = 6;   // rows per tile

}  // namespace

void *ocn_tensormap_encoder() { return reinterpret_cast<void *>(get_encode_impl()); }

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

template <int RK>
static int dispatch_fused(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G,
                          const Rk3Fuse *rk, cudaStream_t s) {
  std::string why;
  if (!fused_applicable(g, m, &why)) return ocn_fail(OCN_ERR_UNSUPPORTED, "fused kernels not applicable: %s", why.c_str());
  const bool hyd = m.hydrostatic != 0;
  if (g->dtype == OCN_F64) {
    if (hyd) return launch_fused_t<double, 2, 2, true, TYD, RK>(g, m, st, phy, G, rk, s);
    return launch_fused_t<double, 2, 5, false, TYD, RK>(g, m, st, phy, G, rk, s);
  }
  if (m.n_tracers == 3) return launch_fused_t<float, 3, 5, false, TYD, RK>(g, m, st, phy, G, rk, s);
  return launch_fused_t<float, 2, 5, false, TYD, RK>(g, m, st, phy, G, rk, s);
}

int launch_tendencies_fused(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G,
                            cudaStream_t s) {
  return dispatch_fused<0>(g, m, st, phy, G, nullptr, s);
}

int launch_tendencies_rk3_fused(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy, const FieldsDev &G,
                                const Rk3Fuse &rk, cudaStream_t s) {
  return rk.use_prev ? dispatch_fused<2>(g, m, st, phy, G, &rk, s) : dispatch_fused<1>(g, m, st, phy, G, &rk, s);
}
