// ocn_internal.h — private declarations shared by the translation units of libocn.so.
// Nothing here is shared with oracle/ (the CPU oracle is independent test infrastructure).
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "../../include/ocn.h"

// ------------------------------------------------------------------------------------------------
// Device-side description of the grid (POD, passed by value to kernels).
// z metrics are double arrays indexed by zi(k) = k + Hz (k = 1-Hz .. Nz+Hz+1 all addressable, plus k-1).
// ------------------------------------------------------------------------------------------------
struct GridDev {
  int Nx, Ny, Nz;
  int Hx, Hy, Hz;
  int topo[3];
  long long sy, sz, off0;   // element strides and offset of interior (1,1,1)
  double dx, dy;
  double rdx, rdy;          // fl(1/dx), fl(1/dy)
  double rdx_lo, rdy_lo;    // 1/dx - rdx (double-double tail), for the compensated divergence
  int uniform_z;
  double dz, rdz, rdz_lo;   // valid when uniform_z
  const double *dzc;        // Δz_c[k]
  const double *dzf;        // Δz_f[k] = z_c[k] - z_c[k-1]
  const double *rdzc;       // fl(1/Δz_c[k])
  const double *rdzc_lo;    // double-double tail of 1/Δz_c[k]
  const double *rdzf;       // fl(1/Δz_f[k])
  const double *Tref;       // reference profiles, indexed like the metrics (0 when absent)
  const double *Sref;
  __host__ __device__ int zi(int k) const { return k + Hz; }
  __host__ __device__ long long idx(int i, int j, int k) const { return off0 + (i - 1) + (long long)(j - 1) * sy + (long long)(k - 1) * sz; }
};

// model terms as the kernels see them
struct ModelDev {
  int n_tracers, idx_T, idx_S;
  int adv[3];
  int momentum, hydrostatic;
  int coriolis, buoyancy;
  int vimplicit;            // N3: vertical diffusion is treated implicitly => dropped from the tendencies
  double weno_eps;
  double f0, beta, y0;
  double g, alpha_T, beta_S;
  double nu, kappa[OCN_MAX_TRACERS];
  double nu_z, kappa_z[OCN_MAX_TRACERS];   // the coefficients of the EXPLICIT vertical diffusion: 0 when vimplicit
};

struct FieldsDev {
  void *u, *v, *w;
  void *c[OCN_MAX_TRACERS];
};

struct ocn_grid {
  int Nx, Ny, Nz, H, Hx, Hy, Hz;
  int topo[3];
  int dtype;
  double dx, dy;
  int uniform_z;
  double dz_uniform;
  ocn_layout lay;
  int nzm;                 // length of every metric array
  double *d_metrics;       // device block: 5 metric arrays + 2 reference arrays, nzm each
  double *d_vdiff;         // device scratch of N3: Thomas pivots, 3 arrays of nzm per distinct (kz, z-location), <= 2 + OCN_MAX_TRACERS sets
  std::vector<double> h_dzc, h_dzf;
  mutable std::vector<double> h_Tref, h_Sref;   // host cache of the reference profiles last uploaded
  mutable bool ref_valid;
  unsigned long long id;   // unique per created grid: objects that keep a grid pointer (ocn_poisson) check it is still alive
  int ext_halo[3];         // 1: the halos along this axis come from the caller (multi-GPU slab exchange); ocn_fill_halos skips them
  int kernel;
  int diag;                // OCN_DIAG_* mask (ocn_grid_set_diag): reference / fallback kernels with identical results, part of the graph key
  int graphs;              // 1: the ocn_step* calls replay CUDA graphs (ocn_grid_set_graphs)
  mutable struct GraphCache *gcache;   // captured ocn_step* sequences, keyed by every argument (api.cu)
  GridDev dev;
};

// live-grid registry (api.cu): true while the grid created with this id has not been destroyed
bool ocn_grid_alive(const ocn_grid *g, unsigned long long id);
// the grid a Poisson solver was created for, NULL (with the error set) if that grid has been destroyed (pressure.cu)
const ocn_grid *ocn_poisson_grid(const ocn_poisson *ps, const char *who);
// field buffers must be aligned to ocn_layout.alignment_bytes (TMA base, 16-byte vector accesses): OCN_ERR_INVALID otherwise
int ocn_check_aligned(const char *who, const ocn_grid *g, const void *ptr, const char *what);
int ocn_check_aligned(const char *who, const ocn_grid *g, const FieldsDev &f, const char *what);
// one-time per-DEVICE set-up (cudaFuncSetAttribute): a process-wide flag would skip the other devices of a multi-GPU process
struct OcnPerDeviceOnce {
  bool done[64] = {};
  bool first() {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess) return true;
    d &= 63;
    if (done[d]) return false;
    done[d] = true;
    return true;
  }
};

// cuTensorMapEncodeTiled through the runtime's driver entry point (no -lcuda symbol needed at load time); NULL if unavailable.
// Returns a PFN_cuTensorMapEncodeTiled_v12000 as void* (tend_fused.cu).
void *ocn_tensormap_encoder();

// error plumbing ---------------------------------------------------------------------------------
int ocn_fail(int code, const char *fmt, ...);
int ocn_check_cuda(cudaError_t e, const char *what);
void ocn_count_launch(int n = 1);
#define OCN_CUDA(call)                                   \
  do {                                                   \
    int rc__ = ocn_check_cuda((call), #call);            \
    if (rc__ != OCN_OK) return rc__;                     \
  } while (0)

// first prognostic index of a face-located field along an axis (wall face 1 excluded on Bounded axes)
static inline __host__ __device__ int first_face(int topo) { return topo == OCN_BOUNDED ? 2 : 1; }

// launchers (one per .cu) ------------------------------------------------------------------------
int launch_fill_halos(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, cudaStream_t s);
// y-slab exchange: copy the H outermost interior rows of every field into / the halo rows out of a packed buffer
int launch_halo_pack_y(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, int side, void *buf, bool unpack, cudaStream_t s);
int launch_compute_w(const ocn_grid *g, const FieldsDev &st, cudaStream_t s);
int launch_compute_phy(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, void *phy, cudaStream_t s);
int launch_tendencies_percell(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy,
                              const FieldsDev &G, cudaStream_t s);
// WENO7 / WENO9 models (tend_hiorder.cu): any topology, Centered(2)/NONE on the other axes
static inline bool hiorder_model(const ModelDev &m) {
  for (int a = 0; a < 3; ++a)
    if (m.adv[a] == OCN_ADV_WENO7 || m.adv[a] == OCN_ADV_WENO9) return true;
  return false;
}
int launch_tendencies_hiorder(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy,
                              const FieldsDev &G, cudaStream_t s);
// returns OCN_ERR_UNSUPPORTED (without enqueuing anything) when the fused kernels do not cover the case
int launch_tendencies_fused(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy,
                            const FieldsDev &G, cudaStream_t s);
bool fused_applicable(const ocn_grid *g, const ModelDev &m, std::string *why);
// tendencies + (A4) substage in one pass: q_new = q + (a G - b G_prev) into the other buffer of a ping-pong pair
struct Rk3Fuse {
  double a, b;          // dt*gamma, dt*zeta
  bool use_prev;        // zeta != 0: G_prev is read
  bool diag_w = false;  // hydrostatic TMA-ring kernel: diagnose w from continuity inside the kernel instead of reading state.w
  // hydrostatic TMA-ring kernel: also accumulate the barotropic slow forcing (A19), F = sum_k dz_c (f_a G - f_b G_prev) of u and v,
  // into these planes (what ocn_barotropic_forcing computes); NULL: not wanted
  void *FU = nullptr, *FV = nullptr;
  double f_a = 0.0, f_b = 0.0;
  FieldsDev Gp, Qn;
};
int launch_tendencies_rk3_fused(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy,
                                const FieldsDev &G, const Rk3Fuse &rk, cudaStream_t s);
// WENO7/9 with the substage fused in (tend_hiorder.cu: staged marching, global-load marching or per-cell kernel)
bool hiorder_rk3_applicable(const ocn_grid *g, const ModelDev &m, std::string *why);
int launch_tendencies_rk3_hiorder(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy,
                                  const FieldsDev &G, const Rk3Fuse &rk, cudaStream_t s);
// the general per-cell kernel with the substage fused in (tend_percell.cu): every model below WENO7
int launch_tendencies_rk3_percell(const ocn_grid *g, const ModelDev &m, const FieldsDev &st, const void *phy,
                                  const FieldsDev &G, const Rk3Fuse &rk, cudaStream_t s);
// does ocn_tendencies_rk3 (tendencies + substage in one pass) apply to this grid and model?  Always, except where
// ocn_compute_tendencies itself refuses a WENO7/9 model (nonhydrostatic momentum on a stretched z axis)
static inline bool rk3_fusable(const ocn_grid *g, const ModelDev &m, std::string *why) {
  return hiorder_model(m) ? hiorder_rk3_applicable(g, m, why) : true;
}
// N3: (1 - dt d_z kz d_z) q_new = q per column for every prognostic field (vdiff.cu)
int launch_implicit_vdiff(const ocn_grid *g, const ModelDev &m, double dt, const FieldsDev &st, cudaStream_t s);
int launch_substage(const ocn_grid *g, const ModelDev &m, double gamma, double zeta, double dt, const FieldsDev &st,
                    const FieldsDev &G, const FieldsDev &Gp, cudaStream_t s);

// (A4) PAPER.md:799 on one point, with the rounding order fixed by intrinsics so that the stand-alone substage
// kernel (rk3.cu) and the substage fused into the tendency kernel (tend_fused.cu) give bit-identical states.
#ifdef __CUDACC__
// explicitly rounded fused multiply-add (no contraction choice left to the compiler) for arithmetic that two kernels must reproduce
// bit for bit (w from continuity: scan.cu and the producer warp of tend_fused.cu)
__device__ __forceinline__ double ocn_fma(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float ocn_fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double rk3_update(double q, double G, double a) { return __fma_rn(a, G, q); }
__device__ __forceinline__ float rk3_update(float q, float G, float a) { return __fmaf_rn(a, G, q); }
__device__ __forceinline__ double rk3_update(double q, double G, double Gp, double a, double b) {
  return __dadd_rn(q, __fma_rn(a, G, -__dmul_rn(b, Gp)));
}
__device__ __forceinline__ float rk3_update(float q, float G, float Gp, float a, float b) {
  return __fadd_rn(q, __fmaf_rn(a, G, -__fmul_rn(b, Gp)));
}
#endif
