/* ocn.h — C ABI of libocn.so: the B200 (sm_100a) hot path of arXiv 2502.14148 (Oceananigans).
 *
 * One RK3 substage of the structured finite-volume algorithm on a halo-padded Arakawa C-grid is
 *
 *     ocn_fill_halos            (PAPER.md:1078  "halo cells are updated before the computation of tendencies")
 *     [ocn_compute_w]           (eq. 15   w from continuity, hydrostatic model only)
 *     [ocn_compute_phy]         (eq. 14 / 817-822, eq. A6   hydrostatic pressure anomaly)
 *     ocn_compute_tendencies    (eq. 6, 361 eq. 9, 506 eq. 17; App. B2 eqs. B2-B9, B21)
 *     ocn_rk3_substage          (eq. A4)
 * or, fused into one pass over the state, ocn_tendencies_rk3 = the last two calls (ping-pong state buffers).
 *
 * Every pointer argument says whether it is HOST or DEVICE memory.  No call synchronises, allocates
 * device memory or launches on any stream other than the one passed in (`stream` is a cudaStream_t
 * cast to void*, NULL = the legacy default stream).  Every call returns OCN_OK or a negative error
 * code; argument errors are detected before anything is enqueued; the message is available from
 * ocn_last_error() (thread-local).  There is no CPU fallback: without a CUDA device every compute call
 * returns OCN_ERR_CUDA.
 *
 * Index convention ("Face indices are left of cell indices"): interior cells i=1..Nx,
 * j=1..Ny, k=1..Nz; face i lies at x_{i-1/2}.  Locations: tracers/pressure at ccc,
 * u at fcc, v at cfc, w at ccf.  A face-located field along a Bounded axis has N+1 faces; faces 1 and
 * N+1 are walls, face N+1 is stored in the first high-side halo slot.  Along a Flat axis N must be 1,
 * there is no halo and no term.
 *
 * Concurrency: a grid owns small per-call scratch on the device (Thomas pivots of ocn_implicit_vertical_diffusion, the reference
 * profiles), so calls that take the SAME grid must be issued on one stream and from one host thread at a time; different grids are
 * independent.
 *
 * The library reads no environment variable and keeps no global switch: the diagnostic kernel choices are per-grid flags
 * (ocn_grid_set_diag), part of the key a captured CUDA graph is looked up by.
 */
#ifndef OCN_H
#define OCN_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ocn_grid ocn_grid; /* opaque; owns small host+device metric arrays only */

enum { OCN_PERIODIC = 0, OCN_BOUNDED = 1, OCN_FLAT = 2 };
enum { OCN_F64 = 0, OCN_F32 = 1 };
enum { OCN_ADV_NONE = 0, OCN_ADV_UPWIND1 = 1, OCN_ADV_CENTERED2 = 2, OCN_ADV_WENO5 = 5, /* (B4),(B5),(B8) */
       OCN_ADV_WENO7 = 7, OCN_ADV_WENO9 = 9 }; /* WENO order 7, 9: halo >= 4, 5 */
enum { OCN_OK = 0, OCN_ERR_INVALID = -1, OCN_ERR_UNSUPPORTED = -2, OCN_ERR_NOMEM = -3, OCN_ERR_CUDA = -4 };
enum { OCN_KERNEL_AUTO = 0,    /* fused 2.5-D kernels where they apply, else the per-cell kernel          */
       OCN_KERNEL_PERCELL = 1, /* one thread per cell, global loads: every scheme/topology; the "before"  */
       OCN_KERNEL_FUSED = 2 }; /* shared-memory x-y tiles + register-sliding z (error if not applicable)  */
#define OCN_MAX_TRACERS 8

/* Create a rectilinear grid.
 *   Nx,Ny,Nz   interior cells (1 along a Flat axis);  halo  halo width H on every non-Flat axis
 *              (>= (order+1)/2 of the widest scheme used later; 3 for WENO5)
 *   dx,dy      uniform horizontal spacings (> 0)
 *   dz_c       HOST, Nz cell thicknesses bottom -> top (copied), or NULL => uniform dz_uniform
 *   topology   HOST, 3 ints OCN_PERIODIC/BOUNDED/FLAT for x,y,z;  dtype  OCN_F64 or OCN_F32 field storage
 * The surface is at z=0: z_f[Nz+1]=0, z_c[k] = (z_f[k]+z_f[k+1])/2 (listing 15).
 * Errors: OCN_ERR_INVALID (NULL out, N<1, N<halo on a Periodic axis, N!=1 on a Flat axis, spacing<=0, halo<1),
 *         OCN_ERR_NOMEM, OCN_ERR_CUDA (metric upload failed / no device). */
int ocn_grid_create(ocn_grid **out, int Nx, int Ny, int Nz, int halo, double dx, double dy, const double *dz_c,
                    double dz_uniform, const int topology[3], int dtype);
int ocn_grid_destroy(ocn_grid *g); /* NULL is allowed */

/* Field storage chosen by the library (row pitch and interior offset are aligned for 16-byte vector
 * access and for TMA).  Element (i,j,k), 1-based with halos at <=0 and >N, of EVERY field lives at
 *     offset0 + (i-1) + (j-1)*stride_y + (k-1)*stride_z            (x fastest)
 * The caller allocates n_alloc elements per field, base aligned to alignment_bytes, zero-initialised. */
typedef struct {
  long long nx_pad, ny_pad, nz_pad; /* padded logical extents incl. halos (N + 2H, or N on a Flat axis)   */
  long long stride_y, stride_z;     /* element strides (stride_x = 1)                                    */
  long long offset0;                /* element offset of interior (1,1,1)                                */
  long long n_alloc;                /* elements to allocate per field                                    */
  int hx, hy, hz;                   /* halo widths actually used (0 on Flat axes)                        */
  int alignment_bytes;              /* required base alignment (128)                                     */
} ocn_layout;
int ocn_grid_layout(const ocn_grid *g, ocn_layout *out);

/* CUDA graphs for ocn_step, ocn_step_fused and ocn_step_model (default: enabled).  A call sequence is identified by EVERY
 * argument (entry point, stream, n_substages, dt, the parameter struct with the contents of T_ref / S_ref, all field
 * pointers, p_hy, the option struct with the contents of bt_weights).  Its first call is enqueued kernel by kernel, its
 * second call is stream-captured, instantiated (host-side work, once) and launched, later calls are ONE cudaGraphLaunch —
 * same kernels, same arguments, bit-identical results; the launch gaps that dominate small grids (C0, C1) disappear
 * (SURVEY 8(f) closing note).  The legacy default stream (NULL), a stream that is already being captured by the caller and
 * any capture failure fall back to the kernel-by-kernel sequence.  At most 16 sequences are cached per grid (LRU).
 * A grid must be used from one host thread at a time. */
int ocn_grid_set_graphs(ocn_grid *g, int enable);
int ocn_grid_graph_replays(const ocn_grid *g, long long *out); /* HOST out: ocn_step* calls served by a graph launch so far */

/* Select the tendency kernel family for this grid (default OCN_KERNEL_AUTO). */
int ocn_grid_set_kernel(ocn_grid *g, int kernel);

/* Diagnostic switches of this grid (default 0): each bit selects a reference / fallback kernel whose results are identical to the
 * default's, so that those kernels stay under test and a caller can ask for their side effects.  The mask is part of the CUDA-graph
 * key: a sequence captured under one mask is never replayed under another.
 *     OCN_DIAG_HI_NOSTAGE        WENO7/9: the global-load marching kernel instead of the TMA-staged one
 *     OCN_DIAG_HALO_ELEMENTWISE  ocn_fill_halos: the per-element kernel instead of the row-wise one
 *     OCN_DIAG_BT_SINGLESTEP     ocn_barotropic_substeps: one launch per substep instead of four substeps per launch
 *     OCN_DIAG_W_SCAN            ocn_step_fused / ocn_step_model, hydrostatic: launch ocn_compute_w (and ocn_barotropic_forcing) instead
 *                                of computing w (and the slow forcing) inside the tendency kernel; state.w is then written every
 *                                substage (see ocn_step_writes_w)
 * Errors: OCN_ERR_INVALID (NULL grid, unknown bits). */
enum { OCN_DIAG_HI_NOSTAGE = 1, OCN_DIAG_HALO_ELEMENTWISE = 2, OCN_DIAG_BT_SINGLESTEP = 4, OCN_DIAG_W_SCAN = 8, OCN_DIAG_ALL = 15 };
int ocn_grid_set_diag(ocn_grid *g, unsigned mask);

/* DEVICE pointers, caller-owned, all with the grid's layout; NULL = field absent
 * (w when z is Flat or never needed, tracers beyond n_tracers).  The velocity component along a Flat axis does not exist
 * (SURVEY 8(c) c.1): the tendency calls ignore a buffer passed for it — it is neither read (no Coriolis partner, no advecting
 * velocity) nor given a tendency. */
typedef struct {
  void *u, *v, *w;
  void *c[OCN_MAX_TRACERS];
} ocn_fields;

/* Model terms ("the model is a choice of terms").  Plain data, HOST. */
typedef struct {
  int n_tracers, idx_T, idx_S;  /* idx_T / idx_S: which tracers are temperature / salinity; -1 => absent (both -1: no buoyancy) */
  int adv_x, adv_y, adv_z;      /* OCN_ADV_* per direction (C3: WENO5, WENO5, CENTERED2); NONE disables advection along it      */
  int momentum_prognostic;      /* 0 => prescribed velocities: tracer tendencies only, u,v,w never updated      */
  int hydrostatic;              /* 1 => no G_w; buoyancy enters through p_hy (eq. 14, 17); w must come from ocn_compute_w       */
  double weno_eps;              /* WENO-Z epsilon (1e-8); > 0 and, on the WENO axes, >= 1e-50 / 1e-38 / 1e-32 for WENO5 / 7 / 9 in
                                 * fp64 and >= 1e-30 in fp32 (OCN_ERR_INVALID below that): the weights are evaluated as products of the
                                 * r regularised indicators (fp64) or with flushed-denormal reciprocals (fp32) and would be 0/0 on a
                                 * constant stencil.  For the same reason field DIFFERENCES across a stencil must stay below ~1e12
                                 * (WENO9), 1e15 (WENO7), 1e20 (WENO5) in fp64 and tau/eps below ~1e19 in fp32 (overflow -> NaN). */
  double f0, beta_coriolis, y0; /* f = f0 + beta*(y - y0), y from the southern face j=1 (PAPER.md:409 FPlane, :60 beta-plane)    */
  double g, alpha_T, beta_S;    /* linear equation of state b = g[alpha_T (T-T_ref) - beta_S (S-S_ref)]      */
  const double *T_ref, *S_ref;  /* HOST, Nz reference values (bottom -> top) or NULL (= 0)                                        */
  double nu, kappa[OCN_MAX_TRACERS]; /* constant Laplacian viscosity / diffusivities (PAPER.md:340 eq. 8 row 1, :385)            */
  int implicit_vertical_diffusion; /* N3: 1 => VerticallyImplicitTimeDiscretization: the vertical part of
                                      nu lap / kappa lap is LEFT OUT of the tendencies and applied by
                                      ocn_implicit_vertical_diffusion after each substage; 0 => explicit (absorbed into G)   */
} ocn_params;

/* a1 — fill every halo element of u, v, w and the first n_tracers tracers in place: Periodic wrap;
 * Bounded + centre-located: even mirror (no-flux, PAPER.md:349-353 default BCs); Bounded + wall-normal
 * face-located: wall faces and everything beyond = 0 (impenetrable).  Edges and corners are filled.
 * hydrostatic=1: w is skipped (it is diagnosed, halos included, by ocn_compute_w).
 * Errors: OCN_ERR_INVALID (NULL grid/params/state, n_tracers out of range, a required field NULL). */
int ocn_fill_halos(const ocn_grid *g, const ocn_params *p, ocn_fields *state, void *stream);

/* Multi-GPU y-slabs (App. C "slab and pencil decomposition ... halo cells are updated before the
 * computation of tendencies").  One process per GPU owns a slab of Ny_local rows of a grid that is PERIODIC in y (never split
 * z: the column scans stay local); its ocn_grid is created with Ny = Ny_local and marked
 *     ocn_grid_set_external_halo(g, 1, 1)     => ocn_fill_halos fills the x and z halos only and leaves every row j < 1, j > Ny alone.
 * One exchange step per halo fill: after ocn_fill_halos (so the packed rows carry their x / z halo elements and the corners
 * come out consistent) each rank packs its H outermost interior rows of a side,
 *     ocn_halo_pack_y(side)    rows 1..H (side 0) or Ny-H+1..Ny (side 1) of u, v, [w], tracers 0..n_tracers-1, all padded levels
 * sends them to the neighbour on that side (NCCL send/recv or peer copies — the transport is the caller's; the Python binding
 * `paper_2502_14148_b200.slab.YSlabs` uses torch.distributed P2P), and writes what it receives into its halo rows
 *     ocn_halo_unpack_y(side)  rows 1-H..0 (side 0, data = the SOUTH neighbour's side-1 pack) or Ny+1..Ny+H (side 1).
 * buf: DEVICE, 16-byte aligned, ocn_halo_slab_elems(g, p) elements of the grid's dtype, layout
 * [field][padded level][H rows][stride_y]: per field and level the rows are contiguous in the layout, so packing is pure
 * 16-byte-vector copying.  No reduction or all-to-all is needed on this path.
 * What a slab grid may be used with: the call-by-call hot path (ocn_fill_halos, pack / unpack, ocn_compute_w / _phy,
 * ocn_compute_tendencies, ocn_rk3_substage, ocn_tendencies_rk3, ocn_implicit_vertical_diffusion and the column integrals of N4).
 * ocn_step, ocn_step_fused, ocn_step_model, ocn_step_host (no exchange hook between their halo fill and their tendencies), the
 * FFT pressure solver (ocn_poisson_create / _solve, ocn_pressure_*) and ocn_barotropic_substeps (both would wrap y inside the
 * local slab) return OCN_ERR_UNSUPPORTED on it.
 * Coriolis on a slab: the kernels evaluate f = f0 + beta_coriolis (y_j - y0) from the LOCAL row index j = 1..Ny_local, so a rank
 * whose first row is global row j0 + 1 must pass y0_local = y0 - j0 * dy in its ocn_params (slab.YSlabs.local_params does).
 * Errors: OCN_ERR_UNSUPPORTED (axis != 1, y not Periodic), OCN_ERR_INVALID (NULLs, side, alignment, Ny < halo). */
int ocn_grid_set_external_halo(ocn_grid *g, int axis, int external);
long long ocn_halo_slab_elems(const ocn_grid *g, const ocn_params *p); /* < 0 on invalid arguments */
int ocn_halo_pack_y(const ocn_grid *g, const ocn_params *p, const ocn_fields *state, int side, void *buf, void *stream);
int ocn_halo_unpack_y(const ocn_grid *g, const ocn_params *p, ocn_fields *state, int side, const void *buf, void *stream);

/* a2 — eq. (15): w[i,j,1] = 0; w[k+1] = w[k] - dz_c[k] * (dx^-1 (u[i+1]-u[i]) + dy^-1 (v[j+1]-v[j])) for every
 * column whose u[i+1], v[j+1] exist in the padded arrays (halos of u,v must be filled).  Writes state->w
 * levels 1..Nz+1; w[Nz+1] is whatever continuity gives (linearised free surface).
 * Errors: OCN_ERR_INVALID (NULL, z Flat). */
int ocn_compute_w(const ocn_grid *g, ocn_fields *state, void *stream);

/* a3 — eq. (14): p[Nz] = -b[Nz] dz_c[Nz]/2; p[k-1] = p[k] - (b[k]+b[k-1])/2 * dz_f[k] over all padded columns
 * (tracer halos must be filled).  p_hy: DEVICE, grid layout, written.  Errors: OCN_ERR_INVALID. */
int ocn_compute_phy(const ocn_grid *g, const ocn_params *p, const ocn_fields *state, void *p_hy, void *stream);

/* a4-a10 — all tendencies of one substage into G (DEVICE, grid layout, interior points written; wall faces
 * of wall-normal velocities get 0; halos of G are not touched):
 *   tracers  G_c = -(1/V)[dx(Ax u [c]x) + dy(Ay v [c]y) + dz(Az w [c]z)] + kappa lap(c)              (B2),(B3)
 *   momentum flux-form advection with upwind-reconstructed advected and centred advecting velocity (B21),
 *            Coriolis with 4-point C-grid averages, buoyancy (+b in G_w, or -grad_h p_hy when hydrostatic),
 *            nu lap(.)                                                                            eq. 6, 17
 *   reconstruction [.]: UpwindBiased(1) (B5), Centered(2) (B4) or WENO5 with WENO-Z weights (B8),(B9).
 *   WENO7 / WENO9 (same construction at r = 4, 5; advecting velocities by Centered(6) / Centered(8)): every non-Flat
 *   axis must use the SAME WENO order or Centered(2)/NONE; halo >= (order+1)/2; run by the general high-order kernel.
 * state halos must be filled.  p_hy: DEVICE or NULL (required iff hydrostatic && buoyancy active).
 * G must not alias state.  Errors: OCN_ERR_INVALID (NULL / missing field / halo < 3 with WENO5),
 * OCN_ERR_UNSUPPORTED (WENO along a stretched axis; mixed WENO orders; OCN_KERNEL_FUSED forced where it does not apply). */
int ocn_compute_tendencies(const ocn_grid *g, const ocn_params *p, const ocn_fields *state, const void *p_hy,
                           ocn_fields *G, void *stream);

/* a11 — eq. (A4): q <- q + dt (gamma^m G^m - zeta^m G^{m-1}), gamma=(8/15,5/12,3/4), zeta=(0,17/60,5/12), on the
 * interior non-wall points of every prognostic field (u,v[,w] if momentum_prognostic; all tracers).
 * stage in {1,2,3}; G_prev may be NULL at stage 1 (zeta^1 = 0: self-starting).  The caller rotates G / G_prev.
 * Errors: OCN_ERR_INVALID (stage, NULLs). */
int ocn_rk3_substage(const ocn_grid *g, const ocn_params *p, int stage, double dt, ocn_fields *state,
                     const ocn_fields *G, const ocn_fields *G_prev, void *stream);

/* the same update with free coefficients: gamma=1, zeta=0 is forward Euler (used by the exact-shift test). */
int ocn_substage(const ocn_grid *g, const ocn_params *p, double gamma, double zeta, double dt, ocn_fields *state,
                 const ocn_fields *G, const ocn_fields *G_prev, void *stream);

/* a4-a11 in ONE pass (the B200 path of a substage): the tendencies of `state` are written to G as
 * by ocn_compute_tendencies AND the substage (A4) is applied on the fly into the OTHER buffer of a ping-pong pair,
 *     state_new = state + dt (gamma^m G - zeta^m G_prev)        on the interior non-wall points of every prognostic field
 * (wall faces of wall-normal velocities: state_new = state), bit-identical to ocn_compute_tendencies followed by
 * ocn_rk3_substage.  In place is impossible (neighbouring cells still read the old values), hence state_new:
 * DEVICE, grid layout, every prognostic field present and distinct from state, G and G_prev; its halos are NOT
 * written (the next ocn_fill_halos does that); fields that carry no tendency (w when hydrostatic; u, v, w when the velocities are
 * prescribed) are not written and are to be shared between the two structs.  G_prev may be NULL at stage 1.
 * Covered: every model ocn_compute_tendencies accepts, with the kernel that call would pick — the TMA-ring kernel of tend_fused.cu
 * where it applies (WENO5 in x, y on 3-D grids with prognostic momentum: nonhydrostatic with WENO5 along a uniform z and 2 tracers
 * (fp64) / 2 or 3 tracers (fp32), or hydrostatic with Centered(2) along z and 2 tracers), else the general per-cell kernel; WENO7 /
 * WENO9: the TMA-staged marching kernel of tend_hiorder.cu (3-D grids, up to 3 tracers), else the global-load marching kernel or
 * the per-cell high-order kernel.
 * Errors: as ocn_compute_tendencies / ocn_rk3_substage (incl. OCN_ERR_UNSUPPORTED for OCN_KERNEL_FUSED forced where it does not
 * apply). */
int ocn_tendencies_rk3(const ocn_grid *g, const ocn_params *p, int stage, double dt, const ocn_fields *state,
                       const void *p_hy, ocn_fields *G, const ocn_fields *G_prev, ocn_fields *state_new, void *stream);

/* Convenience: n_substages (1..3) consecutive substages m = 1..n of ONE time step on device-resident state:
 *   for m: ocn_fill_halos; [hydrostatic: ocn_compute_w; ocn_compute_phy if buoyancy]; ocn_compute_tendencies;
 *          ocn_rk3_substage(m); swap(G, G_prev)
 * exactly the call sequence above, enqueued on `stream`.  G and G_prev are caller-owned scratch (DEVICE, grid
 * layout, the same fields as the prognostic state); p_hy is DEVICE scratch, required iff hydrostatic with
 * buoyancy.  On return *G holds the tendencies of the last substage run if n_substages is odd, *G_prev otherwise
 * (the structs themselves are not modified).  Errors: as the individual calls. */
int ocn_step(const ocn_grid *g, const ocn_params *p, int n_substages, double dt, ocn_fields *state, ocn_fields *G,
             ocn_fields *G_prev, void *p_hy, void *stream);

/* The same sequence with the fused tendency+substage pass:
 *   for m: ocn_fill_halos(cur); [hydrostatic: ocn_compute_w(cur); ocn_compute_phy]; ocn_tendencies_rk3(m, cur -> other);
 *          swap(cur, other); swap(G, G_prev)
 * starting with cur = state, other = state_alt (DEVICE, same fields as state; contents need not be initialised).
 * The updated state is in *state_alt if n_substages is odd (a full step: 3) and in *state if it is even; the
 * structs themselves are not modified.  Hydrostatic models on the TMA-ring kernel: the kernel diagnoses w from continuity
 * (eq. 15) itself, plane by plane, with the arithmetic of ocn_compute_w (bit-identical tendencies), so ocn_compute_w is NOT
 * launched and state.w is neither read nor written by ocn_step_fused / ocn_step_model — call ocn_compute_w when the diagnosed w
 * itself is wanted, ask ocn_step_writes_w whether this grid / model pair is such a case, or set OCN_DIAG_W_SCAN on the grid to
 * keep the ocn_compute_w launch (state.w then holds the w of the last substage's input state, as after ocn_step).
 * Errors: as ocn_tendencies_rk3 (OCN_ERR_UNSUPPORTED => use ocn_step). */
int ocn_step_fused(const ocn_grid *g, const ocn_params *p, int n_substages, double dt, ocn_fields *state,
                   ocn_fields *state_alt, ocn_fields *G, ocn_fields *G_prev, void *p_hy, void *stream);

/* Do ocn_step_fused / ocn_step_model write the diagnosed w (eq. 15) into state.w for this grid (its kernel and
 * diagnostic selection included) and model?  Returns 1 (ocn_compute_w is launched every substage), 0 (hydrostatic model on the
 * TMA-ring kernel: w lives only inside the tendency kernel, state.w keeps what the caller left there) or a negative error code
 * (OCN_ERR_INVALID: NULLs, invalid params).  Nonhydrostatic models: 1 (w is prognostic, always written).  No device work. */
int ocn_step_writes_w(const ocn_grid *g, const ocn_params *p);

/* One step from HOST memory (the end-to-end path): every non-NULL field of host_state (HOST pointers, pinned
 * recommended, n_alloc elements in the grid layout, halos may hold anything) is copied to the matching field of
 * dev_state (DEVICE, caller-owned), the step runs as ocn_step_fused when dev_state_alt is non-NULL and the fused
 * kernel covers the model, else as ocn_step, and every prognostic field is copied back into host_state.  All
 * copies are cudaMemcpyAsync on `stream`; the call does not synchronise.
 * Errors: OCN_ERR_INVALID (a field present on one side only), else as ocn_step. */
int ocn_step_host(const ocn_grid *g, const ocn_params *p, int n_substages, double dt, ocn_fields *host_state,
                  ocn_fields *dev_state, ocn_fields *dev_state_alt, ocn_fields *G, ocn_fields *G_prev, void *p_hy,
                  void *stream);

/* ---------------------------------------------------------------------------------------------------------------
 * the pressure correction of the NonhydrostaticModel, (A8)-(A12) PAPER.md:829-851.  After a substage
 * the velocity is the predictor u~ (A8); the correction makes it discretely solenoidal:
 *     lap p = div(u~) / dt   (A12),        u^{m+1} = u~ - dt grad p   (A11)
 * with the second-order operators of (B2): div at ccc, grad p on the faces, lap = div grad (7-point, stretched-z aware).
 * Solved as the paper does on rectilinear grids: eigenfunction expansion by FFT in the equispaced
 * Periodic directions x, y (cuFFT, a library primitive) + one tridiagonal solve in z per horizontal mode.
 * Readings (R21-R23): dt is whatever interval the caller passes (u^{m+1} does not depend on it, p scales as
 * 1/dt); the wall-normal predictor velocity is taken as 0 on wall faces ("enforcing n.u~ = n.u^{m+1} on boundary
 * cells") => zero-normal-gradient rows for p; the singular mean mode is fixed by: horizontal mean of p at level k=1 is 0
 * (z Flat: mean of p is 0).  No halo of u,v,w or p is read or written: Periodic axes wrap by index.
 * Covered: Periodic x, Periodic y, Bounded or Flat z (the nonhydrostatic configurations C1, C2, C4); anything else
 * returns OCN_ERR_UNSUPPORTED. */
typedef struct ocn_poisson ocn_poisson; /* opaque; owns the cuFFT plans and DEVICE workspace: (Nx/2+1)*Ny*Nz complex
                                           elements of the grid's dtype + as many doubles (Thomas coefficients) */
/* Allocates the workspace and plans (this call, and only this one, allocates device memory and may synchronise).
 * `g` must outlive the solver.  Errors: OCN_ERR_INVALID, OCN_ERR_UNSUPPORTED, OCN_ERR_NOMEM, OCN_ERR_CUDA. */
int ocn_poisson_create(ocn_poisson **out, const ocn_grid *g);
int ocn_poisson_destroy(ocn_poisson *ps); /* NULL is allowed */
/* rhs <- div(u~)/dt on the interior (DEVICE, grid layout; halos untouched).  state: u, v (and w unless z is Flat). */
int ocn_pressure_rhs(const ocn_grid *g, double dt, const ocn_fields *state, void *rhs, void *stream);
/* p <- solution of lap p = rhs on the interior (DEVICE, grid layout; rhs may alias p; halos untouched). */
int ocn_poisson_solve(ocn_poisson *ps, const void *rhs, void *p, void *stream);
/* (A11) in place on the non-wall faces of u, v, w. */
int ocn_pressure_correct(const ocn_grid *g, double dt, ocn_fields *state, const void *p, void *stream);
/* the three calls above in sequence; p (DEVICE, grid layout) receives the nonhydrostatic pressure. */
int ocn_pressure_correction(ocn_poisson *ps, double dt, ocn_fields *state, void *p, void *stream);

/* ---------------------------------------------------------------------------------------------------------------
 * vertically-implicit diffusion, (A2) PAPER.md:785-803 (tracers), (A8),(A9) PAPER.md:829-835 (momentum):
 *     (1 - dt d_z kz d_z) q^{m+1} = q*          per column, for every prognostic field, in place,
 * q* = the field after the explicit substage (A4) computed with implicit_vertical_diffusion = 1 (so that G holds no
 * vertical diffusion), kz = nu for u, v, w and kappa[n] for tracer n (constant ScalarDiffusivity; fields with kz = 0 are
 * skipped: the operator is the identity), second-order flux-form d_z kz d_z on the (possibly stretched) z-metrics, no flux
 * through the walls for fields centred in z and w = 0 on the wall faces.  One Thomas solve per column.
 * dt is the interval the substage covered (reading R24: for RK3 stage m, (gamma^m - zeta^m) times the step).
 * Halos are neither read nor written.  Errors: OCN_ERR_INVALID (NULLs, z not Bounded, negative dt / nu / kappa). */
int ocn_implicit_vertical_diffusion(const ocn_grid *g, const ocn_params *p, double dt, ocn_fields *state, void *stream);

/* ---------------------------------------------------------------------------------------------------------------
 * split-explicit free surface of the HydrostaticFreeSurfaceModel, (A13)-(A21) PAPER.md:857-923.
 * After a substage the horizontal velocity is the predictor u~_h of (A17), computed WITHOUT the free-surface gradient.  Then
 *   (A13)  U = sum_k dz_c u, V = sum_k dz_c v                        ocn_barotropic_init     (once; later steps carry the averages)
 *   (A19)  F = sum_k dz_c (gamma G - zeta G_prev)   for G_u, G_v     ocn_barotropic_forcing  (the slow term, frozen while substepping)
 *   (A18),(A19),(A20)  M forward-backward substeps of dtau = dt/N:   ocn_barotropic_substeps
 *          eta^{n+1} = eta^n - dtau div_h(U^n);  U^{n+1} = U^n - dtau [ g H grad_h eta^{n+1} - F ];  bar = sum_n a_n (eta^n, U^n, V^n)
 *   (A21)  u <- u~ + (Ubar - sum_k dz_c u~) / H                      ocn_barotropic_correct
 * and the barotropic variables are re-initialised with the averages.
 * 2-D fields (eta at cc, U at fc, V at cf, FU, FV) are ONE horizontal plane of the grid layout: DEVICE, stride_z elements,
 * element (i,j) at offset0 - hz*stride_z + (i-1) + (j-1)*stride_y; halos are neither read nor written.
 * Readings (R25-R27): the free surface is the linearised one of eq. (16) on a static grid, so the
 * column integrals run over the resting depth H = sum dz_c and g(H+eta) of (A19) is g H; (A18)-(A20) print both M and N:
 * dtau = dt/N, M substeps n = 1..M are taken and averaged with the caller's weights a_n (HOST, M doubles; "the weights
 * calculated from the provided averaging kernel", M <= 2N centres the kernel at t^{m+1}); U (V) is 0 and stays 0 on wall
 * faces, Periodic axes wrap by index.  gamma, zeta: the right-hand side of (A3)/(A4) divided by the interval's share of the
 * step (RK3 stage m: gamma^m/(gamma^m - zeta^m), zeta^m/(gamma^m - zeta^m) with dt = (gamma^m - zeta^m) x the step).
 * z must be Bounded.  Errors: OCN_ERR_INVALID (NULLs, N or M < 1, dt <= 0). */
typedef struct { void *eta, *U, *V; } ocn_barotropic; /* DEVICE planes, caller-owned */
int ocn_barotropic_init(const ocn_grid *g, const ocn_fields *state, ocn_barotropic *bt, void *stream); /* writes bt->U, bt->V */
int ocn_barotropic_forcing(const ocn_grid *g, double gamma, double zeta, const ocn_fields *G, const ocn_fields *G_prev /* or NULL */,
                           void *FU, void *FV, void *stream);
/* bt: in = the n = 0 state, out = the averages; scratch: DEVICE, 6*stride_z elements of the grid's dtype. */
int ocn_barotropic_substeps(const ocn_grid *g, double grav, double dt, int N, int M, const double *weights, ocn_barotropic *bt,
                            const void *FU, const void *FV, void *scratch, void *stream);
int ocn_barotropic_correct(const ocn_grid *g, ocn_fields *state, const ocn_barotropic *bt, void *stream);

/* ocn_barotropic_substeps without the scratch argument, for callers that cannot come up with six planes of device memory
 * themselves: code running where the CUDA allocator is off limits — a host application that handed all of the GPU's memory to its
 * own pool at start-up (so cudaMalloc would fail or steal from it), a time-critical loop that cannot afford the device-wide
 * synchronisation an allocation implies, a plug-in whose host forbids allocation after initialisation.  The work planes are a
 * fixed array of OCN_BT_STATIC_SCRATCH_BYTES inside libocn.so's device image; EVERY GPU that loads the library holds those bytes
 * from load until the process exits, whether or not this call is ever made.  Same arithmetic, same kernels and same results as
 * ocn_barotropic_substeps given zero-filled scratch (arguments, layouts and readings as documented there); this call itself uses
 * no cudaMalloc, cudaFree or allocating library routine.
 * Limit: 6 * stride_z * sizeof(dtype) <= OCN_BT_STATIC_SCRATCH_BYTES, i.e. horizontal planes of up to 1 Mi fp64 (2 Mi fp32)
 * elements including halos and padding (C3's 1440 x 600 fits; a 1024 x 1024 plane with halos does not).  Larger grids are refused
 * with OCN_ERR_UNSUPPORTED before anything is enqueued — use ocn_barotropic_substeps.
 * First call on each device: looks up the array's device address (with that device current) and, like ocn_barotropic_substeps,
 * may set a kernel attribute; make that first call outside any stream capture.  Later calls only enqueue work on `stream`.
 * Sharing: there is ONE array per GPU, shared by every grid, stream and host thread of the process, and it keeps the previous
 * call's contents (the call clears the part that has to start from zero).  Two calls whose GPU work can overlap — different
 * streams without an event between them, or different host threads — race on it and corrupt each other's result: serialise
 * them on one stream or order them with events.
 * Errors: as ocn_barotropic_substeps (without the scratch NULL check), OCN_ERR_UNSUPPORTED (grid beyond the limit, device ordinal
 * >= 64), OCN_ERR_CUDA (the address look-up failed). */
#define OCN_BT_STATIC_SCRATCH_BYTES (48u << 20)
int ocn_barotropic_substeps_static(const ocn_grid *g, double grav, double dt, int N, int M, const double *weights, ocn_barotropic *bt,
                                   const void *FU, const void *FV, void *stream);

/* ---------------------------------------------------------------------------------------------------------------
 * One time step (n_substages RK3 substages) of a COMPLETE model on device-resident state: the hot path of ocn_step_fused plus
 * the SURVEY 8(f) rows the options select, in the paper's order:
 *   for m: ocn_fill_halos(cur); [hydrostatic: ocn_compute_w, ocn_compute_phy]; ocn_tendencies_rk3(m, cur -> other);
 *          [params->implicit_vertical_diffusion: ocn_implicit_vertical_diffusion(other, dt_m)]                       (A2),(A8)
 *          [free_surface: ocn_barotropic_forcing(gamma/(gamma-zeta), zeta/(gamma-zeta)); ocn_barotropic_substeps(dt_m);
 *                         ocn_barotropic_correct(other)]                                                              (A17)-(A21)
 *          [poisson: ocn_pressure_correction(other, dt_m)]                                                            (A11),(A12)
 *          swap(cur, other); swap(G, G_prev)                       with dt_m = (gamma^m - zeta^m) dt   (readings R21, R24, R26)
 * the results of exactly those calls, enqueued on `stream` (hydrostatic models on the TMA-ring kernel: w from continuity and, with
 * free_surface, the slow forcing FU, FV are computed inside the tendency kernel with the arithmetic of ocn_compute_w /
 * ocn_barotropic_forcing, bit for bit, and those two launches are dropped; state.w is then not written, see ocn_step_fused).
 * Result location as ocn_step_fused.  poisson != NULL requires a nonhydrostatic model, free_surface != 0 a hydrostatic one (bt
 * must have been initialised: ocn_barotropic_init or a previous step).
 * Errors: as the individual calls. */
typedef struct {
  ocn_poisson *poisson;       /* NULL: no pressure correction                                                   */
  void *p_nh;                 /* DEVICE, grid layout: receives the nonhydrostatic pressure (needed with poisson)  */
  int free_surface;           /* 1: split-explicit free surface                                                   */
  ocn_barotropic *bt;         /* HOST struct of DEVICE planes eta, U, V (carried from step to step)               */
  void *FU, *FV, *bt_scratch; /* DEVICE planes / 6 planes of scratch (see ocn_barotropic_substeps)                */
  int bt_N, bt_M;             /* substeps per interval and substeps actually taken / averaged                     */
  const double *bt_weights;   /* HOST, bt_M averaging weights                                                     */
} ocn_step_options;
int ocn_step_model(const ocn_grid *g, const ocn_params *p, const ocn_step_options *o, int n_substages, double dt, ocn_fields *state,
                   ocn_fields *state_alt, ocn_fields *G, ocn_fields *G_prev, void *p_hy, void *stream);

/* thread-local message of the last failing call on this thread (never NULL). */
const char *ocn_last_error(void);

/* number of kernels this library has launched since load (all streams); used by bench.py's gpu_launches. */
long long ocn_launch_count(void);

/* Measurement aid (MEASURED_PEAKS.json holds no ALU peak): enqueue ONE launch of register-resident
 * arithmetic chains on `stream`; the caller times it with CUDA events (bench.py --alu-peak) and divides *flops_out by the
 * duration to get the FP64 / FP32 issue peak that the tendency kernels' roofline is quoted against.
 *   dtype   OCN_F64 / OCN_F32;  blocks x threads_per_block (multiple of 32, <= 1024) threads, each n_iter x 32 operations
 *   mode    must be 0: pure FMA, 8 independent chains per thread (the argument is kept for ABI stability; the exploration
 *           modes of round 2 — other instructions issued beside the FMAs — left the library, their table is profiles/r2_alu_probe.md)
 *   sink    DEVICE, >= blocks*threads_per_block elements of dtype (never written in practice; keeps the chains alive)
 *   flops_out HOST or NULL: floating-point operations of the launch (FMA = 2)
 * Errors: OCN_ERR_INVALID (arguments), OCN_ERR_CUDA. */
int ocn_alu_probe(int dtype, int mode, int blocks, int threads_per_block, int n_iter, void *sink, double *flops_out, void *stream);

/* "major.minor" of this ABI. */
const char *ocn_version(void);

#ifdef __cplusplus
}
#endif
#endif /* OCN_H */
