"""Thin ctypes binding of libocn.so — same call names as include/ocn.h, argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library; torch is used for device memory
and streams.  There is no CPU fallback: `lib()` raises if libocn.so is missing, and every compute
call raises `OcnError` on a non-zero return code (e.g. no CUDA device).

    g   = ocn_grid_create(Nx, Ny, Nz, halo, dx, dy, dz_c, dz_uniform, topology, "f64")
    st  = g.fields(n_tracers=2)                  # zero-initialised device buffers in the grid layout
    g.upload(st.u, dense_padded_array)           # dense (Nz+2Hz, Ny+2Hy, Nx+2Hx) -> library layout
    ocn_fill_halos(g, params, st); ocn_compute_tendencies(g, params, st, None, G); ocn_rk3_substage(...)
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIBPATH = os.path.join(_HERE, "libocn.so")

OCN_PERIODIC, OCN_BOUNDED, OCN_FLAT = 0, 1, 2
OCN_F64, OCN_F32 = 0, 1
OCN_ADV_NONE, OCN_ADV_UPWIND1, OCN_ADV_CENTERED2, OCN_ADV_WENO5, OCN_ADV_WENO7, OCN_ADV_WENO9 = 0, 1, 2, 5, 7, 9
OCN_OK, OCN_ERR_INVALID, OCN_ERR_UNSUPPORTED, OCN_ERR_NOMEM, OCN_ERR_CUDA = 0, -1, -2, -3, -4
OCN_KERNEL_AUTO, OCN_KERNEL_PERCELL, OCN_KERNEL_FUSED = 0, 1, 2
OCN_DIAG_HI_NOSTAGE, OCN_DIAG_HALO_ELEMENTWISE, OCN_DIAG_BT_SINGLESTEP, OCN_DIAG_W_SCAN = 1, 2, 4, 8
OCN_MAX_TRACERS = 8

EXPORTS = ["ocn_grid_create", "ocn_grid_destroy", "ocn_grid_layout", "ocn_grid_set_kernel", "ocn_fill_halos",
           "ocn_compute_w", "ocn_compute_phy", "ocn_compute_tendencies", "ocn_rk3_substage", "ocn_substage",
           "ocn_tendencies_rk3", "ocn_step", "ocn_step_fused", "ocn_step_host", "ocn_last_error", "ocn_launch_count",
           "ocn_version", "ocn_poisson_create", "ocn_poisson_destroy", "ocn_pressure_rhs", "ocn_poisson_solve",
           "ocn_pressure_correct", "ocn_pressure_correction", "ocn_implicit_vertical_diffusion",
           "ocn_barotropic_init", "ocn_barotropic_forcing", "ocn_barotropic_substeps", "ocn_barotropic_substeps_static", "ocn_barotropic_correct", "ocn_step_model",
           "ocn_alu_probe", "ocn_grid_set_graphs", "ocn_grid_set_diag", "ocn_step_writes_w", "ocn_grid_graph_replays",
           "ocn_grid_set_external_halo", "ocn_halo_slab_elems", "ocn_halo_pack_y", "ocn_halo_unpack_y"]


class OcnError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libocn error %d: %s" % (code, msg))
        self.code = code


class ocn_layout(C.Structure):
    _fields_ = [("nx_pad", C.c_longlong), ("ny_pad", C.c_longlong), ("nz_pad", C.c_longlong),
                ("stride_y", C.c_longlong), ("stride_z", C.c_longlong), ("offset0", C.c_longlong),
                ("n_alloc", C.c_longlong), ("hx", C.c_int), ("hy", C.c_int), ("hz", C.c_int),
                ("alignment_bytes", C.c_int)]


class ocn_fields(C.Structure):
    _fields_ = [("u", C.c_void_p), ("v", C.c_void_p), ("w", C.c_void_p), ("c", C.c_void_p * OCN_MAX_TRACERS)]


class ocn_barotropic(C.Structure):
    _fields_ = [("eta", C.c_void_p), ("U", C.c_void_p), ("V", C.c_void_p)]


class ocn_step_options(C.Structure):
    _fields_ = [("poisson", C.c_void_p), ("p_nh", C.c_void_p), ("free_surface", C.c_int), ("bt", C.POINTER(ocn_barotropic)),
                ("FU", C.c_void_p), ("FV", C.c_void_p), ("bt_scratch", C.c_void_p), ("bt_N", C.c_int), ("bt_M", C.c_int),
                ("bt_weights", C.POINTER(C.c_double))]


class ocn_params(C.Structure):
    _fields_ = [("n_tracers", C.c_int), ("idx_T", C.c_int), ("idx_S", C.c_int),
                ("adv_x", C.c_int), ("adv_y", C.c_int), ("adv_z", C.c_int),
                ("momentum_prognostic", C.c_int), ("hydrostatic", C.c_int),
                ("weno_eps", C.c_double),
                ("f0", C.c_double), ("beta_coriolis", C.c_double), ("y0", C.c_double),
                ("g", C.c_double), ("alpha_T", C.c_double), ("beta_S", C.c_double),
                ("T_ref", C.POINTER(C.c_double)), ("S_ref", C.POINTER(C.c_double)),
                ("nu", C.c_double), ("kappa", C.c_double * OCN_MAX_TRACERS),
                ("implicit_vertical_diffusion", C.c_int)]


_lib = None


def lib():
    """Load libocn.so (fails loudly when it has not been built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIBPATH):
            raise ImportError("libocn.so not found at %s — build it with `python -m paper_2502_14148_b200.build`; "
                              "there is no CPU fallback" % LIBPATH)
        L = C.CDLL(LIBPATH)
        vp, i, d = C.c_void_p, C.c_int, C.c_double
        L.ocn_grid_create.argtypes = [C.POINTER(vp), i, i, i, i, d, d, vp, d, C.POINTER(i), i]
        L.ocn_grid_destroy.argtypes = [vp]
        L.ocn_grid_layout.argtypes = [vp, C.POINTER(ocn_layout)]
        L.ocn_grid_set_kernel.argtypes = [vp, i]
        L.ocn_fill_halos.argtypes = [vp, C.POINTER(ocn_params), C.POINTER(ocn_fields), vp]
        L.ocn_compute_w.argtypes = [vp, C.POINTER(ocn_fields), vp]
        L.ocn_compute_phy.argtypes = [vp, C.POINTER(ocn_params), C.POINTER(ocn_fields), vp, vp]
        L.ocn_compute_tendencies.argtypes = [vp, C.POINTER(ocn_params), C.POINTER(ocn_fields), vp, C.POINTER(ocn_fields), vp]
        L.ocn_rk3_substage.argtypes = [vp, C.POINTER(ocn_params), i, d, C.POINTER(ocn_fields), C.POINTER(ocn_fields),
                                       C.POINTER(ocn_fields), vp]
        L.ocn_substage.argtypes = [vp, C.POINTER(ocn_params), d, d, d, C.POINTER(ocn_fields), C.POINTER(ocn_fields),
                                   C.POINTER(ocn_fields), vp]
        L.ocn_step.argtypes = [vp, C.POINTER(ocn_params), i, d, C.POINTER(ocn_fields), C.POINTER(ocn_fields),
                               C.POINTER(ocn_fields), vp, vp]
        L.ocn_step_host.argtypes = [vp, C.POINTER(ocn_params), i, d, C.POINTER(ocn_fields), C.POINTER(ocn_fields),
                                    C.POINTER(ocn_fields), C.POINTER(ocn_fields), C.POINTER(ocn_fields), vp, vp]
        L.ocn_tendencies_rk3.argtypes = [vp, C.POINTER(ocn_params), i, d, C.POINTER(ocn_fields), vp, C.POINTER(ocn_fields),
                                         C.POINTER(ocn_fields), C.POINTER(ocn_fields), vp]
        L.ocn_step_fused.argtypes = [vp, C.POINTER(ocn_params), i, d, C.POINTER(ocn_fields), C.POINTER(ocn_fields),
                                     C.POINTER(ocn_fields), C.POINTER(ocn_fields), vp, vp]
        L.ocn_poisson_create.argtypes = [C.POINTER(vp), vp]
        L.ocn_poisson_destroy.argtypes = [vp]
        L.ocn_pressure_rhs.argtypes = [vp, d, C.POINTER(ocn_fields), vp, vp]
        L.ocn_poisson_solve.argtypes = [vp, vp, vp, vp]
        L.ocn_pressure_correct.argtypes = [vp, d, C.POINTER(ocn_fields), vp, vp]
        L.ocn_pressure_correction.argtypes = [vp, d, C.POINTER(ocn_fields), vp, vp]
        L.ocn_implicit_vertical_diffusion.argtypes = [vp, C.POINTER(ocn_params), d, C.POINTER(ocn_fields), vp]
        L.ocn_barotropic_init.argtypes = [vp, C.POINTER(ocn_fields), C.POINTER(ocn_barotropic), vp]
        L.ocn_barotropic_forcing.argtypes = [vp, d, d, C.POINTER(ocn_fields), C.POINTER(ocn_fields), vp, vp, vp]
        L.ocn_barotropic_substeps.argtypes = [vp, d, d, i, i, C.POINTER(d), C.POINTER(ocn_barotropic), vp, vp, vp, vp]
        L.ocn_barotropic_substeps_static.argtypes = [vp, d, d, i, i, C.POINTER(d), C.POINTER(ocn_barotropic), vp, vp, vp]
        L.ocn_barotropic_correct.argtypes = [vp, C.POINTER(ocn_fields), C.POINTER(ocn_barotropic), vp]
        L.ocn_step_model.argtypes = [vp, C.POINTER(ocn_params), C.POINTER(ocn_step_options), i, d, C.POINTER(ocn_fields),
                                     C.POINTER(ocn_fields), C.POINTER(ocn_fields), C.POINTER(ocn_fields), vp, vp]
        L.ocn_grid_set_graphs.argtypes = [vp, i]
        L.ocn_grid_set_diag.argtypes = [vp, C.c_uint]
        L.ocn_step_writes_w.argtypes = [vp, C.POINTER(ocn_params)]
        L.ocn_grid_set_external_halo.argtypes = [vp, i, i]
        L.ocn_halo_slab_elems.argtypes = [vp, C.POINTER(ocn_params)]
        L.ocn_halo_slab_elems.restype = C.c_longlong
        L.ocn_halo_pack_y.argtypes = [vp, C.POINTER(ocn_params), C.POINTER(ocn_fields), i, vp, vp]
        L.ocn_halo_unpack_y.argtypes = [vp, C.POINTER(ocn_params), C.POINTER(ocn_fields), i, vp, vp]
        L.ocn_grid_graph_replays.argtypes = [vp, C.POINTER(C.c_longlong)]
        L.ocn_alu_probe.argtypes = [i, i, i, i, i, vp, C.POINTER(d), vp]
        L.ocn_last_error.restype = C.c_char_p
        L.ocn_launch_count.restype = C.c_longlong
        L.ocn_version.restype = C.c_char_p
        for name in EXPORTS:
            getattr(L, name)
        _lib = L
    return _lib


def _check(rc):
    if rc != OCN_OK:
        raise OcnError(rc, lib().ocn_last_error().decode())


def _stream(stream):
    if stream is None:
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, torch.cuda.Stream):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


def make_params(p):
    """dict (keys of ocn_params) -> (ocn_params, keepalive list)."""
    if isinstance(p, tuple):
        return p
    cp = ocn_params()
    keep = []
    for k in ("n_tracers", "idx_T", "idx_S", "adv_x", "adv_y", "adv_z", "momentum_prognostic", "hydrostatic"):
        setattr(cp, k, int(p[k]))
    for k in ("weno_eps", "f0", "beta_coriolis", "y0", "g", "alpha_T", "beta_S", "nu"):
        setattr(cp, k, float(p[k]))
    for name in ("T_ref", "S_ref"):
        a = p.get(name)
        if a is not None:
            a = np.ascontiguousarray(a, dtype=np.float64)
            keep.append(a)
            setattr(cp, name, a.ctypes.data_as(C.POINTER(C.c_double)))
    cp.implicit_vertical_diffusion = int(p.get("implicit_vertical_diffusion", 0))
    kap = list(p["kappa"]) + [0.0] * OCN_MAX_TRACERS
    for n in range(OCN_MAX_TRACERS):
        cp.kappa[n] = float(kap[n])
    return cp, keep


class Fields:
    """u, v, w and tracers as flat device tensors in the grid layout (None = absent)."""

    def __init__(self, u=None, v=None, w=None, c=()):
        self.u, self.v, self.w, self.c = u, v, w, list(c)

    def struct(self):
        s = ocn_fields()
        s.u = self.u.data_ptr() if self.u is not None else None
        s.v = self.v.data_ptr() if self.v is not None else None
        s.w = self.w.data_ptr() if self.w is not None else None
        for n, t in enumerate(self.c):
            s.c[n] = t.data_ptr() if t is not None else None
        return s

    def all(self):
        return [t for t in (self.u, self.v, self.w) if t is not None] + [t for t in self.c if t is not None]


def _fs(f):
    if f is None:
        return None
    if isinstance(f, Fields):
        return C.byref(f.struct())
    return C.byref(f)


class Grid:
    """ocn_grid handle + layout + buffer helpers."""

    def __init__(self, Nx, Ny, Nz, halo, dx, dy, dz_c=None, dz_uniform=1.0, topology=(0, 0, 1), dtype="f64",
                 device="cuda"):
        self.Nx, self.Ny, self.Nz, self.halo = int(Nx), int(Ny), int(Nz), int(halo)
        self.topology = tuple(int(t) for t in topology)
        self.dtype = dtype
        self.tdtype = torch.float64 if dtype == "f64" else torch.float32
        self.device = torch.device(device)
        h = C.c_void_p()
        dz = None if dz_c is None else np.ascontiguousarray(dz_c, dtype=np.float64)
        topo = (C.c_int * 3)(*self.topology)
        _check(lib().ocn_grid_create(C.byref(h), self.Nx, self.Ny, self.Nz, self.halo, float(dx), float(dy),
                                     None if dz is None else C.c_void_p(dz.ctypes.data), float(dz_uniform), topo,
                                     OCN_F64 if dtype == "f64" else OCN_F32))
        self._h = h
        self.layout = ocn_layout()
        _check(lib().ocn_grid_layout(self._h, C.byref(self.layout)))
        L = self.layout
        self.shape = (L.nz_pad, L.ny_pad, L.nx_pad)
        self._xo = L.offset0 - L.hz * L.stride_z - L.hy * L.stride_y - L.hx     # array x-index of logical padded x=0

    def __del__(self):
        try:
            lib().ocn_grid_destroy(self._h)
        except Exception:
            pass

    def set_graphs(self, enable):
        _check(lib().ocn_grid_set_graphs(self._h, int(bool(enable))))

    def set_external_halo(self, axis, external=True):
        _check(lib().ocn_grid_set_external_halo(self._h, int(axis), int(bool(external))))

    def graph_replays(self):
        n = C.c_longlong(0)
        _check(lib().ocn_grid_graph_replays(self._h, C.byref(n)))
        return int(n.value)

    def set_diag(self, mask):
        """OCN_DIAG_* mask: reference / fallback kernels with identical results (include/ocn.h)."""
        _check(lib().ocn_grid_set_diag(self._h, int(mask)))

    def set_kernel(self, kernel):
        _check(lib().ocn_grid_set_kernel(self._h, int(kernel)))

    # ---- buffers -------------------------------------------------------------------------------
    def new_field(self):
        t = torch.zeros(self.layout.n_alloc, dtype=self.tdtype, device=self.device)
        assert t.data_ptr() % self.layout.alignment_bytes == 0
        return t

    def fields(self, n_tracers=0, u=True, v=True, w=True):
        return Fields(self.new_field() if u else None, self.new_field() if v else None,
                      self.new_field() if w else None, [self.new_field() for _ in range(n_tracers)])

    def view(self, t):
        """dense-shaped (nz_pad, ny_pad, nx_pad) strided view of a layout buffer."""
        L = self.layout
        return t.view(L.nz_pad, L.ny_pad, L.stride_y)[:, :, self._xo:self._xo + L.nx_pad]

    def upload(self, t, dense):
        """copy a dense halo-padded array (numpy or torch, any device) into the layout buffer t."""
        src = torch.as_tensor(dense)
        self.view(t).copy_(src.to(device=self.device, dtype=self.tdtype))
        return t

    def download(self, t):
        """layout buffer -> dense halo-padded numpy array."""
        return self.view(t).contiguous().cpu().numpy()

    def interior(self, t):
        L = self.layout
        return self.view(t)[L.hz:L.hz + self.Nz, L.hy:L.hy + self.Ny, L.hx:L.hx + self.Nx]

    def fields_from_state(self, state):
        """oracle-style state dict of dense arrays -> Fields."""
        mk = lambda a: None if a is None else self.upload(self.new_field(), a)
        return Fields(mk(state.get("u")), mk(state.get("v")), mk(state.get("w")), [mk(c) for c in state.get("c", [])])

    def state_from_fields(self, f):
        dn = lambda t: None if t is None else self.download(t)
        return {"u": dn(f.u), "v": dn(f.v), "w": dn(f.w), "c": [dn(t) for t in f.c]}


# ---- the calls, named as in include/ocn.h ----------------------------------------------------------
def ocn_grid_create(Nx, Ny, Nz, halo, dx, dy, dz_c=None, dz_uniform=1.0, topology=(0, 0, 1), dtype="f64", device="cuda"):
    return Grid(Nx, Ny, Nz, halo, dx, dy, dz_c, dz_uniform, topology, dtype, device)


def ocn_fill_halos(g, params, state, stream=None):
    cp, keep = make_params(params)
    _check(lib().ocn_fill_halos(g._h, C.byref(cp), _fs(state), _stream(stream)))


def ocn_compute_w(g, state, stream=None):
    _check(lib().ocn_compute_w(g._h, _fs(state), _stream(stream)))


def ocn_compute_phy(g, params, state, p_hy, stream=None):
    cp, keep = make_params(params)
    _check(lib().ocn_compute_phy(g._h, C.byref(cp), _fs(state), C.c_void_p(p_hy.data_ptr()), _stream(stream)))


def ocn_compute_tendencies(g, params, state, p_hy, G, stream=None):
    cp, keep = make_params(params)
    ph = None if p_hy is None else C.c_void_p(p_hy.data_ptr())
    _check(lib().ocn_compute_tendencies(g._h, C.byref(cp), _fs(state), ph, _fs(G), _stream(stream)))


def ocn_rk3_substage(g, params, stage, dt, state, G, G_prev, stream=None):
    cp, keep = make_params(params)
    _check(lib().ocn_rk3_substage(g._h, C.byref(cp), int(stage), float(dt), _fs(state), _fs(G), _fs(G_prev), _stream(stream)))


def ocn_substage(g, params, gamma, zeta, dt, state, G, G_prev, stream=None):
    cp, keep = make_params(params)
    _check(lib().ocn_substage(g._h, C.byref(cp), float(gamma), float(zeta), float(dt), _fs(state), _fs(G), _fs(G_prev),
                              _stream(stream)))


def ocn_step(g, params, n_substages, dt, state, G, G_prev, p_hy=None, stream=None):
    """n_substages consecutive RK3 substages of one step on device-resident state (see include/ocn.h)."""
    cp, keep = make_params(params)
    ph = None if p_hy is None else C.c_void_p(p_hy.data_ptr())
    _check(lib().ocn_step(g._h, C.byref(cp), int(n_substages), float(dt), _fs(state), _fs(G), _fs(G_prev), ph, _stream(stream)))


def ocn_tendencies_rk3(g, params, stage, dt, state, p_hy, G, G_prev, state_new, stream=None):
    """tendencies of `state` into G and the (A4) substage into the ping-pong buffers `state_new`, one pass."""
    cp, keep = make_params(params)
    ph = None if p_hy is None else C.c_void_p(p_hy.data_ptr())
    _check(lib().ocn_tendencies_rk3(g._h, C.byref(cp), int(stage), float(dt), _fs(state), ph, _fs(G), _fs(G_prev),
                                    _fs(state_new), _stream(stream)))


def ocn_step_fused(g, params, n_substages, dt, state, state_alt, G, G_prev, p_hy=None, stream=None):
    """n_substages substages with the fused tendency+substage pass; the result is in state_alt if n_substages is odd."""
    cp, keep = make_params(params)
    ph = None if p_hy is None else C.c_void_p(p_hy.data_ptr())
    _check(lib().ocn_step_fused(g._h, C.byref(cp), int(n_substages), float(dt), _fs(state), _fs(state_alt), _fs(G),
                                _fs(G_prev), ph, _stream(stream)))


def ocn_step_writes_w(g, params):
    """True when ocn_step_fused / ocn_step_model write the diagnosed w into state.w for this grid and model (include/ocn.h)."""
    cp, keep = make_params(params)
    rc = lib().ocn_step_writes_w(g._h, C.byref(cp))
    if rc < 0:
        _check(rc)
    return bool(rc)


def ocn_step_host(g, params, n_substages, dt, host_state, dev_state, dev_state_alt, G, G_prev, p_hy=None, stream=None):
    """one full step from HOST buffers: H2D of every state field, n_substages x {fill halos, [w, p scans],
    tendencies, RK3 substage} (fused pass when dev_state_alt is given and the fused kernel applies), D2H of the
    updated state.  host_state: Fields of pinned host tensors (layout order)."""
    cp, keep = make_params(params)
    ph = None if p_hy is None else C.c_void_p(p_hy.data_ptr())
    _check(lib().ocn_step_host(g._h, C.byref(cp), int(n_substages), float(dt), _fs(host_state), _fs(dev_state),
                               _fs(dev_state_alt), _fs(G), _fs(G_prev), ph, _stream(stream)))


def ocn_implicit_vertical_diffusion(g, params, dt, state, stream=None):
    """(A2)/(A8): q <- (1 - dt d_z kz d_z)^-1 q per column for every prognostic field, in place."""
    cp, keep = make_params(params)
    _check(lib().ocn_implicit_vertical_diffusion(g._h, C.byref(cp), float(dt), _fs(state), _stream(stream)))


class Barotropic:
    """eta, U, V as device planes (one horizontal plane of the grid layout) + the 6-plane scratch of the substepper."""

    def __init__(self, g):
        self.grid = g
        n = g.layout.stride_z
        mk = lambda k=1: torch.zeros(n * k, dtype=g.tdtype, device=g.device)
        self.eta, self.U, self.V, self.FU, self.FV, self.scratch = mk(), mk(), mk(), mk(), mk(), mk(6)

    def struct(self):
        s = ocn_barotropic()
        s.eta, s.U, s.V = self.eta.data_ptr(), self.U.data_ptr(), self.V.data_ptr()
        return s

    def view(self, t):
        """dense (ny_pad, nx_pad) view of a plane."""
        g, L = self.grid, self.grid.layout
        return t.view(L.ny_pad, L.stride_y)[:, g._xo:g._xo + L.nx_pad]

    def upload(self, t, dense):
        self.view(t).copy_(torch.as_tensor(dense).to(device=self.grid.device, dtype=self.grid.tdtype))

    def download(self, t):
        return self.view(t).contiguous().cpu().numpy()


def ocn_barotropic_init(g, state, bt, stream=None):
    _check(lib().ocn_barotropic_init(g._h, _fs(state), C.byref(bt.struct()), _stream(stream)))


def ocn_barotropic_forcing(g, gamma, zeta, G, G_prev, bt, stream=None):
    """writes bt.FU, bt.FV."""
    _check(lib().ocn_barotropic_forcing(g._h, float(gamma), float(zeta), _fs(G), _fs(G_prev), C.c_void_p(bt.FU.data_ptr()),
                                        C.c_void_p(bt.FV.data_ptr()), _stream(stream)))


def ocn_barotropic_substeps(g, grav, dt, N, weights, bt, stream=None):
    a = np.ascontiguousarray(weights, dtype=np.float64)
    _check(lib().ocn_barotropic_substeps(g._h, float(grav), float(dt), int(N), int(a.size), a.ctypes.data_as(C.POINTER(C.c_double)),
                                         C.byref(bt.struct()), C.c_void_p(bt.FU.data_ptr()), C.c_void_p(bt.FV.data_ptr()),
                                         C.c_void_p(bt.scratch.data_ptr()), _stream(stream)))


OCN_BT_STATIC_SCRATCH_BYTES = 48 << 20


def ocn_barotropic_substeps_static(g, grav, dt, N, weights, bt, stream=None):
    """ocn_barotropic_substeps on the library's built-in work planes: bt.scratch is not touched and nothing is allocated, for
    callers that may not use the CUDA allocator (memory handed to their own pool, no allocation after start-up, no device-wide
    synchronisation allowed).  Planes of at most OCN_BT_STATIC_SCRATCH_BYTES / 6 bytes; one shared array per GPU, so calls whose
    GPU work may overlap must be ordered by the caller (include/ocn.h)."""
    a = np.ascontiguousarray(weights, dtype=np.float64)
    _check(lib().ocn_barotropic_substeps_static(g._h, float(grav), float(dt), int(N), int(a.size), a.ctypes.data_as(C.POINTER(C.c_double)),
                                                C.byref(bt.struct()), C.c_void_p(bt.FU.data_ptr()), C.c_void_p(bt.FV.data_ptr()),
                                                _stream(stream)))


def ocn_barotropic_correct(g, state, bt, stream=None):
    _check(lib().ocn_barotropic_correct(g._h, _fs(state), C.byref(bt.struct()), _stream(stream)))


class Poisson:
    """ocn_poisson handle (cuFFT plans + spectral workspace); keeps its Grid alive."""

    def __init__(self, g):
        self.grid = g
        h = C.c_void_p()
        _check(lib().ocn_poisson_create(C.byref(h), g._h))
        self._h = h

    def __del__(self):
        try:
            lib().ocn_poisson_destroy(self._h)
        except Exception:
            pass


def ocn_poisson_create(g):
    return Poisson(g)


def ocn_pressure_rhs(g, dt, state, rhs, stream=None):
    _check(lib().ocn_pressure_rhs(g._h, float(dt), _fs(state), C.c_void_p(rhs.data_ptr()), _stream(stream)))


def ocn_poisson_solve(ps, rhs, p, stream=None):
    _check(lib().ocn_poisson_solve(ps._h, C.c_void_p(rhs.data_ptr()), C.c_void_p(p.data_ptr()), _stream(stream)))


def ocn_pressure_correct(g, dt, state, p, stream=None):
    _check(lib().ocn_pressure_correct(g._h, float(dt), _fs(state), C.c_void_p(p.data_ptr()), _stream(stream)))


def ocn_pressure_correction(ps, dt, state, p, stream=None):
    """(A12) + (A11): rhs, solve, correct; p receives the nonhydrostatic pressure."""
    _check(lib().ocn_pressure_correction(ps._h, float(dt), _fs(state), C.c_void_p(p.data_ptr()), _stream(stream)))


def ocn_step_model(g, params, n_substages, dt, state, state_alt, G, G_prev, p_hy=None, poisson=None, p_nh=None, bt=None,
                   bt_N=0, bt_weights=None, stream=None):
    """one step of a complete model (include/ocn.h): hot path + implicit vertical diffusion (params flag) + split-explicit free
    surface (bt given) + pressure correction (poisson given).  The result is in state_alt if n_substages is odd."""
    cp, keep = make_params(params)
    o = ocn_step_options()
    if poisson is not None:
        o.poisson, o.p_nh = poisson._h, p_nh.data_ptr()
    if bt is not None:
        a = np.ascontiguousarray(bt_weights, dtype=np.float64)
        bs = bt.struct()
        keep += [a, bs]
        o.free_surface, o.bt = 1, C.pointer(bs)
        o.FU, o.FV, o.bt_scratch = bt.FU.data_ptr(), bt.FV.data_ptr(), bt.scratch.data_ptr()
        o.bt_N, o.bt_M, o.bt_weights = int(bt_N), int(a.size), a.ctypes.data_as(C.POINTER(C.c_double))
    ph = None if p_hy is None else C.c_void_p(p_hy.data_ptr())
    _check(lib().ocn_step_model(g._h, C.byref(cp), C.byref(o), int(n_substages), float(dt), _fs(state), _fs(state_alt), _fs(G),
                                _fs(G_prev), ph, _stream(stream)))


def ocn_halo_slab_elems(g, params):
    cp, keep = make_params(params)
    n = int(lib().ocn_halo_slab_elems(g._h, C.byref(cp)))
    if n < 0:
        raise OcnError(OCN_ERR_INVALID, lib().ocn_last_error().decode())
    return n


def ocn_halo_pack_y(g, params, state, side, buf, stream=None):
    cp, keep = make_params(params)
    _check(lib().ocn_halo_pack_y(g._h, C.byref(cp), _fs(state), int(side), C.c_void_p(buf.data_ptr()), _stream(stream)))


def ocn_halo_unpack_y(g, params, state, side, buf, stream=None):
    cp, keep = make_params(params)
    _check(lib().ocn_halo_unpack_y(g._h, C.byref(cp), _fs(state), int(side), C.c_void_p(buf.data_ptr()), _stream(stream)))


def ocn_alu_probe(dtype, mode, blocks, threads_per_block, n_iter, sink, stream=None):
    """Enqueue one launch of the ALU probe; returns its floating-point operation count."""
    flops = C.c_double(0.0)
    _check(lib().ocn_alu_probe(int(dtype), int(mode), int(blocks), int(threads_per_block), int(n_iter), C.c_void_p(sink.data_ptr()),
                               C.byref(flops), _stream(stream)))
    return flops.value


def ocn_launch_count():
    return int(lib().ocn_launch_count())


def ocn_version():
    return lib().ocn_version().decode()
