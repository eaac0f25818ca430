"""ctypes binding of the CPU oracle (oracle/libocnref.so).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this module.  It does not import the product package and the product package does
not import it.

Arrays are dense, halo-padded numpy arrays of shape (Nz+2Hz, Ny+2Hy, Nx+2Hx) (x fastest);
float64 arrays may be evaluated in long double (eval=0, the parity reference) or double
(eval=1, the timed baseline); float32 arrays are evaluated in float (timed baseline only —
for fp32 parity upcast the inputs to float64 and use eval=0).

A *state* is a dict {"u": a|None, "v": a|None, "w": a|None, "c": [a, ...]}; a *params* is a
plain dict with the keys of `ocn_params` (include/ocn.h), see `default_params`.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libocnref.so")

PERIODIC, BOUNDED, FLAT = 0, 1, 2
ADV_NONE, ADV_UPWIND1, ADV_CENTERED2, ADV_WENO5, ADV_WENO7, ADV_WENO9 = 0, 1, 2, 5, 7, 9
EVAL_LONGDOUBLE, EVAL_DOUBLE = 0, 1
MAX_TRACERS = 8
LOC = {"u": (1, 0, 0), "v": (0, 1, 0), "w": (0, 0, 1), "c": (0, 0, 0)}


class _CParams(C.Structure):
    _fields_ = [("n_tracers", C.c_int), ("idx_T", C.c_int), ("idx_S", C.c_int),
                ("adv_x", C.c_int), ("adv_y", C.c_int), ("adv_z", C.c_int),
                ("momentum_prognostic", C.c_int), ("hydrostatic", C.c_int),
                ("weno_eps", C.c_double),
                ("f0", C.c_double), ("beta_coriolis", C.c_double), ("y0", C.c_double),
                ("g", C.c_double), ("alpha_T", C.c_double), ("beta_S", C.c_double),
                ("T_ref", C.POINTER(C.c_double)), ("S_ref", C.POINTER(C.c_double)),
                ("nu", C.c_double), ("kappa", C.c_double * MAX_TRACERS),
                ("implicit_vertical_diffusion", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            import importlib.util
            spec = importlib.util.spec_from_file_location("_ocnref_build", os.path.join(_HERE, "build.py"))
            mod = importlib.util.module_from_spec(spec)
            spec.loader.exec_module(mod)
            mod.build()
        L = C.CDLL(_LIBPATH)
        L.ocnref_grid_create.restype = C.c_void_p
        L.ocnref_grid_create.argtypes = [C.c_int] * 4 + [C.c_double, C.c_double, C.c_void_p, C.c_double, C.c_void_p]
        L.ocnref_grid_destroy.argtypes = [C.c_void_p]
        L.ocnref_weno5z.restype = C.c_double
        L.ocnref_weno5z.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.ocnref_reconstruct.restype = C.c_double
        L.ocnref_reconstruct.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double]
        L.ocnref_upwind_flux.restype = C.c_double
        L.ocnref_upwind_flux.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double]
        L.ocnref_num_threads.restype = C.c_int
        _lib = L
    return _lib


def default_params(**kw):
    p = dict(n_tracers=0, idx_T=-1, idx_S=-1, adv_x=ADV_WENO5, adv_y=ADV_WENO5, adv_z=ADV_WENO5,
             momentum_prognostic=1, hydrostatic=0, weno_eps=1e-8, f0=0.0, beta_coriolis=0.0, y0=0.0,
             g=0.0, alpha_T=0.0, beta_S=0.0, T_ref=None, S_ref=None, nu=0.0, kappa=[0.0] * MAX_TRACERS,
             implicit_vertical_diffusion=0)
    p.update(kw)
    return p


def _cparams(params):
    cp = _CParams()
    keep = []
    for k in ("n_tracers", "idx_T", "idx_S", "adv_x", "adv_y", "adv_z", "momentum_prognostic", "hydrostatic"):
        setattr(cp, k, int(params[k]))
    for k in ("weno_eps", "f0", "beta_coriolis", "y0", "g", "alpha_T", "beta_S", "nu"):
        setattr(cp, k, float(params[k]))
    for name in ("T_ref", "S_ref"):
        a = params.get(name)
        if a is not None:
            a = np.ascontiguousarray(a, dtype=np.float64)
            keep.append(a)
            setattr(cp, name, a.ctypes.data_as(C.POINTER(C.c_double)))
    cp.implicit_vertical_diffusion = int(params.get("implicit_vertical_diffusion", 0))
    kap = list(params["kappa"]) + [0.0] * MAX_TRACERS
    for n in range(MAX_TRACERS):
        cp.kappa[n] = float(kap[n])
    return cp, keep


def _ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def _ptr_array(arrs):
    n = max(len(arrs), 1)
    pa = (C.c_void_p * n)()
    for i, a in enumerate(arrs):
        pa[i] = a.ctypes.data
    return pa


def _i3(t):
    return (C.c_int * 3)(*[int(x) for x in t])


class RefGrid:
    """Grid + metrics (listing 15)."""

    def __init__(self, Nx, Ny, Nz, halo, dx, dy, dz_c=None, dz_uniform=1.0, topology=(PERIODIC, PERIODIC, BOUNDED)):
        self.Nx, self.Ny, self.Nz, self.halo = int(Nx), int(Ny), int(Nz), int(halo)
        self.dx, self.dy = float(dx), float(dy)
        self.topology = tuple(int(t) for t in topology)
        dz = None if dz_c is None else np.ascontiguousarray(dz_c, dtype=np.float64)
        self._h = lib().ocnref_grid_create(self.Nx, self.Ny, self.Nz, self.halo, self.dx, self.dy,
                                           _ptr(dz), float(dz_uniform), _i3(self.topology))
        self._h = C.c_void_p(self._h)
        n = [C.c_long(), C.c_long(), C.c_long()]
        h = [C.c_int(), C.c_int(), C.c_int()]
        lib().ocnref_grid_dims(self._h, *[C.byref(x) for x in n], *[C.byref(x) for x in h])
        self.nxp, self.nyp, self.nzp = (x.value for x in n)
        self.Hx, self.Hy, self.Hz = (x.value for x in h)
        self.shape = (self.nzp, self.nyp, self.nxp)

    def __del__(self):
        try:
            lib().ocnref_grid_destroy(self._h)
        except Exception:
            pass

    def metric(self, which):
        n = {"zf": self.Nz + 1, "zc": self.Nz, "dzc": self.Nz, "dzf": self.Nz - 1}[which]
        out = np.zeros(max(n, 1))
        lib().ocnref_grid_metric(self._h, {"zf": 0, "zc": 1, "dzc": 2, "dzf": 3}[which], _ptr(out))
        return out[:n]

    def zeros(self, dtype=np.float64):
        return np.zeros(self.shape, dtype=dtype)

    def interior(self, a):
        return a[self.Hz:self.Hz + self.Nz, self.Hy:self.Hy + self.Ny, self.Hx:self.Hx + self.Nx]

    def at(self, a, i, j, k):
        """element (i,j,k) in the paper's 1-based indexing (halos: <=0 and >N)."""
        return a[k - 1 + self.Hz, j - 1 + self.Hy, i - 1 + self.Hx]


def num_threads():
    return lib().ocnref_num_threads()


def set_num_threads(n):
    lib().ocnref_set_num_threads(C.c_int(int(n)))


def weno5z(q5, eps=1e-8, eval=0):
    q = np.ascontiguousarray(q5, dtype=np.float64)
    return lib().ocnref_weno5z(_ptr(q), float(eps), int(eval))


def reconstruct(q, m, kind, eps=1e-8):
    """kind: 2=C2, 4=C4, 1/-1=U1 left/right, 3/-3=U3, 5/-5=W5; target between q[m-1] and q[m] (0-based q)."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    return lib().ocnref_reconstruct(_ptr(q), int(m), int(kind), float(eps))


def upwind_flux(q, m, scheme, a, eps=1e-8):
    q = np.ascontiguousarray(q, dtype=np.float64)
    return lib().ocnref_upwind_flux(_ptr(q), int(m), int(scheme), float(a), float(eps))


def rk3_coefficients(stage):
    g, z = C.c_double(), C.c_double()
    lib().ocnref_rk3_coefficients_f64(int(stage), C.byref(g), C.byref(z))
    return g.value, z.value


def _fields(state):
    """[(name, array, loc)] of the fields present."""
    out = []
    for nm in ("u", "v", "w"):
        if state.get(nm) is not None:
            out.append((nm, state[nm], LOC[nm]))
    for n, a in enumerate(state.get("c", [])):
        out.append(("c%d" % n, a, LOC["c"]))
    return out


def _is32(a):
    return a.dtype == np.float32


def fill_halos(grid, params, state):
    """a1 — in place.  Hydrostatic: w is diagnosed by compute_w (halos included) and is skipped."""
    for nm, a, loc in _fields(state):
        if nm == "w" and params["hydrostatic"]:
            continue
        f = lib().ocnref_fill_halos_field_f32 if _is32(a) else lib().ocnref_fill_halos_field_f64
        f(grid._h, _ptr(a), _i3(loc))


def fill_halos_field(grid, a, loc):
    f = lib().ocnref_fill_halos_field_f32 if _is32(a) else lib().ocnref_fill_halos_field_f64
    f(grid._h, _ptr(a), _i3(loc))


def compute_w(grid, state, eval=0):
    """a2, eq (15) — writes state['w'] (must exist)."""
    u, v, w = state["u"], state["v"], state["w"]
    if _is32(w):
        lib().ocnref_compute_w_f32(grid._h, _ptr(u), _ptr(v), _ptr(w))
    else:
        lib().ocnref_compute_w_f64(grid._h, _ptr(u), _ptr(v), _ptr(w), int(eval))


def compute_phy(grid, params, state, eval=0):
    """a3, eq (14) — returns p_hy on all padded columns."""
    cp, keep = _cparams(params)
    T = state["c"][params["idx_T"]] if params["idx_T"] >= 0 else None
    S = state["c"][params["idx_S"]] if params["idx_S"] >= 0 else None
    ref = T if T is not None else S
    p = np.zeros_like(ref)
    if _is32(ref):
        lib().ocnref_compute_phy_f32(grid._h, C.byref(cp), _ptr(T), _ptr(S), _ptr(p))
    else:
        lib().ocnref_compute_phy_f64(grid._h, C.byref(cp), _ptr(T), _ptr(S), _ptr(p), int(eval))
    return p


def compute_tendencies(grid, params, state, p_hy=None, eval=0):
    """a4-a10 — returns G = {"u","v","w","c":[...]} (None for absent / non-prognostic fields)."""
    cp, keep = _cparams(params)
    cs = list(state.get("c", []))[:params["n_tracers"]]
    ref = cs[0] if cs else state["u"]
    mk = lambda: np.zeros_like(ref)
    G = {"u": None, "v": None, "w": None, "c": [mk() for _ in cs]}
    if params["momentum_prognostic"]:
        if state.get("u") is not None:
            G["u"] = mk()
        if state.get("v") is not None:
            G["v"] = mk()
        if state.get("w") is not None and not params["hydrostatic"] and grid.topology[2] != FLAT:
            G["w"] = mk()
    args = [grid._h, C.byref(cp), _ptr(state.get("u")), _ptr(state.get("v")), _ptr(state.get("w")),
            _ptr_array(cs), _ptr(p_hy), _ptr(G["u"]), _ptr(G["v"]), _ptr(G["w"]), _ptr_array(G["c"])]
    if _is32(ref):
        lib().ocnref_compute_tendencies_f32(*args)
    else:
        lib().ocnref_compute_tendencies_f64(*args, int(eval))
    return G


def tendencies_at(grid, params, state, p_hy, ijk, eval=0):
    """Tendencies at sample points ijk (ns,3) 1-based -> (ns, 3+n_tracers) [u,v,w,c0..] (float64 inputs only)."""
    cp, keep = _cparams(params)
    cs = list(state.get("c", []))[:params["n_tracers"]]
    ijk = np.ascontiguousarray(ijk, dtype=np.int32)
    out = np.zeros((ijk.shape[0], 3 + params["n_tracers"]))
    lib().ocnref_tendencies_at_f64(grid._h, C.byref(cp), _ptr(state.get("u")), _ptr(state.get("v")),
                                   _ptr(state.get("w")), _ptr_array(cs), _ptr(p_hy), C.c_long(ijk.shape[0]),
                                   _ptr(ijk), _ptr(out), int(eval))
    return out


def _prognostic(grid, params, state):
    out = []
    for nm, a, loc in _fields(state):
        if nm in ("u", "v", "w") and not params["momentum_prognostic"]:
            continue
        if nm == "w" and (params["hydrostatic"] or grid.topology[2] == FLAT):
            continue
        out.append((nm, a, loc))
    return out


def _get(G, nm):
    if G is None:
        return None
    return G["c"][int(nm[1:])] if nm.startswith("c") else G[nm]


def substage(grid, params, gamma, zeta, dt, state, G, G_prev, eval=0):
    """generic q += dt (gamma G - zeta G_prev) on interior non-wall points (a11 with free coefficients)."""
    for nm, a, loc in _prognostic(grid, params, state):
        g, gp = _get(G, nm), _get(G_prev, nm)
        if _is32(a):
            lib().ocnref_substage_field_f32(grid._h, _ptr(a), _ptr(g), _ptr(gp), C.c_double(gamma), C.c_double(zeta),
                                            C.c_double(dt), _i3(loc))
        else:
            lib().ocnref_substage_field_f64(grid._h, _ptr(a), _ptr(g), _ptr(gp), C.c_double(gamma), C.c_double(zeta),
                                            C.c_double(dt), _i3(loc), int(eval))


def rk3_substage(grid, params, stage, dt, state, G, G_prev, eval=0):
    """a11, eq (A4), stage in {1,2,3}."""
    for nm, a, loc in _prognostic(grid, params, state):
        g, gp = _get(G, nm), _get(G_prev, nm)
        if _is32(a):
            lib().ocnref_rk3_substage_field_f32(grid._h, _ptr(a), _ptr(g), _ptr(gp), int(stage), C.c_double(dt), _i3(loc))
        else:
            lib().ocnref_rk3_substage_field_f64(grid._h, _ptr(a), _ptr(g), _ptr(gp), int(stage), C.c_double(dt),
                                                _i3(loc), int(eval))


def step(grid, params, n_substages, dt, state, eval=0, timings=None):
    """n_substages consecutive substages m = 1..n of ONE time step, the call sequence of SURVEY 8(c) c.5
    (PAPER.md:793-801, 1078): for m { fill halos; [hydrostatic: w scan (15), p scan (14)]; tendencies;
    RK3 substage (A4); G becomes G_prev }.  `state` is updated in place; returns the last tendencies."""
    G_prev, G = None, None
    for m in range(1, n_substages + 1):
        fill_halos(grid, params, state)
        p_hy = None
        if params["hydrostatic"] and grid.topology[2] != FLAT:
            compute_w(grid, state, eval=eval)
            if params["idx_T"] >= 0 or params["idx_S"] >= 0:
                p_hy = compute_phy(grid, params, state, eval=eval)
        G = compute_tendencies(grid, params, state, p_hy, eval=eval)
        rk3_substage(grid, params, m, dt, state, G, G_prev, eval=eval)
        G_prev = G
    return G


# ---------------------------------------------------------------------------------------------------------
# pressure correction (A8),(A11),(A12) PAPER.md:829-851 and N3 — vertically-implicit
# diffusion (A2),(A8) PAPER.md:785-803.  float64 arrays only (fp32 parity: upcast the inputs); long double inside.
# ---------------------------------------------------------------------------------------------------------
def divergence(grid, state, scale=1.0):
    """scale * div(u,v,w) at ccc (B2); face N+1 = face 1 (Periodic) or the wall, 0 (Bounded) — reading R22."""
    ref = state["u"] if state.get("u") is not None else state["v"]
    out = np.zeros_like(ref)
    lib().ocnref_divergence_f64(grid._h, _ptr(state.get("u")), _ptr(state.get("v")), _ptr(state.get("w")), _ptr(out),
                                C.c_double(scale))
    return out


def poisson_solve(grid, rhs):
    """(A12): p with lap p = rhs on the interior (eigenfunction expansion in x,y + tridiagonal in z; gauge R23)."""
    p = np.zeros_like(rhs)
    lib().ocnref_poisson_solve_f64(grid._h, _ptr(rhs), _ptr(p))
    return p


def pressure_correct(grid, dt, state, p):
    """(A11): u,v,w -= dt grad p on non-wall faces, in place."""
    lib().ocnref_pressure_correct_f64(grid._h, C.c_double(dt), _ptr(state.get("u")), _ptr(state.get("v")),
                                      _ptr(state.get("w")), _ptr(p))


def pressure_correction(grid, dt, state):
    """(A12) + (A11) in long double end to end: state's u,v,w corrected in place; returns p (rounded to double)."""
    ref = state["u"] if state.get("u") is not None else state["v"]
    p = np.zeros_like(ref)
    lib().ocnref_pressure_correction_f64(grid._h, C.c_double(dt), _ptr(state.get("u")), _ptr(state.get("v")),
                                         _ptr(state.get("w")), _ptr(p))
    return p


def implicit_vertical_diffusion(grid, params, dt_stage, state):
    """(A2)/(A8): every prognostic field q <- (1 - dt d_z kz d_z)^-1 q per column, kz = nu (momentum) / kappa[n]."""
    for nm, a, loc in _prognostic(grid, params, state):
        kz = params["nu"] if nm in ("u", "v", "w") else params["kappa"][int(nm[1:])]
        lib().ocnref_implicit_vertical_diffusion_field_f64(grid._h, _ptr(a), int(loc[2]), C.c_double(kz),
                                                           C.c_double(dt_stage))


# ---------------------------------------------------------------------------------------------------------
# split-explicit free surface (A13)-(A21) PAPER.md:857-923.  Barotropic fields are dense
# padded planes of shape (Ny+2Hy, Nx+2Hx), float64; a barotropic state is {"eta", "U", "V"}.
# ---------------------------------------------------------------------------------------------------------
def plane(grid):
    return np.zeros((grid.nyp, grid.nxp))


def plane_interior(grid, a):
    return a[grid.Hy:grid.Hy + grid.Ny, grid.Hx:grid.Hx + grid.Nx]


def column_integral(grid, q, axis):
    """(A13): sum_k dz_c q on the non-wall faces of the component along axis (0: u, 1: v)."""
    out = plane(grid)
    lib().ocnref_column_integral_f64(grid._h, _ptr(q), _ptr(out), int(axis))
    return out


def barotropic_init(grid, state):
    return {"eta": plane(grid), "U": column_integral(grid, state["u"], 0), "V": column_integral(grid, state["v"], 1)}


def barotropic_forcing(grid, gamma, zeta, G, G_prev):
    """the slow term of (A19): (FU, FV) = sum_k dz_c (gamma G - zeta G_prev) for G_u, G_v."""
    out = []
    for axis, nm in ((0, "u"), (1, "v")):
        F = plane(grid)
        gp = None if G_prev is None else G_prev[nm]
        lib().ocnref_barotropic_forcing_f64(grid._h, C.c_double(gamma), C.c_double(zeta), _ptr(G[nm]), _ptr(gp), _ptr(F), axis)
        out.append(F)
    return out[0], out[1]


def barotropic_substeps(grid, grav, dt, N, weights, bt, FU, FV):
    """(A18)-(A20): M = len(weights) forward-backward substeps of dt/N; bt is replaced by the weighted averages."""
    a = np.ascontiguousarray(weights, dtype=np.float64)
    lib().ocnref_barotropic_substeps_f64(grid._h, C.c_double(grav), C.c_double(dt), int(N), int(a.size), _ptr(a),
                                         _ptr(bt["eta"]), _ptr(bt["U"]), _ptr(bt["V"]), _ptr(FU), _ptr(FV))


def barotropic_correct(grid, state, bt):
    """(A21): u, v <- predictor + (Ubar - column integral of the predictor) / H."""
    lib().ocnref_barotropic_correct_f64(grid._h, _ptr(state.get("u")), _ptr(state.get("v")), _ptr(bt["U"]), _ptr(bt["V"]))
