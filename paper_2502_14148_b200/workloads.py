"""Seeded synthetic workloads C0–C4 (BASELINE.json `configs`).

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path: it only
*generates inputs* — grids, parameter dictionaries and seeded initial fields with the shapes,
value distributions and structure of the paper's workloads.  It holds none of the method's
arithmetic (no reconstruction, no tendency, no halo fill, no time stepping) and imports
neither `oracle/` nor the CUDA binding.

The paper measures this path on no public benchmark suite or dataset (PAPER.md reports only
whole-model timings), so nothing here stands in for third-party items: the fields are the
config descriptions of BASELINE.json made concrete (recipe: DESIGN.md "Input recipe").

Fields are dense halo-padded arrays of shape (Nz+2Hz, Ny+2Hy, Nx+2Hx), x fastest, interior
filled and halos zero (the hot path's own `ocn_fill_halos` fills them).  Generation runs in
torch float64 on `device` ("cpu" for tests, "cuda" for the full-size benchmark configs) and is
cast to the config dtype at the end.  The same arrays are handed to the oracle and to the CUDA
path, so parity never depends on reproducing a random stream.
"""
import math

import numpy as np
import torch

PERIODIC, BOUNDED, FLAT = 0, 1, 2
ADV_NONE, ADV_UPWIND1, ADV_CENTERED2, ADV_WENO5, ADV_WENO7, ADV_WENO9 = 0, 1, 2, 5, 7, 9
MAX_TRACERS = 8
BASE_SEED = 20250214 * 10

_SIZES = {"C0": (64, 64, 1), "C1": (128, 128, 64), "C2": (512, 512, 256), "C3": (1440, 600, 50),
          "C4": (1024, 1024, 128)}


def _params(**kw):
    p = dict(n_tracers=0, idx_T=-1, idx_S=-1, adv_x=ADV_WENO5, adv_y=ADV_WENO5, adv_z=ADV_WENO5,
             momentum_prognostic=1, hydrostatic=0, weno_eps=1e-8, f0=0.0, beta_coriolis=0.0, y0=0.0,
             g=0.0, alpha_T=0.0, beta_S=0.0, T_ref=None, S_ref=None, nu=0.0, kappa=[0.0] * MAX_TRACERS)
    p.update(kw)
    return p


def c3_dz(Nz):
    """C3 stretched column: from the surface down min(250, 10*1.08^n); returned bottom -> top."""
    top_down = np.minimum(250.0, 10.0 * 1.08 ** np.arange(Nz, dtype=np.float64))
    return top_down[::-1].copy()


def z_centres(dz_c):
    """cell-centre heights for thicknesses bottom->top with the surface at z=0 (grid geometry only)."""
    zf = np.concatenate([[0.0], np.cumsum(np.asarray(dz_c, dtype=np.float64))]) - float(np.sum(dz_c))
    return 0.5 * (zf[:-1] + zf[1:])


def get_config(name, size=None, weno_order=5):
    """Return the workload description for 'C0'..'C4'.  `size=(Nx,Ny,Nz)` shrinks the grid, same recipe.
    `weno_order` = 7 or 9 replaces WENO5 on every axis that uses it and widens the halo to
    (order+1)/2; fields and all other parameters are unchanged."""
    idx = int(name[1])
    Nx, Ny, Nz = size if size is not None else _SIZES[name]
    cfg = dict(name=name, index=idx, seed=BASE_SEED + idx, dtype="f64", n_substages=3)
    les = dict(n_tracers=2, idx_T=0, idx_S=1, alpha_T=2e-4, beta_S=8e-4, g=9.81, f0=1e-4, nu=1e-4,
               kappa=[1e-4] * 2 + [0.0] * (MAX_TRACERS - 2))
    if name == "C0":
        cfg.update(grid=dict(Nx=Nx, Ny=Ny, Nz=1, halo=3, dx=1.0, dy=1.0, dz_c=None, dz_uniform=1.0,
                             topology=(PERIODIC, PERIODIC, FLAT)),
                   params=_params(n_tracers=1, adv_z=ADV_NONE, momentum_prognostic=0,
                                  kappa=[1e-2] + [0.0] * (MAX_TRACERS - 1)),
                   dt=0.1, has_w=False, description="2D tracer advection-diffusion, doubly periodic, WENO5")
    elif name in ("C1", "C2"):
        cfg.update(grid=dict(Nx=Nx, Ny=Ny, Nz=Nz, halo=3, dx=1.0, dy=1.0, dz_c=None, dz_uniform=1.0,
                             topology=(PERIODIC, PERIODIC, BOUNDED)),
                   params=_params(**les), dt=0.05, has_w=True,
                   description="3D nonhydrostatic LES tendencies, Periodic x,y / Bounded z, WENO5")
    elif name == "C3":
        dz = c3_dz(Nz)
        zc = z_centres(dz)
        cfg.update(grid=dict(Nx=Nx, Ny=Ny, Nz=Nz, halo=3, dx=5000.0, dy=5000.0, dz_c=dz, dz_uniform=0.0,
                             topology=(PERIODIC, BOUNDED, BOUNDED)),
                   params=_params(n_tracers=2, idx_T=0, idx_S=1, adv_z=ADV_CENTERED2, hydrostatic=1,
                                  alpha_T=2e-4, beta_S=8e-4, g=9.81, f0=1e-4, beta_coriolis=2e-11, y0=0.0,
                                  nu=1e-4, kappa=[1e-4] * 2 + [0.0] * (MAX_TRACERS - 2),
                                  T_ref=20.0 + 0.004 * zc, S_ref=35.0 - 0.0002 * zc),
                   dt=5.0, has_w=True,
                   description="hydrostatic channel, stretched z, WENO5 horizontal / Centered2 vertical, beta-plane")
    elif name == "C4":
        les4 = dict(les)
        les4.update(n_tracers=3, kappa=[1e-4] * 3 + [0.0] * (MAX_TRACERS - 3))
        cfg.update(grid=dict(Nx=Nx, Ny=Ny, Nz=Nz, halo=3, dx=1.0, dy=1.0, dz_c=None, dz_uniform=1.0,
                             topology=(PERIODIC, PERIODIC, BOUNDED)),
                   params=_params(**les4), dt=0.05, has_w=True, dtype="f32",
                   description="largest single-GPU case: LES physics, fp32, 3 tracers (T,S,dye)")
    else:
        raise KeyError(name)
    if weno_order != 5:
        if weno_order not in (7, 9):
            raise ValueError("weno_order must be 5, 7 or 9")
        for ax in ("adv_x", "adv_y", "adv_z"):
            if cfg["params"][ax] == ADV_WENO5:
                cfg["params"][ax] = weno_order
        cfg["grid"]["halo"] = (weno_order + 1) // 2
        cfg["description"] = cfg["description"].replace("WENO5", "WENO%d" % weno_order)
        cfg["weno_order"] = weno_order
    return cfg


def padded_shape(grid):
    H = grid["halo"]
    Hx, Hy, Hz = [0 if t == FLAT else H for t in grid["topology"]]
    return (grid["Nz"] + 2 * Hz, grid["Ny"] + 2 * Hy, grid["Nx"] + 2 * Hx), (Hx, Hy, Hz)


def _pad(grid, interior):
    """embed an (Nz,Ny,Nx) interior into a zero halo-padded array."""
    shape, (Hx, Hy, Hz) = padded_shape(grid)
    out = torch.zeros(shape, dtype=interior.dtype, device=interior.device)
    out[Hz:Hz + grid["Nz"], Hy:Hy + grid["Ny"], Hx:Hx + grid["Nx"]] = interior
    return out


class _Streams:
    """one independent child random stream per field (numpy SeedSequence -> torch.Generator)."""

    def __init__(self, seed, device):
        self.ss = np.random.SeedSequence(seed)
        self.device = torch.device(device)

    def next(self):
        child = self.ss.spawn(1)[0]
        g = torch.Generator(device=self.device)
        g.manual_seed(int(child.generate_state(1, dtype=np.uint64)[0] >> 1))
        return g

    def normal(self, shape):
        return torch.randn(shape, dtype=torch.float64, device=self.device, generator=self.next())

    def uniform(self, shape):
        return torch.rand(shape, dtype=torch.float64, device=self.device, generator=self.next())


def _wavenumbers(n, d, device, real=False):
    f = torch.fft.rfftfreq(n, d=d) if real else torch.fft.fftfreq(n, d=d)
    return (2.0 * math.pi * f).to(device=device, dtype=torch.float64)


def _gauss_filter_xy(a, sigma_x, sigma_y):
    """periodic Gaussian filter exp(-sigma^2 |k|^2 / 2) along the last two axes."""
    ny, nx = a.shape[-2:]
    ky = _wavenumbers(ny, 1.0, a.device)[:, None]
    kx = _wavenumbers(nx, 1.0, a.device, real=True)[None, :]
    filt = torch.exp(-0.5 * ((sigma_x * kx) ** 2 + (sigma_y * ky) ** 2))
    return torch.fft.irfft2(torch.fft.rfft2(a) * filt, s=(ny, nx))


def _shape_spectrum(a, power):
    """multiply the periodic Fourier amplitudes of a 3-D array by |k|^power (k in grid units, k=0 -> 0)."""
    nz, ny, nx = a.shape
    kz = _wavenumbers(nz, 1.0, a.device)[:, None, None]
    ky = _wavenumbers(ny, 1.0, a.device)[None, :, None]
    kx = _wavenumbers(nx, 1.0, a.device, real=True)[None, None, :]
    k2 = kx ** 2 + ky ** 2 + kz ** 2
    k2[0, 0, 0] = 1.0
    filt = k2 ** (0.5 * power)
    filt[0, 0, 0] = 0.0
    return torch.fft.irfftn(torch.fft.rfftn(a) * filt, s=(nz, ny, nx))


def _curl_bounded_z(Ax, Ay, Az, dx, dy, dz):
    """discrete curl of a vector potential (A_x at cff, A_y at fcf, A_z at ffc), periodic in x,y; A_x, A_y carry
    Nz+1 z-faces (zero on both walls).  Returns u (fcc), v (cfc), w (ccf, faces 1..Nz) — discretely solenoidal."""
    rx = lambda a: torch.roll(a, -1, dims=-1)
    ry = lambda a: torch.roll(a, -1, dims=-2)
    u = (ry(Az) - Az) / dy - (Ay[1:] - Ay[:-1]) / dz
    v = (Ax[1:] - Ax[:-1]) / dz - (rx(Az) - Az) / dx
    w = (rx(Ay) - Ay) / dx - (ry(Ax) - Ax) / dy
    return u, v, w[:-1]


def _rescale_rms(fields, rms):
    tot = sum(float((f * f).sum()) for f in fields)
    n = sum(f.numel() for f in fields)
    s = rms / math.sqrt(tot / n)
    return [f * s for f in fields]


def _dct_matrix(n, device):
    """orthonormal DCT-II matrix C[m,k] = s_m cos(pi m (k+1/2)/n)."""
    k = torch.arange(n, dtype=torch.float64, device=device)
    m = k[:, None]
    Cm = torch.cos(math.pi * m * (k[None, :] + 0.5) / n) * math.sqrt(2.0 / n)
    Cm[0] *= math.sqrt(0.5)
    return Cm


def _project_solenoidal(u, v, w, dx, dy, dz):
    """discrete pressure projection (FFT in x,y; DCT-II in z) of C-grid velocities with w=0 on both z-walls.
    u,v: (Nz,Ny,Nx); w: (Nz,Ny,Nx) holding z-faces 1..Nz (face Nz+1 = 0 implied)."""
    nz, ny, nx = u.shape
    rx = lambda a: torch.roll(a, -1, dims=-1)
    ry = lambda a: torch.roll(a, -1, dims=-2)

    def div(u, v, w):
        wt = torch.cat([w, torch.zeros_like(w[:1])], dim=0)
        return (rx(u) - u) / dx + (ry(v) - v) / dy + (wt[1:] - wt[:-1]) / dz

    Cm = _dct_matrix(nz, u.device)
    lx = -4.0 * torch.sin(0.5 * _wavenumbers(nx, 1.0, u.device)) ** 2 / dx ** 2
    ly = -4.0 * torch.sin(0.5 * _wavenumbers(ny, 1.0, u.device)) ** 2 / dy ** 2
    lz = -4.0 * torch.sin(0.5 * math.pi * torch.arange(nz, dtype=torch.float64, device=u.device) / nz) ** 2 / dz ** 2
    lam = lz[:, None, None] + ly[None, :, None] + lx[None, None, :]
    lam[0, 0, 0] = 1.0
    for _ in range(2):   # second pass removes the rounding residue of the first
        d = div(u, v, w)
        dh = torch.fft.fft2(torch.einsum("mk,kji->mji", Cm, d).to(torch.complex128))
        ph = dh / lam
        ph[0, 0, 0] = 0.0
        phi = torch.einsum("mk,mji->kji", Cm, torch.fft.ifft2(ph).real)
        u = u - (phi - torch.roll(phi, 1, dims=-1)) / dx
        v = v - (phi - torch.roll(phi, 1, dims=-2)) / dy
        w = w.clone()
        w[1:] = w[1:] - (phi[1:] - phi[:-1]) / dz
    return u, v, w


def _les_tracers(cfg, rs, zc, spectrum=None):
    g = cfg["grid"]
    shp = (g["Nz"], g["Ny"], g["Nx"])
    z = torch.as_tensor(zc, dtype=torch.float64, device=rs.device)[:, None, None]
    nT, nS = rs.normal(shp), rs.normal(shp)
    if spectrum is not None:
        nT, nS = _shape_spectrum(nT, spectrum), _shape_spectrum(nS, spectrum)
        nT, = _rescale_rms([nT], 1.0)
        nS, = _rescale_rms([nS], 1.0)
    T = 20.0 + 0.01 * z + 1e-3 * nT
    S = 35.0 + 1e-3 * nS
    return T, S


def generate_state(cfg, device="cpu", as_numpy=None):
    """Seeded initial fields of a config: {"u","v","w","c":[...]} dense halo-padded (halos zero).

    Returns numpy arrays when the device is the CPU (default) unless as_numpy=False; torch tensors
    on `device` otherwise.  dtype follows cfg["dtype"].
    """
    g = cfg["grid"]
    name = cfg["name"]
    Nx, Ny, Nz = g["Nx"], g["Ny"], g["Nz"]
    dx, dy = g["dx"], g["dy"]
    rs = _Streams(cfg["seed"], device)
    dz_c = np.full(Nz, g["dz_uniform"]) if g["dz_c"] is None else np.asarray(g["dz_c"], dtype=np.float64)
    zc = z_centres(dz_c)
    state = {"u": None, "v": None, "w": None, "c": []}
    if name == "C0":
        psi = _gauss_filter_xy(rs.normal((Ny, Nx)), 4.0, 4.0)           # at cell corners (ff)
        u = -(torch.roll(psi, -1, dims=0) - psi) / dy                    # fc
        v = (torch.roll(psi, -1, dims=1) - psi) / dx                     # cf
        c = rs.normal((Ny, Nx))
        u, v, c = u[None], v[None], c[None]
        tr = [c]
        w = None
    elif name == "C1":
        shp = (Nz, Ny, Nx)
        u, v, w = (0.01 * rs.normal(shp) for _ in range(3))
        w[0] = 0.0                                                       # bottom wall face
        u, v, w = _project_solenoidal(u, v, w, dx, dy, g["dz_uniform"])
        tr = list(_les_tracers(cfg, rs, zc))
    elif name in ("C2", "C4"):
        shp = (Nz, Ny, Nx)
        taper = torch.sin(math.pi * torch.arange(Nz, dtype=torch.float64, device=rs.device) / Nz)[:, None, None]
        A = []
        for comp in range(3):
            a = rs.normal(shp)
            if name == "C2":
                a = _shape_spectrum(a, -17.0 / 6.0)
            A.append(a)
        zero = torch.zeros((1, Ny, Nx), dtype=torch.float64, device=rs.device)
        Ax = torch.cat([A[0] * taper, zero], dim=0)                      # Nz+1 z-faces, zero on both walls
        Ay = torch.cat([A[1] * taper, zero], dim=0)
        u, v, w = _curl_bounded_z(Ax, Ay, A[2], dx, dy, g["dz_uniform"])
        del A, Ax, Ay
        u, v, w = _rescale_rms([u, v, w], 0.01)
        tr = list(_les_tracers(cfg, rs, zc, spectrum=(-11.0 / 6.0 if name == "C2" else None)))
        if name == "C4":
            tr.append(rs.uniform(shp))                                   # passive dye ~ U(0,1)
    elif name == "C3":
        p = cfg["params"]
        z = torch.as_tensor(zc, dtype=torch.float64, device=rs.device)[:, None, None]
        sig = 6.0
        # psi at ffc corners: x-faces 1..Nx (periodic), y-faces 1..Ny+1, zero on both y-walls
        wall = torch.sin(math.pi * torch.arange(Ny + 1, dtype=torch.float64, device=rs.device) / Ny)[None, :, None]
        wall[:, -1] = 0.0
        p1 = _gauss_filter_xy(rs.normal((Ny + 1, Nx)), sig, sig)[None]
        p2 = _gauss_filter_xy(rs.normal((Ny + 1, Nx)), sig, sig)[None]
        psi = (p1 * torch.exp(z / 1000.0) + 0.3 * p2 * torch.exp(z / 300.0)) * wall     # (Nz, Ny+1, Nx)
        jj = torch.arange(Ny, dtype=torch.float64, device=rs.device)
        f_c = p["f0"] + p["beta_coriolis"] * ((jj + 0.5) * dy - p["y0"])                 # at y-centres
        f_f = p["f0"] + p["beta_coriolis"] * (jj * dy - p["y0"])                         # at y-faces 1..Ny
        u = -(p["f0"] / f_c)[None, :, None] * (psi[:, 1:] - psi[:, :-1]) / dy
        v = (p["f0"] / f_f)[None, :, None] * (torch.roll(psi[:, :-1], -1, dims=-1) - psi[:, :-1]) / dx
        u, v = _rescale_rms([u, v], 0.1)
        w = torch.zeros_like(u)                                          # diagnosed by ocn_compute_w
        shp = (Nz, Ny, Nx)
        T = 20.0 + 0.004 * z + 0.05 * rs.normal(shp)
        S = 35.0 - 0.0002 * z + 0.05 * rs.normal(shp)
        tr = [T, S]
    else:
        raise KeyError(name)

    tdt = torch.float64 if cfg["dtype"] == "f64" else torch.float32
    conv = lambda a: _pad(g, a).to(tdt)
    state["u"], state["v"] = conv(u), conv(v)
    state["w"] = conv(w) if w is not None else None
    state["c"] = [conv(t) for t in tr]
    if as_numpy is None:
        as_numpy = torch.device(device).type == "cpu"
    if as_numpy:
        tonp = lambda a: None if a is None else a.cpu().numpy()
        state = {"u": tonp(state["u"]), "v": tonp(state["v"]), "w": tonp(state["w"]), "c": [tonp(t) for t in state["c"]]}
    return state


def barotropic_weights(N, p=2, q=4, r=0.18927):
    """Averaging weights a_n, n = 1..M <= 2N, for the split-explicit free surface ((A20) PAPER.md:887-919: "the weights
    calculated from the provided averaging kernel", by default a minimal-dispersion power-law filter).  INPUT DATA for
    ocn_barotropic_substeps, no method arithmetic: the power-law shape  A(t) = (t/t0)^p [1 - (t/t0)^q] - r (t/t0),
    t = n/N, t0 = (p+2)(p+q+2) / ((p+1)(p+q+1)), kept while positive, normalised to sum 1 (its first moment then sits close to
    t = 1, i.e. the kernel is centred at the end of the baroclinic step and M overshoots N)."""
    t0 = (p + 2.0) * (p + q + 2.0) / ((p + 1.0) * (p + q + 1.0))
    n = np.arange(1, 2 * N + 1)
    t = n / float(N) / t0
    A = t ** p * (1.0 - t ** q) - r * t
    M = int(np.max(np.nonzero(A > 0)[0])) + 1
    a = np.where(A[:M] > 0, A[:M], 0.0)
    return a / a.sum()
