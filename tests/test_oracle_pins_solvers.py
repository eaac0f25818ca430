"""Pins of the oracle's N2 (pressure correction, (A8),(A11),(A12) PAPER.md:829-851) and N3 (vertically-implicit
diffusion, (A2) PAPER.md:785-803) routines against what the mathematics fixes — none of them re-types the oracle's
own arithmetic: the operator is re-applied by independent numpy slicing, solved densely by LAPACK on tiny grids,
checked on closed-form eigenfunctions, and through the defining property div(u^{m+1}) = 0."""
import numpy as np
import pytest

from oracle import ocnref as ref

P, B, F = ref.PERIODIC, ref.BOUNDED, ref.FLAT


def stretched(Nz, seed=0):
    r = np.random.default_rng(seed)
    return 0.5 + r.random(Nz) * 1.5


def make_grid(Nx, Ny, Nz, topo, dz=None, dx=1.0, dy=1.0, H=3):
    return ref.RefGrid(Nx, Ny, Nz, H, dx, dy, dz_c=dz, dz_uniform=1.0, topology=topo)


def numpy_laplacian(g, p_int, dz):
    """7-point flux-form Laplacian of an interior array (Nz,Ny,Nx): periodic wrap / zero wall flux, stretched z.
    Written with np.roll / concatenation — independent of the oracle's loops."""
    Nz, Ny, Nx = p_int.shape
    out = np.zeros_like(p_int)
    for axis, (N, topo, d) in {2: (Nx, g.topology[0], g.dx), 1: (Ny, g.topology[1], g.dy)}.items():
        if topo == F:
            continue
        if topo == P:
            flux = (p_int - np.roll(p_int, 1, axis=axis)) / d          # flux at the low face of each cell
            out += (np.roll(flux, -1, axis=axis) - flux) / d
        else:
            dif = np.diff(p_int, axis=axis) / d                        # interior faces
            z = np.zeros_like(np.take(p_int, [0], axis=axis))
            flux = np.concatenate([z, dif, z], axis=axis)              # wall fluxes are zero
            out += np.diff(flux, axis=axis) / d
    if g.topology[2] != F:
        zc = np.concatenate([[0.0], np.cumsum(dz)])
        zc = 0.5 * (zc[1:] + zc[:-1])
        dzf = np.diff(zc)                                              # centre-to-centre, Nz-1 values
        dif = np.diff(p_int, axis=0) / dzf[:, None, None]
        z = np.zeros((1, Ny, Nx))
        flux = np.concatenate([z, dif, z], axis=0)
        out += np.diff(flux, axis=0) / dz[:, None, None]
    return out


def random_velocity(g, seed):
    r = np.random.default_rng(seed)
    st = {"u": None, "v": None, "w": None, "c": []}
    for nm, axis in (("u", 0), ("v", 1), ("w", 2)):
        if g.topology[axis] == F:
            continue
        a = g.zeros()
        g.interior(a)[...] = r.standard_normal((g.Nz, g.Ny, g.Nx))
        if g.topology[axis] == B:                                      # wall faces hold 0
            sl = [slice(None)] * 3
            sl[2 - axis] = 0
            g.interior(a)[tuple(sl)] = 0.0
        st[nm] = a
    return st


TOPOS = [((P, P, B), (12, 10, 7)), ((P, B, B), (9, 8, 6)), ((B, B, B), (6, 7, 5)), ((P, P, F), (12, 9, 1)),
         ((B, P, F), (8, 10, 1))]


@pytest.mark.parametrize("topo,n", TOPOS)
def test_poisson_residual_independent_operator(topo, n):
    """lap(p) == rhs with the operator re-applied by numpy slicing (not the oracle's code)."""
    Nx, Ny, Nz = n
    dz = stretched(Nz) if topo[2] != F else None
    g = make_grid(Nx, Ny, Nz, topo, dz)
    st = random_velocity(g, 1)
    rhs = ref.divergence(g, st)
    p = ref.poisson_solve(g, rhs)
    res = numpy_laplacian(g, g.interior(p), dz if dz is not None else np.ones(1)) - g.interior(rhs)
    assert np.abs(res).max() <= 2e-13 * np.abs(g.interior(rhs)).max()


@pytest.mark.parametrize("topo,n", [((P, P, B), (4, 3, 5)), ((P, B, B), (3, 4, 4)), ((P, P, F), (5, 4, 1))])
def test_poisson_dense_brute_force(topo, n):
    """tiny grids: assemble the operator as a dense matrix column by column with the numpy Laplacian, impose the
    gauge row (R23) and solve with LAPACK."""
    Nx, Ny, Nz = n
    dz = stretched(Nz, 3) if topo[2] != F else np.ones(1)
    g = make_grid(Nx, Ny, Nz, topo, dz if topo[2] != F else None)
    N = Nx * Ny * Nz
    A = np.zeros((N, N))
    for c in range(N):
        e = np.zeros(N)
        e[c] = 1.0
        A[:, c] = numpy_laplacian(g, e.reshape(Nz, Ny, Nx), dz).ravel()
    st = random_velocity(g, 5)
    rhs = ref.divergence(g, st)
    b = g.interior(rhs).ravel().copy()
    # gauge: horizontal mean of level 1 is zero, appended as an extra equation (least squares on a consistent system)
    row = np.zeros(N)
    row[:Nx * Ny] = 1.0
    sol = np.linalg.lstsq(np.vstack([A, row]), np.concatenate([b, [0.0]]), rcond=None)[0]
    p = ref.poisson_solve(g, rhs)
    assert np.abs(g.interior(p).ravel() - sol).max() <= 1e-12 * np.abs(sol).max()
    assert abs(g.interior(p)[0].mean()) <= 1e-14 * np.abs(sol).max()


def test_poisson_closed_form_eigenfunction():
    """uniform grid: cos(2 pi a (i-1)/Nx) cos(2 pi b (j-1)/Ny) cos(pi c (k-1/2)/Nz) is an eigenfunction with the
    textbook eigenvalue -4 sum sin^2(.)/d^2 => p = rhs / lambda."""
    Nx, Ny, Nz, a, b, c = 16, 12, 10, 3, 2, 4
    dx, dy, dz = 0.5, 2.0, 0.25
    g = ref.RefGrid(Nx, Ny, Nz, 3, dx, dy, dz_c=None, dz_uniform=dz, topology=(P, P, B))
    i = np.arange(Nx)[None, None, :]
    j = np.arange(Ny)[None, :, None]
    k = np.arange(Nz)[:, None, None]
    f = np.cos(2 * np.pi * a * i / Nx + 0.3) * np.sin(2 * np.pi * b * j / Ny) * np.cos(np.pi * c * (k + 0.5) / Nz)
    lam = -(4 / dx**2) * np.sin(np.pi * a / Nx)**2 - (4 / dy**2) * np.sin(np.pi * b / Ny)**2 \
          - (4 / dz**2) * np.sin(np.pi * c / (2 * Nz))**2
    rhs = g.zeros()
    g.interior(rhs)[...] = f
    p = ref.poisson_solve(g, rhs)
    assert np.abs(g.interior(p) - f / lam).max() <= 1e-14 * np.abs(f / lam).max()


@pytest.mark.parametrize("topo,n", TOPOS)
def test_projection_makes_velocity_solenoidal_and_is_idempotent(topo, n):
    Nx, Ny, Nz = n
    dz = stretched(Nz, 7) if topo[2] != F else None
    g = make_grid(Nx, Ny, Nz, topo, dz)
    st = random_velocity(g, 11)
    d0 = np.abs(g.interior(ref.divergence(g, st))).max()
    ref.pressure_correction(g, 0.37, st)
    d1 = np.abs(g.interior(ref.divergence(g, st))).max()
    assert d0 > 0.5 and d1 <= 1e-14 * d0
    before = {k: (None if v is None or k == "c" else v.copy()) for k, v in st.items() if k != "c"}
    ref.pressure_correction(g, 0.37, st)
    for nm in ("u", "v", "w"):
        if st[nm] is not None:
            assert np.abs(st[nm] - before[nm]).max() <= 1e-14


def test_projection_removes_a_pure_gradient_and_is_dt_independent():
    """u = discrete grad(phi) with zero wall-normal component is removed entirely (sign and index of (A11));
    the corrected velocity does not depend on dt (R21) while p scales as 1/dt."""
    g = make_grid(10, 8, 6, (P, P, B), stretched(6, 2))
    r = np.random.default_rng(4)
    phi = g.zeros()
    g.interior(phi)[...] = r.standard_normal((6, 8, 10))
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": []}
    ref.pressure_correct(g, -1.0, st, phi)            # u = +grad(phi) on non-wall faces
    assert np.abs(g.interior(st["w"])[0]).max() == 0.0
    sol = random_velocity(g, 9)
    ref.pressure_correction(g, 1.0, sol)              # a solenoidal field
    mix = {nm: st[nm] + sol[nm] for nm in ("u", "v", "w")}
    mix["c"] = []
    mix2 = {nm: mix[nm].copy() for nm in ("u", "v", "w")}
    mix2["c"] = []
    p1 = ref.pressure_correction(g, 1.0, mix)
    p2 = ref.pressure_correction(g, 0.01, mix2)
    for nm in ("u", "v", "w"):
        assert np.abs(mix[nm] - sol[nm]).max() <= 1e-13
        assert np.abs(mix[nm] - mix2[nm]).max() <= 1e-13
    assert np.abs(g.interior(p2) * 0.01 - g.interior(p1)).max() <= 1e-12 * np.abs(p1).max()
    # p equals phi up to the gauge constant: p - phi is uniform
    dif = g.interior(p1) - g.interior(phi)
    assert np.ptp(dif) <= 1e-12 * np.abs(g.interior(phi)).max()


def test_separate_calls_equal_the_long_double_chain():
    g = make_grid(9, 7, 5, (P, P, B), stretched(5, 8))
    a = random_velocity(g, 21)
    b = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in a.items()}
    dt = 0.2
    p = ref.poisson_solve(g, ref.divergence(g, a, 1.0 / dt))
    ref.pressure_correct(g, dt, a, p)
    p2 = ref.pressure_correction(g, dt, b)
    for nm in ("u", "v", "w"):
        assert np.abs(a[nm] - b[nm]).max() <= 1e-13
    assert np.abs(p - p2).max() <= 1e-12 * np.abs(p2).max()


# ------------------------------------------------------------------ N3
def _params(nu=0.3, kappa=(0.7, 0.2)):
    return ref.default_params(n_tracers=len(kappa), nu=nu, kappa=list(kappa) + [0.0] * (8 - len(kappa)))


def _state(g, seed, ntr=2):
    st = random_velocity(g, seed)
    r = np.random.default_rng(seed + 100)
    for _ in range(ntr):
        a = g.zeros()
        g.interior(a)[...] = r.standard_normal((g.Nz, g.Ny, g.Nx))
        st["c"].append(a)
    return st


def _second_difference_z(q, dz, face):
    """numpy: d_z(d_z q) of an interior (Nz,..) array; centred: no-flux walls; face (w at faces 1..Nz, wall at index 0
    and the implicit top wall): Dirichlet 0."""
    zc = np.concatenate([[0.0], np.cumsum(dz)])
    dzf = np.diff(0.5 * (zc[1:] + zc[:-1]))
    if not face:
        dif = np.diff(q, axis=0) / dzf[:, None, None]
        z = np.zeros((1,) + q.shape[1:])
        return np.diff(np.concatenate([z, dif, z], axis=0), axis=0) / dz[:, None, None]
    full = np.concatenate([q, np.zeros((1,) + q.shape[1:])], axis=0)      # faces 1..Nz+1, both walls 0
    dif = np.diff(full, axis=0) / dz[:, None, None]                        # at centres 1..Nz
    out = np.zeros_like(q)
    out[1:] = np.diff(dif, axis=0) / dzf[:, None, None]                    # faces 2..Nz
    return out


def test_implicit_diffusion_inverts_the_numpy_operator():
    Nz = 9
    dz = stretched(Nz, 5)
    g = make_grid(6, 5, Nz, (P, P, B), dz)
    par = _params()
    st = _state(g, 3)
    old = {nm: st[nm].copy() for nm in ("u", "v", "w")}
    oldc = [a.copy() for a in st["c"]]
    dt = 2.5
    ref.implicit_vertical_diffusion(g, par, dt, st)
    for nm, kz in (("u", par["nu"]), ("v", par["nu"]), ("w", par["nu"])):
        q = g.interior(st[nm])
        back = q - dt * kz * _second_difference_z(q, dz, nm == "w")
        assert np.abs(back - g.interior(old[nm])).max() <= 1e-14 * np.abs(old[nm]).max() * 10
    for n, a in enumerate(st["c"]):
        q = g.interior(a)
        back = q - dt * par["kappa"][n] * _second_difference_z(q, dz, False)
        assert np.abs(back - g.interior(oldc[n])).max() <= 1e-13
        # no-flux walls: the column integral is conserved
        assert np.abs(((q - g.interior(oldc[n])) * dz[:, None, None]).sum(axis=0)).max() <= 1e-13
        assert q.max() <= g.interior(oldc[n]).max() + 1e-14 and q.min() >= g.interior(oldc[n]).min() - 1e-14


def test_implicit_diffusion_closed_form_modes():
    """uniform dz: cos(pi m (k-1/2)/Nz) (centred, no-flux) and sin(pi m (k-1)/Nz) (w, zero on the walls) are
    eigenvectors: amplification 1 / (1 + dt kz (4/dz^2) sin^2(pi m / 2Nz))."""
    Nz, m, dzv, dt = 12, 5, 0.5, 3.0
    g = ref.RefGrid(4, 3, Nz, 3, 1.0, 1.0, dz_c=None, dz_uniform=dzv, topology=(P, P, B))
    par = _params(nu=0.4, kappa=(0.9,))
    k = np.arange(Nz)[:, None, None]
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": [g.zeros()]}
    fc = np.cos(np.pi * m * (k + 0.5) / Nz) * np.ones((Nz, 3, 4))
    fw = np.sin(np.pi * m * k / Nz) * np.ones((Nz, 3, 4))
    g.interior(st["c"][0])[...] = fc
    g.interior(st["u"])[...] = fc
    g.interior(st["w"])[...] = fw
    ref.implicit_vertical_diffusion(g, par, dt, st)
    lam = (4 / dzv**2) * np.sin(np.pi * m / (2 * Nz))**2
    assert np.abs(g.interior(st["c"][0]) - fc / (1 + dt * 0.9 * lam)).max() <= 1e-15
    assert np.abs(g.interior(st["u"]) - fc / (1 + dt * 0.4 * lam)).max() <= 1e-15
    assert np.abs(g.interior(st["w"]) - fw / (1 + dt * 0.4 * lam)).max() <= 1e-15


def test_implicit_diffusion_small_dt_is_the_explicit_laplacian():
    """(q_new - q)/dt -> kz d_zz q as dt -> 0: ties (A2) to the oracle's own explicit Laplacian (eq. 8 row 1)."""
    Nz = 8
    dz = stretched(Nz, 6)
    g = make_grid(5, 4, Nz, (P, P, B), dz)
    st = _state(g, 8, ntr=1)
    par = ref.default_params(n_tracers=1, nu=0.0, kappa=[0.6] + [0.0] * 7, adv_x=0, adv_y=0, adv_z=0,
                             momentum_prognostic=0)
    ref.fill_halos(g, par, st)
    # explicit vertical part = full Laplacian tendency of a field that is uniform in x,y
    c = st["c"][0]
    c[...] = c[:, 3:4, 3:4]
    G = ref.compute_tendencies(g, par, st)["c"][0]
    dt = 1e-7
    new = {"u": None, "v": None, "w": None, "c": [c.copy()]}
    ref.implicit_vertical_diffusion(g, par, dt, new)
    rate = (g.interior(new["c"][0]) - g.interior(c)) / dt
    assert np.abs(rate - g.interior(G)).max() <= 1e-5 * np.abs(g.interior(G)).max()


def test_implicit_flag_removes_exactly_the_vertical_diffusion_from_G():
    """(A1) PAPER.md:785-789: with a VerticallyImplicitTimeDiscretization the vertical diffusion is not part of G:
    G(explicit) - G(implicit flag) == kz d_z d_z q, the right-hand operator evaluated by numpy."""
    Nz = 7
    dz = stretched(Nz, 12)
    g = make_grid(6, 5, Nz, (P, P, B), dz)
    st = _state(g, 13, ntr=1)
    par = ref.default_params(n_tracers=1, nu=0.3, kappa=[0.6] + [0.0] * 7, adv_x=0, adv_y=0, adv_z=0)
    ref.fill_halos(g, par, st)
    Ge = ref.compute_tendencies(g, par, st)
    Gi = ref.compute_tendencies(g, dict(par, implicit_vertical_diffusion=1), st)
    for nm, a, b, kz, face in (("u", Ge["u"], Gi["u"], 0.3, False), ("v", Ge["v"], Gi["v"], 0.3, False),
                               ("w", Ge["w"], Gi["w"], 0.3, True), ("c", Ge["c"][0], Gi["c"][0], 0.6, False)):
        q = g.interior(st[nm] if nm != "c" else st["c"][0])
        want = kz * _second_difference_z(q, dz, face)
        got = g.interior(a) - g.interior(b)
        assert np.abs(got - want).max() <= 1e-13 * max(np.abs(want).max(), 1.0), nm
