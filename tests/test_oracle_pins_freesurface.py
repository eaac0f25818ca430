"""Pins of the oracle's N4 routines (split-explicit free surface, (A13)-(A21) PAPER.md:857-923) against what the
mathematics fixes: the closed-form amplification of the forward-backward scheme on a discrete gravity wave, volume
conservation, linear growth under a uniform forcing with the weighted average in closed form, the defining property of
the correction (A21), and numpy column sums."""
import numpy as np
import pytest

from oracle import ocnref as ref

P, B = ref.PERIODIC, ref.BOUNDED


def _grid(Nx, Ny, Nz, topo=(P, P, B), dz=None, dx=1.0, dy=1.0):
    return ref.RefGrid(Nx, Ny, Nz, 3, dx, dy, dz_c=dz, dz_uniform=1.0, topology=topo)


def _dz(Nz, seed=1):
    return 0.5 + 1.5 * np.random.default_rng(seed).random(Nz)


def test_gravity_wave_closed_form_amplification():
    """f = 0, no forcing, one Fourier mode in x: the forward-backward scheme (A18),(A19) is
    eta^{n+1} = eta^n - dtau D+ U^n, U^{n+1} = U^n - dtau g H D- eta^{n+1}; for eta^0 = cos(kx i dx), U^0 = 0 the mode
    amplitude obeys e^{n+1} - 2 e^n + e^{n-1} = -mu e^n, mu = g H dtau^2 (4/dx^2) sin^2(kx dx/2), with e^1 = e^0 (eta
    moves first, with the OLD transport U^0 = 0)  =>  e^n = cos(n theta) + (mu/2) sin(n theta)/sin(theta),
    cos(theta) = 1 - mu/2.  A scheme that used the old eta in (A19), or updated U first, fails this."""
    Nx, Ny, Nz, m = 32, 4, 5, 3
    dz = _dz(Nz)
    H = dz.sum()
    dx, grav, dt, N, M = 2.0, 9.81, 0.9, 6, 11
    g = _grid(Nx, Ny, Nz, dz=dz, dx=dx)
    i = np.arange(Nx)
    bt = {"eta": ref.plane(g), "U": ref.plane(g), "V": ref.plane(g)}
    ref.plane_interior(g, bt["eta"])[...] = np.cos(2 * np.pi * m * i / Nx)[None, :]
    dtau = dt / N
    mu = grav * H * dtau**2 * (4 / dx**2) * np.sin(np.pi * m / Nx)**2
    assert mu < 4                                            # inside the stability limit
    # amplitude recurrence, written for the scalar mode amplitude only: e1 = e0 since U^0 = 0
    e = [1.0, 1.0]
    for n in range(2, M + 1):
        e.append((2 - mu) * e[-1] - e[-2])
    theta = np.arccos(1 - mu / 2)
    n = np.arange(M + 1)
    closed = np.cos(n * theta) + (mu / 2) * np.sin(n * theta) / np.sin(theta)
    assert np.abs(np.array(e) - closed).max() < 1e-12
    for last in (1, 4, M):
        b = {k: v.copy() for k, v in bt.items()}
        w = np.zeros(last)
        w[-1] = 1.0                                          # "average" = the last substep
        ref.barotropic_substeps(g, grav, dt, N, w, b, ref.plane(g), ref.plane(g))
        got = ref.plane_interior(g, b["eta"])
        want = closed[last] * np.cos(2 * np.pi * m * i / Nx)[None, :] * np.ones((Ny, 1))
        assert np.abs(got - want).max() < 1e-13, last
        assert np.abs(ref.plane_interior(g, b["V"])).max() == 0.0


@pytest.mark.parametrize("topo", [(P, P, B), (P, B, B), (B, B, B)])
def test_volume_conservation_and_walls(topo):
    Nx, Ny, Nz = 12, 9, 4
    g = _grid(Nx, Ny, Nz, topo=topo, dz=_dz(Nz, 2))
    r = np.random.default_rng(3)
    bt = {k: ref.plane(g) for k in ("eta", "U", "V")}
    for k in bt:
        ref.plane_interior(g, bt[k])[...] = r.standard_normal((Ny, Nx))
    if topo[0] == B:
        ref.plane_interior(g, bt["U"])[:, 0] = 0
    if topo[1] == B:
        ref.plane_interior(g, bt["V"])[0, :] = 0
    FU, FV = ref.plane(g), ref.plane(g)
    ref.plane_interior(g, FU)[...] = r.standard_normal((Ny, Nx))
    ref.plane_interior(g, FV)[...] = r.standard_normal((Ny, Nx))
    vol0 = ref.plane_interior(g, bt["eta"]).sum()
    w = r.random(7)
    w /= w.sum()
    ref.barotropic_substeps(g, 9.81, 0.05, 5, w, bt, FU, FV)
    assert abs(ref.plane_interior(g, bt["eta"]).sum() - vol0) < 1e-12          # (A16) in flux form, closed / periodic
    if topo[0] == B:
        assert np.abs(ref.plane_interior(g, bt["U"])[:, 0]).max() == 0.0
    if topo[1] == B:
        assert np.abs(ref.plane_interior(g, bt["V"])[0, :]).max() == 0.0


def test_uniform_forcing_gives_linear_growth_and_the_weighted_average():
    """eta = 0, U = U0 uniform, F uniform, periodic: grad eta = 0 forever => U^n = U0 + n dtau F, so
    Ubar = sum a_n (U0 + n dtau F) in closed form, eta stays 0."""
    g = _grid(8, 6, 3, dz=_dz(3, 4))
    bt = {k: ref.plane(g) for k in ("eta", "U", "V")}
    ref.plane_interior(g, bt["U"])[...] = 0.7
    ref.plane_interior(g, bt["V"])[...] = -0.2
    FU, FV = ref.plane(g), ref.plane(g)
    ref.plane_interior(g, FU)[...] = 0.3
    ref.plane_interior(g, FV)[...] = 0.11
    a = np.array([0.1, 0.0, 0.25, 0.4, 0.25])
    dt, N = 2.0, 4
    ref.barotropic_substeps(g, 9.81, dt, N, a, bt, FU, FV)
    n = np.arange(1, 6)
    assert np.abs(ref.plane_interior(g, bt["U"]) - (a * (0.7 + n * dt / N * 0.3)).sum()).max() < 1e-15
    assert np.abs(ref.plane_interior(g, bt["V"]) - (a * (-0.2 + n * dt / N * 0.11)).sum()).max() < 1e-15
    assert np.abs(bt["eta"]).max() == 0.0


def test_column_integral_and_forcing_are_numpy_dot_products():
    Nx, Ny, Nz = 7, 5, 6
    dz = _dz(Nz, 5)
    g = _grid(Nx, Ny, Nz, topo=(P, B, B), dz=dz)
    r = np.random.default_rng(6)
    u, v, Gp = g.zeros(), g.zeros(), g.zeros()
    for a in (u, v, Gp):
        g.interior(a)[...] = r.standard_normal((Nz, Ny, Nx))
    U = ref.column_integral(g, u, 0)
    V = ref.column_integral(g, v, 1)
    assert np.abs(ref.plane_interior(g, U) - np.tensordot(dz, g.interior(u), axes=(0, 0))).max() < 1e-14
    wantV = np.tensordot(dz, g.interior(v), axes=(0, 0))
    wantV[0, :] = 0                                                              # wall face j = 1
    assert np.abs(ref.plane_interior(g, V) - wantV).max() < 1e-14
    FU, FV = ref.barotropic_forcing(g, 0.75, 0.4, {"u": u, "v": v}, {"u": Gp, "v": Gp})
    assert np.abs(ref.plane_interior(g, FU) - np.tensordot(dz, 0.75 * g.interior(u) - 0.4 * g.interior(Gp), axes=(0, 0))).max() < 1e-14
    FU1, _ = ref.barotropic_forcing(g, 0.5, 0.0, {"u": u, "v": v}, None)
    assert np.abs(ref.plane_interior(g, FU1) - 0.5 * np.tensordot(dz, g.interior(u), axes=(0, 0))).max() < 1e-14


def test_correction_sets_the_transport_and_keeps_the_baroclinic_part():
    """(A21): afterwards sum_k dz u = Ubar exactly, and u - (depth mean of u) is unchanged."""
    Nx, Ny, Nz = 9, 8, 7
    dz = _dz(Nz, 7)
    H = dz.sum()
    g = _grid(Nx, Ny, Nz, topo=(P, B, B), dz=dz)
    r = np.random.default_rng(8)
    st = {"u": g.zeros(), "v": g.zeros()}
    for a in st.values():
        g.interior(a)[...] = r.standard_normal((Nz, Ny, Nx))
    g.interior(st["v"])[:, 0, :] = 0
    old = {k: a.copy() for k, a in st.items()}
    bt = {"eta": ref.plane(g), "U": ref.plane(g), "V": ref.plane(g)}
    ref.plane_interior(g, bt["U"])[...] = r.standard_normal((Ny, Nx))
    ref.plane_interior(g, bt["V"])[...] = r.standard_normal((Ny, Nx))
    ref.barotropic_correct(g, st, bt)
    for nm, key in (("u", "U"), ("v", "V")):
        q, q0 = g.interior(st[nm]), g.interior(old[nm])
        tr = np.tensordot(dz, q, axes=(0, 0))
        want = ref.plane_interior(g, bt[key]).copy()
        mean0 = np.tensordot(dz, q0, axes=(0, 0)) / H
        dev_new = q - tr / H
        dev_old = q0 - mean0
        if nm == "v":
            want[0, :] = 0
            assert np.abs(q[:, 0, :]).max() == 0.0                               # wall faces untouched
            dev_new, dev_old, tr, want = dev_new[:, 1:], dev_old[:, 1:], tr[1:], want[1:]
        assert np.abs(tr - want).max() < 1e-13
        assert np.abs(dev_new - dev_old).max() < 1e-13


def test_instability_beyond_the_forward_backward_limit():
    """mu > 4 (c dtau K > 2) must blow up, mu < 4 must stay bounded: pins dtau = dt / N."""
    Nx = 16
    g = _grid(Nx, 4, 2)
    H, grav = 2.0, 9.81
    i = np.arange(Nx)
    kmax = 4.0                                                # (4/dx^2) sin^2(pi/2) at the grid scale
    for N, bounded in ((10, True), (4, False)):
        dt = 1.0
        mu = grav * H * (dt / N)**2 * kmax
        assert (mu < 4) == bounded
        bt = {k: ref.plane(g) for k in ("eta", "U", "V")}
        ref.plane_interior(g, bt["eta"])[...] = ((-1.0) ** i)[None, :]
        w = np.zeros(60)
        w[-1] = 1
        ref.barotropic_substeps(g, grav, dt, N, w, bt, ref.plane(g), ref.plane(g))
        amp = np.abs(ref.plane_interior(g, bt["eta"])).max()
        assert (amp < 10) == bounded, (N, amp)
