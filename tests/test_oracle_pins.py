"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in the
oracle (dropped term, wrong sign or index, transposed operand, wrong constant) fails at least one.
"""
import itertools
import math
import os
from fractions import Fraction

import numpy as np
import pytest

P, B, F = 0, 1, 2
GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- helpers
def mkgrid(ref, Nx, Ny, Nz, topo, dx=1.0, dy=1.0, dz=1.0, dz_c=None, H=3):
    return ref.RefGrid(Nx, Ny, Nz, H, dx, dy, dz_c=dz_c, dz_uniform=dz, topology=topo)


def setint(g, a, vals):
    g.interior(a)[...] = vals


def rand_state(ref, g, rng, n_tracers=1, with_w=True, scale=1.0):
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros() if with_w else None, "c": [g.zeros() for _ in range(n_tracers)]}
    for k in ("u", "v", "w"):
        if st[k] is not None:
            setint(g, st[k], scale * rng.standard_normal((g.Nz, g.Ny, g.Nx)))
    for c in st["c"]:
        setint(g, c, rng.standard_normal((g.Nz, g.Ny, g.Nx)))
    return st


def solenoidal_periodic(g, rng, scale=1.0):
    """discrete curl of a random periodic vector potential: exactly non-divergent to rounding."""
    A = [rng.standard_normal((g.Nz, g.Ny, g.Nx)) for _ in range(3)]
    rx = lambda a: np.roll(a, -1, axis=2)
    ry = lambda a: np.roll(a, -1, axis=1)
    rz = lambda a: np.roll(a, -1, axis=0)
    u = (ry(A[2]) - A[2]) / g.dy - (rz(A[1]) - A[1]) / 1.0
    v = (rz(A[0]) - A[0]) / 1.0 - (rx(A[2]) - A[2]) / g.dx
    w = (rx(A[1]) - A[1]) / g.dx - (ry(A[0]) - A[0]) / g.dy
    return scale * u, scale * v, scale * w


def volumes(g):
    dzc = g.metric("dzc")
    return g.dx * g.dy * dzc[:, None, None] * np.ones((g.Nz, g.Ny, g.Nx))


# ----------------------------------------------------------------------------- grid metrics
def test_grid_listing15_centres(ref):
    """faces [0,.2,.3,.7,1] -> centres [.1,.25,.5,.85] (here along z, surface at 0)."""
    with open(os.path.join(GOLD, "listing15_grid.txt")) as fh:
        rows = [l.split("#")[0].split() for l in fh if l.strip() and not l.startswith("#")]
    faces = np.array([float(x) for x in rows[0]])
    centres = np.array([float(x) for x in rows[1]])
    dz = np.diff(faces)
    g = mkgrid(ref, 4, 4, 4, (P, P, B), dz_c=dz)
    assert np.allclose(g.metric("zf"), faces - faces[-1], atol=1e-15)
    assert np.allclose(g.metric("zc"), centres - faces[-1], atol=1e-15)
    assert np.allclose(g.metric("dzf"), np.diff(centres), atol=1e-15)
    assert np.allclose(g.metric("dzc"), dz, atol=0)


def test_grid_c3_column(ref):
    """C3 column: min(250, 10*1.08^n), 42 geometric + 8 capped levels, depth 5042.435 m (arithmetic)."""
    from paper_2502_14148_b200.workloads import c3_dz
    dz = c3_dz(50)
    assert dz[-1] == 10.0 and np.sum(dz == 250.0) == 8
    depth = sum(min(250.0, 10.0 * 1.08 ** n) for n in range(50))
    g = mkgrid(ref, 4, 4, 50, (P, B, B), dz_c=dz)
    assert abs(g.metric("zf")[0] + depth) < 1e-9 and abs(depth - 5042.435) < 1e-3
    assert g.metric("zf")[-1] == 0.0


# ----------------------------------------------------------------------------- halo fill
def test_halo_periodic_shift_commutes(ref):
    rng = np.random.default_rng(1)
    g = mkgrid(ref, 7, 6, 5, (P, P, P))
    a = g.zeros(); setint(g, a, rng.standard_normal((5, 6, 7)))
    b = g.zeros(); setint(g, b, np.roll(g.interior(a), 1, axis=2))
    ref.fill_halos_field(g, a, (0, 0, 0)); ref.fill_halos_field(g, b, (1, 0, 0))
    # shifting by one cell then filling == filling then reading one cell to the left
    assert np.array_equal(b[:, :, 1:], a[:, :, :-1])
    # periodic wrap, corners included
    assert g.at(a, 0, 0, 0) == g.at(a, 7, 6, 5) and g.at(a, 8, 7, 6) == g.at(a, 1, 1, 1)
    assert g.at(a, -2, 3, 8) == g.at(a, 5, 3, 3)


def test_halo_bounded_mirror_and_walls(ref):
    rng = np.random.default_rng(2)
    g = mkgrid(ref, 6, 5, 4, (B, B, B))
    c = g.zeros(); setint(g, c, rng.standard_normal((4, 5, 6)))
    ref.fill_halos_field(g, c, (0, 0, 0))
    for m in (1, 2, 3):
        assert g.at(c, 1 - m, 2, 2) == g.at(c, m, 2, 2) and g.at(c, 6 + m, 2, 2) == g.at(c, 7 - m, 2, 2)
        assert g.at(c, 2, 1 - m, 2) == g.at(c, 2, m, 2) and g.at(c, 2, 2, 4 + m) == g.at(c, 2, 2, 5 - m)
    assert g.at(c, 0, 0, 0) == g.at(c, 1, 1, 1) and g.at(c, -1, 7, 6) == g.at(c, 2, 4, 3)   # corners
    u = g.zeros(); setint(g, u, rng.standard_normal((4, 5, 6)))
    ref.fill_halos_field(g, u, (1, 0, 0))
    assert np.all(u[:, :, :4] == 0.0) and np.all(u[:, :, 3 + 6:] == 0.0)     # wall face 1, beyond, face N+1, beyond
    assert g.at(u, 2, 0, 1) == g.at(u, 2, 1, 1)                               # tangential direction mirrors
    # order of axes does not matter for the result: fill twice == fill once
    u2 = u.copy(); ref.fill_halos_field(g, u2, (1, 0, 0))
    assert np.array_equal(u, u2)


# ----------------------------------------------------------------------------- 1-D reconstructions
def _cell_averages(poly, edges):
    P_ = np.polynomial.Polynomial(poly).integ()
    return (P_(edges[1:]) - P_(edges[:-1])) / np.diff(edges)


def test_weno_candidates_exact_for_quadratics(ref):
    """(B9) PAPER.md:1039: each candidate — hence W5 for any weights — is exact for cell averages of degree<=2."""
    rng = np.random.default_rng(3)
    for _ in range(20):
        poly = rng.standard_normal(3)
        h = rng.uniform(0.3, 2.0)
        edges = h * (np.arange(6) - 3.0)          # cells m-3..m+1, interface at x=0 between cell 2 and 3
        qa = _cell_averages(poly, edges)
        exact = np.polynomial.Polynomial(poly)(0.0)
        assert abs(ref.weno5z(qa, 1e-8) - exact) < 1e-13 * (1 + abs(exact))
        # right-biased: mirror image about the interface
        edges_r = h * (np.arange(6) - 2.0)
        qr = _cell_averages(poly, edges_r)[::-1]
        assert abs(ref.weno5z(qr, 1e-8) - exact) < 1e-13 * (1 + abs(exact))


def test_weno_linear_limit_fifth_order(ref):
    """huge eps => ideal weights (1/10,6/10,3/10) => (2a-13b+47c+27d-3e)/60, exact to degree 4."""
    rng = np.random.default_rng(4)
    q = rng.standard_normal(5)
    lin = (2 * q[0] - 13 * q[1] + 47 * q[2] + 27 * q[3] - 3 * q[4]) / 60.0
    assert abs(ref.weno5z(q, 1e40) - lin) < 1e-14
    poly = rng.standard_normal(5)
    edges = np.arange(6) - 3.0
    qa = _cell_averages(poly, edges)
    assert abs(ref.weno5z(qa, 1e40) - poly[0]) < 1e-12
    # linear data: all indicators equal => tau5 = 0 => ideal weights even with the small eps
    a = 0.3 + 0.7 * np.arange(5)
    assert abs(ref.weno5z(a, 1e-8) - (0.3 + 0.7 * 2.5)) < 1e-14


def _beta_from_definition(q3, offset):
    """Jiang-Shu smoothness indicator from its definition: sum_l h^(2l-1) int (d^l p/dx^l)^2 dx over the upwind
    cell [-1,0], p = the quadratic whose cell averages on the three cells starting at x=offset are q3."""
    M = np.zeros((3, 3))
    for r in range(3):
        lo, hi = offset + r, offset + r + 1
        for n in range(3):
            M[r, n] = (hi ** (n + 1) - lo ** (n + 1)) / (n + 1)
    p = np.polynomial.Polynomial(np.linalg.solve(M, q3))
    d1, d2 = p.deriv(1), p.deriv(2)
    I1 = (d1 * d1).integ(); I2 = (d2 * d2).integ()
    return (I1(0.0) - I1(-1.0)) + (I2(0.0) - I2(-1.0))


def test_weno_z_weights_from_indicator_definition(ref):
    """WENO-Z (R1,R2): indicators computed from their integral definition, tau5=|b1-b-1|, exponent 2."""
    rng = np.random.default_rng(5)
    for trial in range(20):
        q = rng.standard_normal(5) * 10.0 ** rng.integers(-3, 2)
        eps = 1e-8
        a, b, c, d, e = q
        beta = [_beta_from_definition(q[0:3], -3.0), _beta_from_definition(q[1:4], -2.0), _beta_from_definition(q[2:5], -1.0)]
        cand = [(2 * a - 7 * b + 11 * c) / 6, (-b + 5 * c + 2 * d) / 6, (2 * c + 5 * d - e) / 6]   # (B9)
        dk = [0.1, 0.6, 0.3]
        tau = abs(beta[0] - beta[2])
        al = [dk[s] * (1 + (tau / (beta[s] + eps)) ** 2) for s in range(3)]
        expect = sum(al[s] * cand[s] for s in range(3)) / sum(al)
        got = ref.weno5z(q, eps)
        assert abs(got - expect) < 2e-12 * max(1.0, np.abs(q).max()), (trial, got, expect)


def test_weno_properties(ref):
    rng = np.random.default_rng(6)
    q = rng.standard_normal(9)
    m = 4
    # W5R(q) == W5L(reversed q) about the interface
    qr = q[::-1].copy()
    assert ref.reconstruct(q, m, -5) == pytest.approx(ref.reconstruct(qr, len(q) - m, 5), abs=1e-15)
    # translation equivariance and scaling of the convex combination
    assert ref.reconstruct(q + 7.5, m, 5) == pytest.approx(ref.reconstruct(q, m, 5) + 7.5, abs=1e-13)
    # essentially non-oscillatory at a step: (0,0,0,1,1) -> ~0 and within [min,max]
    val = ref.weno5z([0, 0, 0, 1, 1])
    assert -1e-12 <= val < 1e-6
    val = ref.weno5z([1, 1, 1, 0, 0])
    assert 1 - 1e-6 < val <= 1 + 1e-12
    # float and double instantiations agree with long double to their precision
    x = ref.weno5z(q[:5], 1e-8, 0)
    assert abs(ref.weno5z(q[:5], 1e-8, 1) - x) < 1e-14 and abs(ref.weno5z(q[:5], 1e-8, 2) - x) < 2e-6


def test_centered_and_upwind_stencils(ref):
    """(B4), (B5), (B6), (B7) PAPER.md:1007-1026."""
    rng = np.random.default_rng(7)
    q = rng.standard_normal(8); m = 4
    assert ref.reconstruct(q, m, 2) == pytest.approx(0.5 * (q[m] + q[m - 1]), abs=1e-16)
    assert ref.reconstruct(q, m, 3) == pytest.approx((-q[m - 2] + 5 * q[m - 1] + 2 * q[m]) / 6, abs=1e-15)
    assert ref.reconstruct(q, m, -3) == pytest.approx((2 * q[m - 1] + 5 * q[m] - q[m + 1]) / 6, abs=1e-15)
    # Centered(4) is the symmetric part of UpwindBiased(3)  (B7)
    assert ref.reconstruct(q, m, 4) == pytest.approx(0.5 * (ref.reconstruct(q, m, 3) + ref.reconstruct(q, m, -3)), abs=1e-15)
    # (B6): u [c]^1 = u <c> - (|u| dx/2) (c_i - c_{i-1})/dx, both signs; zero velocity gives zero
    for uu in (0.7, -1.3):
        lhs = ref.upwind_flux(q, m, 1, uu)
        rhs = uu * 0.5 * (q[m] + q[m - 1]) - abs(uu) / 2 * (q[m] - q[m - 1])
        assert lhs == pytest.approx(rhs, abs=1e-15)
    for sch in (1, 2, 5):
        assert ref.upwind_flux(q, m, sch, 0.0) == 0.0
    # upwind selection of WENO: a>0 left-biased, a<0 right-biased
    assert ref.upwind_flux(q, m, 5, 2.0) == pytest.approx(2.0 * ref.reconstruct(q, m, 5), abs=1e-15)
    assert ref.upwind_flux(q, m, 5, -2.0) == pytest.approx(-2.0 * ref.reconstruct(q, m, -5), abs=1e-15)


# ----------------------------------------------------------------------------- RK3
def test_rk3_constants_and_amplification(ref):
    """(A4) PAPER.md:799-801: gamma=(8/15,5/12,3/4), zeta=(0,17/60,5/12); self-starting; third order."""
    with open(os.path.join(GOLD, "rk3_coefficients.txt")) as fh:
        rows = [l.split() for l in fh if l.strip() and not l.startswith("#")]
    gam = [Fraction(x) for x in rows[0]]; zet = [Fraction(x) for x in rows[1]]
    for s in (1, 2, 3):
        gg, zz = ref.rk3_coefficients(s)
        assert gg == float(gam[s - 1]) and zz == float(zet[s - 1])
    assert zet[0] == 0 and sum(g - z for g, z in zip(gam, zet)) == 1
    # dq/dt = lambda q through the oracle's substage: q3/q0 = 1 + z + z^2/2 + z^3/6
    g = mkgrid(ref, 4, 4, 4, (P, P, P))
    prm = ref.default_params(n_tracers=1, momentum_prognostic=0)
    lam, dt = -0.37, 0.9
    c = g.zeros(); setint(g, c, 1.25)
    st = {"u": None, "v": None, "w": None, "c": [c]}
    Gp = None
    for s in (1, 2, 3):
        G = {"c": [lam * c.copy()]}
        ref.rk3_substage(g, prm, s, dt, st, G, Gp)
        Gp = G
    z = lam * dt
    assert np.allclose(g.interior(c), 1.25 * (1 + z + z * z / 2 + z ** 3 / 6), rtol=1e-15)
    assert np.all(c[0] == 0.0)   # halos untouched


def test_substage_skips_walls(ref):
    g = mkgrid(ref, 5, 4, 3, (B, P, B))
    prm = ref.default_params(n_tracers=1)
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": [g.zeros()]}
    G = {"u": g.zeros() + 1.0, "v": g.zeros() + 1.0, "w": g.zeros() + 1.0, "c": [g.zeros() + 1.0]}
    ref.substage(g, prm, 1.0, 0.0, 2.0, st, G, None)
    assert np.all(g.interior(st["c"][0]) == 2.0) and np.all(g.interior(st["v"]) == 2.0)
    assert np.all(g.interior(st["u"])[:, :, 0] == 0.0) and np.all(g.interior(st["u"])[:, :, 1:] == 2.0)
    assert np.all(g.interior(st["w"])[0] == 0.0) and np.all(g.interior(st["w"])[1:] == 2.0)


# ----------------------------------------------------------------------------- tendencies: invariants
def test_constant_fields_zero_tendency(ref):
    """constant c + discretely non-divergent velocity => G_c = 0; uniform flow => advective G_u = 0."""
    rng = np.random.default_rng(8)
    g = mkgrid(ref, 10, 9, 8, (P, P, P))
    u, v, w = solenoidal_periodic(g, rng)
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": [g.zeros()]}
    setint(g, st["u"], u); setint(g, st["v"], v); setint(g, st["w"], w); setint(g, st["c"][0], 3.7)
    prm = ref.default_params(n_tracers=1, momentum_prognostic=0, kappa=[0.3] + [0] * 7)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    assert np.abs(g.interior(G["c"][0])).max() < 1e-13
    st2 = {"u": g.zeros() + 0.3, "v": g.zeros() - 0.2, "w": g.zeros() + 0.1, "c": []}
    prm2 = ref.default_params(n_tracers=0, nu=0.5)
    G2 = ref.compute_tendencies(g, prm2, st2)
    for k in "uvw":
        assert np.abs(g.interior(G2[k])).max() < 1e-15


@pytest.mark.parametrize("topo", [(P, P, P), (P, P, B), (B, B, B)])
def test_conservation(ref, topo):
    """(B1),(B2) PAPER.md:927-931, 990-994: sum V G = 0 for flux-divergence terms on periodic / closed domains."""
    rng = np.random.default_rng(9)
    dz = np.array([0.5, 0.7, 1.0, 1.4, 0.9, 0.6, 0.8]) if topo[2] == B else None
    g = mkgrid(ref, 9, 8, 7, topo, dx=0.8, dy=1.3, dz_c=dz)
    st = rand_state(ref, g, rng, n_tracers=1)
    adv_z = 2 if dz is not None else 5
    prm = ref.default_params(n_tracers=1, nu=0.2, kappa=[0.3] + [0] * 7, adv_z=adv_z)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    V = volumes(g)
    scale = np.abs(g.interior(G["c"][0]) * V).sum()
    assert abs((g.interior(G["c"][0]) * V).sum()) < 1e-13 * scale
    if topo[0] == P:   # momentum: u control volumes tile the periodic domain (uniform dx)
        su = np.abs(g.interior(G["u"]) * V).sum()
        assert abs((g.interior(G["u"]) * V).sum()) < 1e-13 * su
        assert abs((g.interior(G["v"]) * V).sum()) < 1e-13 * su


def test_axis_swap_symmetry(ref):
    """x<->y and x<->z relabelling of all inputs relabels the outputs (tests the y/z code against the x code)."""
    rng = np.random.default_rng(10)
    n = 8
    g = mkgrid(ref, n, n, n, (P, P, P))
    st = rand_state(ref, g, rng, n_tracers=1)
    prm = ref.default_params(n_tracers=1, nu=0.1, kappa=[0.2] + [0] * 7)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    for perm, names in (((0, 2, 1), ("v", "u", "w")), ((2, 1, 0), ("w", "v", "u"))):
        # arrays are indexed (k,j,i): transposing array axes (1,2) swaps x<->y, (0,2) swaps x<->z
        st2 = {"u": np.ascontiguousarray(st[names[0]].transpose(perm)),
               "v": np.ascontiguousarray(st[names[1]].transpose(perm)),
               "w": np.ascontiguousarray(st[names[2]].transpose(perm)),
               "c": [np.ascontiguousarray(st["c"][0].transpose(perm))]}
        G2 = ref.compute_tendencies(g, prm, st2)
        for a, b in zip(("u", "v", "w"), names):
            assert np.allclose(g.interior(G2[a]), g.interior(G[b].transpose(perm)), rtol=0, atol=1e-13)
        assert np.allclose(g.interior(G2["c"][0]), g.interior(G["c"][0].transpose(perm)), rtol=0, atol=1e-13)


def test_laplacian_eigenmodes(ref):
    """periodic: cos(k.x) eigenvalue -kappa sum 4/d^2 sin^2(k d/2); bounded (mirror halos): cos(pi n (i-1/2)/N)."""
    g = mkgrid(ref, 12, 10, 8, (P, P, P), dx=0.5, dy=0.8, dz=1.25)
    n = (2, 3, 1)
    kx, ky, kz = 2 * np.pi * n[0] / (12 * 0.5), 2 * np.pi * n[1] / (10 * 0.8), 2 * np.pi * n[2] / (8 * 1.25)
    K, J, I = np.meshgrid(np.arange(8), np.arange(10), np.arange(12), indexing="ij")
    mode = np.cos(kx * (I + 0.5) * 0.5 + ky * (J + 0.5) * 0.8 + kz * (K + 0.5) * 1.25 + 0.3)
    kap = 0.7
    lam = -kap * (4 / 0.25 * np.sin(kx * 0.5 / 2) ** 2 + 4 / 0.64 * np.sin(ky * 0.8 / 2) ** 2 + 4 / 1.5625 * np.sin(kz * 1.25 / 2) ** 2)
    st = {"u": None, "v": None, "w": None, "c": [g.zeros()]}
    setint(g, st["c"][0], mode)
    prm = ref.default_params(n_tracers=1, momentum_prognostic=0, kappa=[kap] + [0] * 7)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    assert np.allclose(g.interior(G["c"][0]), lam * mode, rtol=0, atol=1e-13)
    # momentum Laplacians use the same operator (nu): u-field with the same mode
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": []}
    for kname in "uvw":
        setint(g, st[kname], 1e-9 * mode)      # tiny amplitude: advection is O(1e-18)
    prm = ref.default_params(nu=kap)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    for kname in "uvw":
        assert np.allclose(g.interior(G[kname]), lam * 1e-9 * mode, rtol=0, atol=1e-17)
    # bounded in z: Neumann cosine mode
    g = mkgrid(ref, 6, 6, 10, (P, P, B), dz=0.4)
    K = np.arange(10)[:, None, None] * np.ones((10, 6, 6))
    mode = np.cos(np.pi * 3 * (K + 0.5) / 10)
    st = {"u": None, "v": None, "w": None, "c": [g.zeros()]}
    setint(g, st["c"][0], mode)
    prm = ref.default_params(n_tracers=1, momentum_prognostic=0, kappa=[kap] + [0] * 7)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    assert np.allclose(g.interior(G["c"][0]), -kap * 4 / 0.16 * np.sin(np.pi * 3 / 20) ** 2 * mode, rtol=0, atol=1e-13)


def test_laplacian_stretched_symmetric(ref):
    """stretched z: the operator V*Lap is symmetric and sums to zero (closed column)."""
    dz = np.array([0.3, 0.5, 0.9, 1.4, 0.7, 0.4])
    g = mkgrid(ref, 4, 4, 6, (P, P, B), dz_c=dz)
    prm = ref.default_params(n_tracers=1, momentum_prognostic=0, kappa=[1.0] + [0] * 7)
    M = np.zeros((6, 6))
    for k in range(6):
        st = {"u": None, "v": None, "w": None, "c": [g.zeros()]}
        g.interior(st["c"][0])[k] = 1.0
        ref.fill_halos(g, prm, st)
        G = ref.compute_tendencies(g, prm, st)
        M[:, k] = g.interior(G["c"][0])[:, 0, 0] * dz
    assert np.allclose(M, M.T, atol=1e-14) and np.allclose(M.sum(axis=0), 0, atol=1e-14)
    # interior row equals the textbook three-point formula
    zc = g.metric("zc")
    k = 2
    assert M[k, k + 1] == pytest.approx(1.0 / (zc[k + 1] - zc[k]), rel=1e-14)
    assert M[k, k - 1] == pytest.approx(1.0 / (zc[k] - zc[k - 1]), rel=1e-14)


def test_coriolis_and_buoyancy_uniform(ref):
    """uniform (u0,v0) on an f-plane: G_u = f v0, G_v = -f u0; uniform T,S: G_w = g(alpha T - beta S), walls 0."""
    g = mkgrid(ref, 6, 5, 4, (P, P, B))
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": [g.zeros(), g.zeros()]}
    setint(g, st["u"], 0.3); setint(g, st["v"], -0.2); setint(g, st["c"][0], 20.0); setint(g, st["c"][1], 35.0)
    prm = ref.default_params(n_tracers=2, idx_T=0, idx_S=1, f0=1e-4, g=9.81, alpha_T=2e-4, beta_S=8e-4)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    assert np.allclose(g.interior(G["u"]), 1e-4 * -0.2, rtol=1e-14)
    assert np.allclose(g.interior(G["v"]), -1e-4 * 0.3, rtol=1e-14)
    b = 9.81 * (2e-4 * 20.0 - 8e-4 * 35.0)
    assert np.allclose(g.interior(G["w"])[1:], b, rtol=1e-14) and np.all(g.interior(G["w"])[0] == 0.0)
    # beta-plane: f evaluated at the tendency's own y (R8, R12)
    prm = ref.default_params(n_tracers=0, f0=1e-4, beta_coriolis=2e-11, y0=0.0, adv_x=0, adv_y=0, adv_z=0)
    g2 = mkgrid(ref, 6, 5, 4, (P, B, B), dy=5000.0)
    st = {"u": g2.zeros(), "v": g2.zeros(), "w": None, "c": []}
    setint(g2, st["u"], 0.3); setint(g2, st["v"], -0.2)
    prm["hydrostatic"] = 1
    ref.fill_halos(g2, prm, st)
    G = ref.compute_tendencies(g2, prm, st)
    j = np.arange(1, 6)
    fu = 1e-4 + 2e-11 * (j - 0.5) * 5000.0
    vbar = np.array([-0.1, -0.2, -0.2, -0.2, -0.1])       # wall faces j=1 and Ny+1 carry v=0
    assert np.allclose(g2.interior(G["u"])[0, :, 0], fu * vbar, rtol=1e-13)
    fv = 1e-4 + 2e-11 * (j - 1.0) * 5000.0
    assert g2.interior(G["v"])[0, 0, 0] == 0.0
    assert np.allclose(g2.interior(G["v"])[0, 1:, 0], -fv[1:] * 0.3, rtol=1e-13)


def test_coriolis_energy_neutral(ref):
    """periodic f-plane: sum(u f vbar - v f ubar) = 0 (the two 4-point averages are adjoint)."""
    rng = np.random.default_rng(11)
    g = mkgrid(ref, 8, 7, 3, (P, P, P))
    st = rand_state(ref, g, rng, n_tracers=0)
    prm = ref.default_params(f0=0.9, adv_x=0, adv_y=0, adv_z=0)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    e = (g.interior(st["u"]) * g.interior(G["u"]) + g.interior(st["v"]) * g.interior(G["v"])).sum()
    assert abs(e) < 1e-12 and np.abs(g.interior(G["w"])).max() == 0.0


# ----------------------------------------------------------------------------- column scans
def test_w_from_continuity(ref):
    """(15) PAPER.md:456-458: after the scan the discrete divergence vanishes; u = a x => w = -a (z - z_bottom)."""
    rng = np.random.default_rng(12)
    dz = np.array([4.0, 3.0, 2.0, 1.5, 1.0])
    g = mkgrid(ref, 7, 6, 5, (P, B, B), dx=2.0, dy=3.0, dz_c=dz)
    st = rand_state(ref, g, rng, n_tracers=0)
    prm = ref.default_params(hydrostatic=1, adv_z=2)
    ref.fill_halos(g, prm, st)
    st["w"][...] = np.nan
    ref.compute_w(g, st)
    u, v, w = st["u"], st["v"], st["w"]
    H = 3
    div = ((u[H:H + 5, H:H + 6, H + 1:H + 8] - u[H:H + 5, H:H + 6, H:H + 7]) / 2.0
           + (v[H:H + 5, H + 1:H + 7, H:H + 7] - v[H:H + 5, H:H + 6, H:H + 7]) / 3.0
           + (w[H + 1:H + 6, H:H + 6, H:H + 7] - w[H:H + 5, H:H + 6, H:H + 7]) / dz[:, None, None])
    assert np.abs(div).max() < 1e-15
    assert np.all(w[H, H:H + 6, H:H + 7] == 0.0)
    # horizontal halos of w come out consistent with periodic wrap in x
    assert np.allclose(w[H:H + 6, H:H + 6, H - 1], w[H:H + 6, H:H + 6, H + 6], atol=1e-16)
    # analytic: u = a x_f (x bounded to avoid the periodic jump), v = 0
    g = mkgrid(ref, 6, 4, 5, (B, B, B), dx=2.0, dy=3.0, dz_c=dz)
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": []}
    a = 0.05
    # fill u directly everywhere (including halos) with the linear profile; no halo fill
    for i in range(1 - 3, 6 + 3 + 1):
        st["u"][:, :, i - 1 + 3] = a * (i - 1) * 2.0
    ref.compute_w(g, st)
    zf = g.metric("zf")
    assert np.allclose(st["w"][3:3 + 6, 4, 5], -a * (zf - zf[0]), rtol=1e-14, atol=1e-16)


def test_hydrostatic_pressure(ref):
    """(14) PAPER.md:452-454: uniform b0 => p = b0 z_c, zero horizontal gradient."""
    dz = np.array([4.0, 3.0, 2.0, 1.5, 1.0])
    g = mkgrid(ref, 5, 4, 5, (P, B, B), dz_c=dz)
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": [g.zeros() + 20.0, g.zeros() + 35.0]}
    prm = ref.default_params(n_tracers=2, idx_T=0, idx_S=1, g=9.81, alpha_T=2e-4, beta_S=8e-4, hydrostatic=1, adv_z=2)
    p = ref.compute_phy(g, prm, st)
    b0 = 9.81 * (2e-4 * 20 - 8e-4 * 35)
    assert np.allclose(p[3:8], (b0 * g.metric("zc"))[:, None, None] * np.ones((5, 10, 11)), rtol=1e-14)
    # linear-in-z stratification: trapezoid rule is exact for the quadratic pressure up to the surface half cell
    zc = g.metric("zc")
    T = g.zeros(); T[3:8] = (20 + 0.01 * zc)[:, None, None]
    st["c"][0] = T
    prm["T_ref"] = 20 + 0.01 * zc; prm["S_ref"] = np.full(5, 35.0)
    p = ref.compute_phy(g, prm, st)
    assert np.abs(p[3:8]).max() < 1e-15   # anomalies vanish identically with matching references


# ----------------------------------------------------------------------------- exact shift and top hat
def test_upwind1_exact_shift(ref):
    """north_star: uniform u>0, u dt/dx = 1, first-order upwind, forward Euler => exact one-cell shift (bitwise)."""
    rng = np.random.default_rng(13)
    g = mkgrid(ref, 16, 4, 1, (P, P, F), dx=0.5)
    c0 = rng.integers(-50, 50, size=(1, 4, 16)).astype(np.float64)
    st = {"u": g.zeros(), "v": g.zeros(), "w": None, "c": [g.zeros()]}
    setint(g, st["u"], 2.0); setint(g, st["c"][0], c0)
    prm = ref.default_params(n_tracers=1, momentum_prognostic=0, adv_x=1, adv_y=1, adv_z=0)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    ref.substage(g, prm, 1.0, 0.0, 0.25, st, G, None)
    assert np.array_equal(g.interior(st["c"][0]), np.roll(c0, 1, axis=2))
    # negative velocity along y shifts the other way
    g = mkgrid(ref, 4, 12, 1, (P, P, F), dy=2.0)
    c0 = rng.integers(-50, 50, size=(1, 12, 4)).astype(np.float64)
    st = {"u": g.zeros(), "v": g.zeros(), "w": None, "c": [g.zeros()]}
    setint(g, st["v"], -4.0); setint(g, st["c"][0], c0)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    ref.substage(g, prm, 1.0, 0.0, 0.5, st, G, None)
    assert np.array_equal(g.interior(st["c"][0]), np.roll(c0, -1, axis=1))


def test_top_hat_advection_listing16(ref):
    """Listing 16 / fig. B3 set-up with WENO5 + RK3: mass conserved, essentially non-oscillatory."""
    N = 128
    g = mkgrid(ref, N, 1, 1, (P, F, F), dx=12.0 / N)
    x = -4 + (np.arange(N) + 0.5) * 12.0 / N
    c0 = (np.abs(x) <= 1).astype(np.float64)
    prm = ref.default_params(n_tracers=1, momentum_prognostic=0, adv_y=0, adv_z=0)
    out = {}
    for scheme in (5, 2):
        prm["adv_x"] = scheme
        st = {"u": g.zeros() + 1.0, "v": None, "w": None, "c": [g.zeros()]}
        setint(g, st["c"][0], c0[None, None, :])
        dt, Gp = 1.0 / N, None
        for step in range(2 * N):          # t = 2: the hat has moved 2 units
            for s in (1, 2, 3):
                ref.fill_halos(g, prm, st)
                G = ref.compute_tendencies(g, prm, st, eval=1)
                ref.rk3_substage(g, prm, s, dt, st, G, Gp, eval=1)
                Gp = G
        out[scheme] = g.interior(st["c"][0])[0, 0].copy()
    assert abs(out[5].sum() - c0.sum()) < 1e-11 and abs(out[2].sum() - c0.sum()) < 1e-11
    over5 = max(out[5].max() - 1, -out[5].min())
    over2 = max(out[2].max() - 1, -out[2].min())
    assert over5 < 0.01 and over2 > 0.1               # Centered(2) oscillates, WENO does not (fig. B3)
    centre = (out[5] * x).sum() / out[5].sum()
    assert abs(centre - 2.0) < 0.02


def test_smooth_convergence(ref):
    """cell averages of u = 2 + sin x: the x-advection tendency converges at high order (SURVEY c.8)."""
    errs = []
    for N in (16, 32, 64):
        L = 2 * np.pi
        dx = L / N
        g = mkgrid(ref, N, 1, 1, (P, F, F), dx=dx)
        xf = np.arange(N) * dx                               # u lives on faces: control volume [xf-dx/2, xf+dx/2]
        ubar = 2 + (np.cos(xf - dx / 2) - np.cos(xf + dx / 2)) / dx
        st = {"u": g.zeros(), "v": None, "w": None, "c": []}
        setint(g, st["u"], ubar[None, None, :])
        prm = ref.default_params(adv_y=0, adv_z=0)
        ref.fill_halos(g, prm, st)
        G = ref.compute_tendencies(g, prm, st)
        # exact cell-averaged -d(u^2)/dx over the control volume
        F_ = lambda x: (2 + np.sin(x)) ** 2
        exact = -(F_(xf + dx / 2) - F_(xf - dx / 2)) / dx
        errs.append(np.abs(g.interior(G["u"])[0, 0] - exact).max())
    assert errs[0] / errs[1] > 8 and errs[1] / errs[2] > 8 and errs[2] < 5e-5


# ----------------------------------------------------------------------------- brute force, 8^3 periodic
def _weno_np(a, b, c, d, e, eps=1e-8):
    p1 = (2 * a - 7 * b + 11 * c) / 6; p0 = (-b + 5 * c + 2 * d) / 6; pm = (2 * c + 5 * d - e) / 6
    b1 = 13 / 12 * (a - 2 * b + c) ** 2 + 0.25 * (a - 4 * b + 3 * c) ** 2
    b0 = 13 / 12 * (b - 2 * c + d) ** 2 + 0.25 * (b - d) ** 2
    bm = 13 / 12 * (c - 2 * d + e) ** 2 + 0.25 * (3 * c - 4 * d + e) ** 2
    t = np.abs(b1 - bm)
    a1 = 0.1 * (1 + (t / (b1 + eps)) ** 2); a0 = 0.6 * (1 + (t / (b0 + eps)) ** 2); am = 0.3 * (1 + (t / (bm + eps)) ** 2)
    return (a1 * p1 + a0 * p0 + am * pm) / (a1 + a0 + am)


def _brute(q, adv, ax_q, ax_flux, target_shift):
    """Upwinded flux adv * recon(q) with np.roll (no halos).  The reconstruction point lies between q[m-1] and q[m]
    along array axis `ax_flux`; `target_shift`=0 means m = own index (centre->face), 1 means m = own+1 (face->centre)."""
    s = lambda off: np.roll(q, -(off + target_shift), axis=ax_flux)     # s(off) = q[m + off]
    left = _weno_np(s(-3), s(-2), s(-1), s(0), s(1))
    right = _weno_np(s(2), s(1), s(0), s(-1), s(-2))
    return adv * np.where(adv > 0, left, right)


def _c4(q, axis, target_shift):
    s = lambda off: np.roll(q, -(off + target_shift), axis=axis)
    return (-s(-2) + 7 * s(-1) + 7 * s(0) - s(1)) / 12


def test_brute_force_8cubed(ref):
    """north_star: brute-force comparison on an 8^3 periodic grid — modular indexing, no halo arrays."""
    rng = np.random.default_rng(14)
    n = 8
    g = mkgrid(ref, n, n, n, (P, P, P))
    st = rand_state(ref, g, rng, n_tracers=1, scale=0.5)
    prm = ref.default_params(n_tracers=1, nu=0.05, kappa=[0.07] + [0] * 7, f0=0.3)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    u, v, w = (g.interior(st[k]).copy() for k in "uvw")
    c = g.interior(st["c"][0]).copy()
    AX = {"x": 2, "y": 1, "z": 0}
    dn = lambda a, ax: a - np.roll(a, 1, axis=ax)          # value[m] - value[m-1]
    up = lambda a, ax: np.roll(a, -1, axis=ax) - a         # value[m+1] - value[m]
    lap = lambda a: sum(np.roll(a, 1, axis=ax) - 2 * a + np.roll(a, -1, axis=ax) for ax in (0, 1, 2))
    # tracer: fluxes at the low faces, divergence = F[i+1]-F[i]
    Gc = -(up(_brute(c, u, 2, 2, 0), 2) + up(_brute(c, v, 1, 1, 0), 1) + up(_brute(c, w, 0, 0, 0), 0)) + 0.07 * lap(c)
    assert np.allclose(g.interior(G["c"][0]), Gc, rtol=0, atol=2e-13)
    # u: Fxu at centres (shift 1), Fyu at ffc with v interpolated in x, Fzu at fcf with w interpolated in x
    Fxu = _brute(u, _c4(u, 2, 1), 2, 2, 1)
    Fyu = _brute(u, _c4(v, 2, 0), 1, 1, 0)
    Fzu = _brute(u, _c4(w, 2, 0), 0, 0, 0)
    vbar = 0.25 * (np.roll(v, 1, axis=2) + v + np.roll(np.roll(v, 1, axis=2), -1, axis=1) + np.roll(v, -1, axis=1))
    Gu = -(dn(Fxu, 2) + up(Fyu, 1) + up(Fzu, 0)) + 0.3 * vbar + 0.05 * lap(u)
    assert np.allclose(g.interior(G["u"]), Gu, rtol=0, atol=2e-13)
    Fxv = _brute(v, _c4(u, 1, 0), 2, 2, 0)
    Fyv = _brute(v, _c4(v, 1, 1), 1, 1, 1)
    Fzv = _brute(v, _c4(w, 1, 0), 0, 0, 0)
    ubar = 0.25 * (np.roll(u, 1, axis=1) + np.roll(np.roll(u, 1, axis=1), -1, axis=2) + u + np.roll(u, -1, axis=2))
    Gv = -(up(Fxv, 2) + dn(Fyv, 1) + up(Fzv, 0)) - 0.3 * ubar + 0.05 * lap(v)
    assert np.allclose(g.interior(G["v"]), Gv, rtol=0, atol=2e-13)
    Fxw = _brute(w, _c4(u, 0, 0), 2, 2, 0)
    Fyw = _brute(w, _c4(v, 0, 0), 1, 1, 0)
    Fzw = _brute(w, _c4(w, 0, 1), 0, 0, 1)
    Gw = -(up(Fxw, 2) + up(Fyw, 1) + dn(Fzw, 0)) + 0.05 * lap(w)
    assert np.allclose(g.interior(G["w"]), Gw, rtol=0, atol=2e-13)


def test_tendencies_at_matches_full(ref):
    rng = np.random.default_rng(15)
    g = mkgrid(ref, 9, 7, 6, (P, P, B))
    st = rand_state(ref, g, rng, n_tracers=2, scale=0.1)
    prm = ref.default_params(n_tracers=2, idx_T=0, idx_S=1, nu=0.01, kappa=[0.02, 0.03] + [0] * 6, f0=0.1, g=9.81, alpha_T=2e-4, beta_S=8e-4)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    ijk = np.array([[1, 1, 1], [9, 7, 6], [4, 3, 2], [2, 7, 1]], dtype=np.int32)
    out = ref.tendencies_at(g, prm, st, None, ijk)
    for s, (i, j, k) in enumerate(ijk):
        exp = [g.at(G["u"], i, j, k), g.at(G["v"], i, j, k), g.at(G["w"], i, j, k), g.at(G["c"][0], i, j, k), g.at(G["c"][1], i, j, k)]
        assert np.array_equal(out[s], np.array(exp))


def test_double_instantiation_close_to_long_double(ref):
    """the timed baseline (double) is the same algorithm: it agrees with the long-double reference to rounding."""
    rng = np.random.default_rng(16)
    g = mkgrid(ref, 10, 9, 8, (P, P, B))
    st = rand_state(ref, g, rng, n_tracers=1, scale=0.1)
    prm = ref.default_params(n_tracers=1, nu=0.01, kappa=[0.02] + [0] * 7, f0=0.1)
    ref.fill_halos(g, prm, st)
    G0 = ref.compute_tendencies(g, prm, st, eval=0)
    G1 = ref.compute_tendencies(g, prm, st, eval=1)
    for k in "uvw":
        assert np.abs(G0[k] - G1[k]).max() < 1e-13 * np.abs(G0[k]).max()
    st32 = {k: (None if st[k] is None else st[k].astype(np.float32)) for k in "uvw"}
    st32["c"] = [st["c"][0].astype(np.float32)]
    G2 = ref.compute_tendencies(g, prm, st32)
    assert G2["u"].dtype == np.float32 and np.abs(G2["u"] - G0["u"]).max() < 2e-4 * np.abs(G0["u"]).max()


# ----------------------------------------------------------------------------- hydrostatic pressure gradient in G_u, G_v
def _hydro_only_params(ref, **kw):
    """hydrostatic model with every other term off: G_u = -d_x p_hy / dx, G_v = -d_y p_hy / dy (eq. 17, (A6) 817-822)."""
    return ref.default_params(hydrostatic=1, adv_x=0, adv_y=0, adv_z=0, **kw)


def test_hydrostatic_pressure_gradient_linear_closed_form(ref):
    """p_hy = a x_c + b y_c + c z_c handed to compute_tendencies with all other terms off: G_u = -a, G_v = -b exactly
    where the linear continuation is in the halos; wall faces of v give 0; with the periodic x-halo the wrap face sees
    the jump -(p[1] - p[Nx])/dx = +a (Nx - 1).  Fails for a wrong sign, a forward instead of backward difference
    (wall rows / wrap column), x <-> y transposition (a != b, dx != dy) or a dropped 1/dx."""
    dzc = np.array([4.0, 3.0, 2.0, 1.5])
    g = mkgrid(ref, 7, 6, 4, (P, B, B), dx=2.0, dy=3.0, dz_c=dzc)
    a, b, c = 0.75, -1.25, 0.5
    H = 3
    i = np.arange(1 - H, 7 + H + 1); j = np.arange(1 - H, 6 + H + 1)
    xc = (i - 0.5) * 2.0; yc = (j - 0.5) * 3.0
    zc = np.concatenate([np.zeros(H), g.metric("zc"), np.zeros(H)])
    p = a * xc[None, None, :] + b * yc[None, :, None] + c * zc[:, None, None] + np.zeros(g.shape)
    st = {"u": g.zeros(), "v": g.zeros(), "w": None, "c": []}
    prm = _hydro_only_params(ref)
    G = ref.compute_tendencies(g, prm, st, p_hy=p)
    assert np.allclose(g.interior(G["u"]), -a, rtol=0, atol=1e-15)
    Gv = g.interior(G["v"])
    assert np.all(Gv[:, 0, :] == 0.0)                      # wall face j = 1: no tendency
    assert np.allclose(Gv[:, 1:, :], -b, rtol=0, atol=1e-15)
    assert G["w"] is None
    # periodic wrap in x: halo i = 0 holds p[Nx]
    pw = p.copy()
    pw[:, :, :H] = p[:, :, 7:7 + H]; pw[:, :, H + 7:] = p[:, :, H:2 * H]
    Gw = ref.compute_tendencies(g, prm, st, p_hy=pw)
    gu = g.interior(Gw["u"])
    assert np.allclose(gu[:, :, 1:], -a, rtol=0, atol=1e-15)
    assert np.allclose(gu[:, :, 0], a * (7 - 1), rtol=0, atol=1e-14)


def test_hydrostatic_pressure_gradient_random_numpy(ref):
    """random p_hy on the padded array: G_u, G_v equal the backward differences by numpy slicing (index and sign)."""
    rng = np.random.default_rng(77)
    g = mkgrid(ref, 9, 5, 3, (P, B, B), dx=0.7, dy=1.9)
    p = rng.standard_normal(g.shape)
    st = {"u": g.zeros(), "v": g.zeros(), "w": None, "c": []}
    G = ref.compute_tendencies(g, _hydro_only_params(ref), st, p_hy=p)
    H = 3
    I = p[H:H + 3, H:H + 5, H:H + 9]
    want_u = -(I - p[H:H + 3, H:H + 5, H - 1:H + 8]) / 0.7
    want_v = -(I - p[H:H + 3, H - 1:H + 4, H:H + 9]) / 1.9
    want_v[:, 0, :] = 0.0
    assert np.allclose(g.interior(G["u"]), want_u, rtol=1e-15, atol=1e-15)
    assert np.allclose(g.interior(G["v"]), want_v, rtol=1e-15, atol=1e-15)
    # the term is additive: with Coriolis on, G changes by exactly the Coriolis closed form of a uniform flow
    setint(g, st["u"], 0.3); setint(g, st["v"], 0.0)
    prm = _hydro_only_params(ref, f0=1e-4)
    ref.fill_halos(g, prm, st)
    G2 = ref.compute_tendencies(g, prm, st, p_hy=p)
    assert np.allclose(g.interior(G2["v"])[:, 1:, :], want_v[:, 1:, :] - 1e-4 * 0.3, rtol=1e-13, atol=1e-15)
    # nonhydrostatic model ignores p_hy
    st3 = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": []}
    G3 = ref.compute_tendencies(g, ref.default_params(adv_x=0, adv_y=0, adv_z=0), st3, p_hy=p)
    assert np.all(g.interior(G3["u"]) == 0.0) and np.all(g.interior(G3["v"]) == 0.0)


def test_hydrostatic_buoyancy_end_to_end_closed_form(ref):
    """The only way buoyancy enters the hydrostatic model (R10): T = T_ref(z) + s x_c, S = S_ref(z) + r y_c gives
    b = g (alpha s x_c - beta r y_c), uniform in z, so (14) integrates to p_hy = b z_c and
    G_u = -g alpha s z_c[k] (> 0 at depth for warm water to the east), G_v = +g beta r z_c[k]  — compute_phy -> compute_tendencies."""
    dzc = np.array([250.0, 120.0, 60.0, 25.0, 10.0])
    g = mkgrid(ref, 8, 7, 5, (B, B, B), dx=5000.0, dy=4000.0, dz_c=dzc)
    grav, alpha, beta, s, r = 9.81, 2e-4, 8e-4, 3e-5, -2e-5
    zc = g.metric("zc")
    Tref, Sref = 20.0 + 0.004 * zc, 35.0 - 0.0002 * zc
    H = 3
    i = np.arange(1 - H, 8 + H + 1); j = np.arange(1 - H, 7 + H + 1)
    xc = (i - 0.5) * 5000.0; yc = (j - 0.5) * 4000.0
    T = g.zeros(); S = g.zeros()
    T[H:H + 5] = Tref[:, None, None] + s * xc[None, None, :] + 0.0 * yc[None, :, None]
    S[H:H + 5] = Sref[:, None, None] + r * yc[None, :, None] + 0.0 * xc[None, None, :]
    st = {"u": g.zeros(), "v": g.zeros(), "w": None, "c": [T, S]}
    prm = _hydro_only_params(ref, n_tracers=2, idx_T=0, idx_S=1, g=grav, alpha_T=alpha, beta_S=beta, T_ref=Tref, S_ref=Sref)
    p = ref.compute_phy(g, prm, st)
    G = ref.compute_tendencies(g, prm, st, p_hy=p)
    gu, gv = g.interior(G["u"]), g.interior(G["v"])
    want_u = -grav * alpha * s * zc
    want_v = grav * beta * r * zc
    assert np.all(gu[:, :, 0] == 0.0) and np.all(gv[:, 0, :] == 0.0)                     # wall faces
    assert np.allclose(gu[:, :, 1:], want_u[:, None, None] * np.ones((5, 7, 7)), rtol=1e-10)
    assert np.allclose(gv[:, 1:, :], want_v[:, None, None] * np.ones((5, 6, 8)), rtol=1e-10)
    assert want_u[0] > 0 and want_v[0] > 0                                               # the signs the physics fixes
    # tracer tendencies see no pressure: constant-in-(their own advecting direction) fields with zero velocity stay put
    assert np.abs(g.interior(G["c"][0])).max() == 0.0
