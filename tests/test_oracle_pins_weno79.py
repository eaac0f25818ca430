"""Pins of the oracle's WENO7 / WENO9 against what the paper and the mathematics fix.

The paper prints only the r = 3 candidates (B9); the r = 4, 5 tables come from the same DEFINITION (candidate polynomials
matching cell averages, Jiang-Shu smoothness integrals, ideal weights reproducing the (2r-1)-cell linear scheme), generated in
exact rational arithmetic by oracle/gen_weno_tables.py.  None of these tests touches the CUDA path.
"""
import importlib.util
import os
from fractions import Fraction as Fr

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
P, B, F = 0, 1, 2


def _gen():
    spec = importlib.util.spec_from_file_location("_gen_weno_tables", os.path.join(ROOT, "oracle", "gen_weno_tables.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def _cell_averages(poly, edges):
    P_ = np.polynomial.Polynomial(poly).integ()
    return (P_(edges[1:]) - P_(edges[:-1])) / np.diff(edges)


def mkgrid(ref, Nx, Ny, Nz, topo, H, dx=1.0, dy=1.0, dz=1.0):
    return ref.RefGrid(Nx, Ny, Nz, H, dx, dy, dz_c=None, dz_uniform=dz, topology=topo)


# ----------------------------------------------------------------------------- the generator against the paper
def test_generator_reproduces_paper_B9_and_classical_indicators():
    """r = 3: candidates = (B9) PAPER.md:1037-1040; indicators = 13/12 (a-2b+c)^2 + 1/4 (...)^2 (reading R1) expanded;
    ideal weights (1/10, 6/10, 3/10); linear scheme (2,-13,47,27,-3)/60."""
    G = _gen()
    t = G.tables(3)
    assert t["cand"] == [[Fr(2, 6), Fr(-7, 6), Fr(11, 6)], [Fr(-1, 6), Fr(5, 6), Fr(2, 6)], [Fr(2, 6), Fr(5, 6), Fr(-1, 6)]]
    assert t["d"] == [Fr(1, 10), Fr(6, 10), Fr(3, 10)]
    assert t["lin"] == [Fr(x, 60) for x in (2, -13, 47, 27, -3)]

    def quad(lin1, lin2):     # 13/12 lin1^2 + 1/4 lin2^2 as a symmetric matrix
        return [[Fr(13, 12) * lin1[a] * lin1[b] + Fr(1, 4) * lin2[a] * lin2[b] for b in range(3)] for a in range(3)]
    assert G.beta_matrix(t, 0) == quad((1, -2, 1), (1, -4, 3))
    assert G.beta_matrix(t, 1) == quad((1, -2, 1), (1, 0, -1))
    assert G.beta_matrix(t, 2) == quad((1, -2, 1), (3, -4, 1))


def test_generator_tables_r4_r5_structure():
    """r = 4, 5: weights positive, sum 1, mirror-symmetric pairs of candidates, indicators positive semi-definite and
    blind to constants, tau combination annihilates the common leading term (all beta_k = slope^2 on linear data)."""
    G = _gen()
    for r in (4, 5):
        t = G.tables(r)
        assert sum(t["d"]) == 1 and all(x > 0 for x in t["d"])
        for k in range(r):
            assert sum(t["cand"][k]) == 1                                  # reproduces constants
            Bk = G.beta_matrix(t, k)
            for a in range(r):
                assert sum(Bk[a]) == 0                                     # translation invariant
                assert Bk[a] == [Bk[b][a] for b in range(r)]               # symmetric
            lin = [Fr(j) for j in range(r)]
            assert sum(Bk[a][b] * lin[a] * lin[b] for a in range(r) for b in range(r)) == 1    # slope^2
            M = np.array([[float(x) for x in row] for row in Bk])
            assert np.linalg.eigvalsh(M).min() > -1e-9
        assert sum(t["tau"]) == 0
        # the full linear scheme is exact for degree <= 2r-2: check the monomial x^(2r-2) cell averages -> (1/2)^(2r-2)
        n = 2 * r - 2
        avg = [G.cell_average_of_monomial(n, j) for j in range(-(r - 1), r)]
        assert sum(w * a for w, a in zip(t["lin"], avg)) == Fr(1, 2) ** n


def test_committed_table_file_is_the_generators_output():
    G = _gen()
    with open(os.path.join(ROOT, "oracle", "weno_tables.inc")) as f:
        assert f.read() == G.emit()


def test_centered_weights():
    """Centered(4) = (-1,7,7,-1)/12 (symmetric part of (B5)); Centered(6), (8) the same construction."""
    G = _gen()
    assert G.centered_weights(2) == [Fr(1, 2), Fr(1, 2)]                                  # (B4) PAPER.md:1007
    assert G.centered_weights(4) == [Fr(-1, 12), Fr(7, 12), Fr(7, 12), Fr(-1, 12)]
    assert G.centered_weights(6) == [Fr(x, 60) for x in (1, -8, 37, 37, -8, 1)]
    assert G.centered_weights(8) == [Fr(x, 840) for x in (-3, 29, -139, 533, 533, -139, 29, -3)]


# ----------------------------------------------------------------------------- the C++ routine against the tables
def _weno_exact(G, r, v, eps):
    """WENO(2r-1)-Z in exact rationals, VALUE form (beta = v^T B v, candidates = rows of `cand`): a different
    evaluation route from the oracle's (monomial coefficients of shifted data)."""
    t = G.tables(r)
    v = [Fr(x) for x in v]
    p, beta = [], []
    for k in range(r):
        vs = v[k:k + r]
        p.append(sum(c * x for c, x in zip(t["cand"][k], vs)))
        Bk = G.beta_matrix(t, k)
        beta.append(sum(Bk[a][b] * vs[a] * vs[b] for a in range(r) for b in range(r)))
    tau = abs(sum(c * b for c, b in zip(t["tau"], beta)))
    al = [t["d"][k] * (1 + (tau / (beta[k] + Fr(eps))) ** 2) for k in range(r)]
    return float(sum(a * x for a, x in zip(al, p)) / sum(al))


@pytest.mark.parametrize("r", [3, 4, 5])
def test_general_routine_equals_exact_rational_evaluation(ref, r):
    G = _gen()
    rng = np.random.default_rng(40 + r)
    kind = {3: 55, 4: 7, 5: 9}[r]
    for trial in range(12):
        scale = 10.0 ** rng.integers(-3, 2)
        mean = (0.0, 35.0, -20.0)[trial % 3]
        q = mean + scale * rng.standard_normal(2 * r + 3)
        m = r + 1
        left = q[m - r:m + r - 1]
        right = q[m - r + 1:m + r][::-1]
        eL, eR = _weno_exact(G, r, left, 1e-8), _weno_exact(G, r, right, 1e-8)
        tol = 2e-15 * max(abs(mean), scale) + 1e-13 * scale
        assert abs(ref.reconstruct(q, m, kind) - eL) < tol, (trial, ref.reconstruct(q, m, kind), eL)
        assert abs(ref.reconstruct(q, m, -kind) - eR) < tol


def test_general_routine_r3_equals_weno5z(ref):
    rng = np.random.default_rng(44)
    for _ in range(50):
        q = rng.standard_normal(9) * 10.0 ** rng.integers(-4, 3)
        assert ref.reconstruct(q, 4, 55) == pytest.approx(ref.reconstruct(q, 4, 5), rel=0, abs=2e-15 * np.abs(q).max())
        assert ref.reconstruct(q, 4, -55) == pytest.approx(ref.reconstruct(q, 4, -5), rel=0, abs=2e-15 * np.abs(q).max())
        assert ref.reconstruct(q, 4, 44) == pytest.approx(ref.reconstruct(q, 4, 4), rel=0, abs=2e-15 * np.abs(q).max())


@pytest.mark.parametrize("r,kind", [(4, 7), (5, 9)])
def test_candidates_exact_for_degree_r_minus_1(ref, r, kind):
    """each candidate — hence the convex combination for ANY weights — returns the interface point value exactly from
    cell averages of a polynomial of degree <= r-1 (PAPER.md:1039 for r = 3)."""
    rng = np.random.default_rng(50 + r)
    for _ in range(10):
        poly = rng.standard_normal(r)
        h = rng.uniform(0.3, 1.5)
        n = 2 * r + 2
        m = r + 1                                     # interface between q[m-1] and q[m], placed at x = 0
        edges = h * (np.arange(n + 1) - m)
        qa = _cell_averages(poly, edges)
        exact = poly[0]
        assert abs(ref.reconstruct(qa, m, kind) - exact) < 1e-12 * (1 + np.abs(qa).max())
        assert abs(ref.reconstruct(qa, m, -kind) - exact) < 1e-12 * (1 + np.abs(qa).max())


@pytest.mark.parametrize("r,kind", [(4, 7), (5, 9)])
def test_linear_limit_is_order_2r_minus_1(ref, r, kind):
    """huge eps => ideal weights => the (2r-1)-cell linear scheme, exact for degree <= 2r-2."""
    rng = np.random.default_rng(60 + r)
    poly = rng.standard_normal(2 * r - 1)
    n = 2 * r + 2
    m = r + 1
    edges = 0.5 * (np.arange(n + 1) - m)
    qa = _cell_averages(poly, edges)
    assert abs(ref.reconstruct(qa, m, kind, eps=1e40) - poly[0]) < 1e-11 * (1 + np.abs(qa).max())
    assert abs(ref.reconstruct(qa, m, -kind, eps=1e40) - poly[0]) < 1e-11 * (1 + np.abs(qa).max())
    # linear data: all indicators equal => tau = 0 => exact with the small eps as well
    lin = 0.3 + 0.7 * np.arange(n)
    assert abs(ref.reconstruct(lin, m, kind) - (0.3 + 0.7 * (m - 0.5))) < 1e-13


@pytest.mark.parametrize("kind", [7, 9])
def test_weno79_properties(ref, kind):
    rng = np.random.default_rng(70 + kind)
    q = rng.standard_normal(14)
    m = 7
    qr = q[::-1].copy()
    assert ref.reconstruct(q, m, -kind) == pytest.approx(ref.reconstruct(qr, len(q) - m, kind), abs=1e-15)      # mirror (R3)
    assert ref.reconstruct(q + 7.5, m, kind) == pytest.approx(ref.reconstruct(q, m, kind) + 7.5, abs=1e-13)    # translation
    assert ref.reconstruct(3.0 * q, m, kind, eps=0.0) == pytest.approx(3.0 * ref.reconstruct(q, m, kind, eps=0.0), abs=1e-13)
    # essentially non-oscillatory at a step: upwind side flat => the value of the flat side
    step = np.array([0.0] * 7 + [1.0] * 7)
    assert -1e-10 <= ref.reconstruct(step, 7, kind) < 1e-5
    assert 1 - 1e-5 < ref.reconstruct(step, 7, -kind) <= 1 + 1e-10


@pytest.mark.parametrize("kind,order", [(7, 7), (9, 9), (6, 6), (8, 8)])
def test_smooth_convergence_order(ref, kind, order):
    """cell averages of sin: the interface error falls as h^order (WENO-Z keeps the design order away from critical points)."""
    errs = []
    for n in (8, 16):
        h = 1.0 / n
        x0 = 0.3
        m = 6
        edges = x0 + h * (np.arange(13) - m)
        qa = (np.cos(edges[:-1]) - np.cos(edges[1:])) / h
        errs.append(abs(ref.reconstruct(qa, m, kind) - np.sin(x0)))
    rate = np.log2(errs[0] / errs[1])
    assert rate > order - 0.6, (errs, rate)


# ----------------------------------------------------------------------------- tendencies with WENO7 / WENO9
def _rand_state(g, rng, n_tracers=1):
    st = {"u": g.zeros(), "v": g.zeros(), "w": g.zeros(), "c": [g.zeros() for _ in range(n_tracers)]}
    for k in ("u", "v", "w"):
        g.interior(st[k])[...] = rng.standard_normal((g.Nz, g.Ny, g.Nx))
    for c in st["c"]:
        g.interior(c)[...] = rng.standard_normal((g.Nz, g.Ny, g.Nx))
    return st


@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("topo", [(P, P, P), (P, P, B)])
def test_conservation_and_constants_weno79(ref, order, topo):
    rng = np.random.default_rng(80 + order)
    H = (order + 1) // 2
    g = mkgrid(ref, 10, 9, 8, topo, H, dx=0.8, dy=1.3)
    st = _rand_state(g, rng)
    prm = ref.default_params(n_tracers=1, nu=0.2, kappa=[0.3] + [0] * 7, adv_x=order, adv_y=order, adv_z=order)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    Gc = g.interior(G["c"][0])
    assert abs(Gc.sum()) < 1e-13 * np.abs(Gc).sum()                         # sum V G = 0 (B2), uniform volumes
    Gu = g.interior(G["u"])
    assert abs(Gu.sum()) < 1e-13 * np.abs(Gu).sum()
    # uniform flow, constant tracer => zero advective tendencies
    st2 = {"u": g.zeros() + 0.3, "v": g.zeros() - 0.2, "w": g.zeros() + (0.1 if topo[2] == P else 0.0), "c": [g.zeros() + 3.7]}
    prm2 = ref.default_params(n_tracers=1, adv_x=order, adv_y=order, adv_z=order)
    ref.fill_halos(g, prm2, st2)
    G2 = ref.compute_tendencies(g, prm2, st2)
    assert np.abs(g.interior(G2["c"][0])).max() < 1e-13
    if topo[2] == P:
        for k in "uvw":
            assert np.abs(g.interior(G2[k])).max() < 1e-15


@pytest.mark.parametrize("order", [7, 9])
def test_axis_swap_symmetry_weno79(ref, order):
    rng = np.random.default_rng(90 + order)
    n = 10
    g = mkgrid(ref, n, n, n, (P, P, P), (order + 1) // 2)
    st = _rand_state(g, rng)
    prm = ref.default_params(n_tracers=1, nu=0.1, kappa=[0.2] + [0] * 7, adv_x=order, adv_y=order, adv_z=order)
    ref.fill_halos(g, prm, st)
    G = ref.compute_tendencies(g, prm, st)
    for perm, names in (((0, 2, 1), ("v", "u", "w")), ((2, 1, 0), ("w", "v", "u"))):
        st2 = {"u": np.ascontiguousarray(st[names[0]].transpose(perm)), "v": np.ascontiguousarray(st[names[1]].transpose(perm)),
               "w": np.ascontiguousarray(st[names[2]].transpose(perm)), "c": [np.ascontiguousarray(st["c"][0].transpose(perm))]}
        G2 = ref.compute_tendencies(g, prm, st2)
        for a, b in zip(("u", "v", "w"), names):
            assert np.allclose(g.interior(G2[a]), g.interior(G[b].transpose(perm)), rtol=0, atol=1e-13)
        assert np.allclose(g.interior(G2["c"][0]), g.interior(G["c"][0].transpose(perm)), rtol=0, atol=1e-13)


@pytest.mark.parametrize("order", [7, 9])
def test_tracer_flux_brute_force_1d(ref, order):
    """1-D periodic tracer advection tendency written with modular indexing, no halo arrays, and the exact-rational
    WENO evaluation above: G_c[i] = -(u[i+1] F[i+1] - u[i] F[i]) / dx must agree with the oracle's 3-D machinery."""
    G_ = _gen()
    r = (order + 1) // 2
    rng = np.random.default_rng(100 + order)
    n = 12
    g = mkgrid(ref, n, 1, 1, (P, F, F), r, dx=0.7)
    c = rng.standard_normal(n)
    u = rng.standard_normal(n)
    st = {"u": g.zeros(), "v": None, "w": None, "c": [g.zeros()]}
    g.interior(st["u"])[0, 0, :] = u
    g.interior(st["c"][0])[0, 0, :] = c
    prm = ref.default_params(n_tracers=1, momentum_prognostic=0, adv_x=order, adv_y=0, adv_z=0)
    ref.fill_halos(g, prm, st)
    Gc = g.interior(ref.compute_tendencies(g, prm, st)["c"][0])[0, 0, :]
    Fx = np.zeros(n)
    for i in range(n):            # face i (0-based) lies between cells i-1 and i
        if u[i] > 0:
            v = [c[(i - r + t) % n] for t in range(2 * r - 1)]
        else:
            v = [c[(i + r - 1 - t) % n] for t in range(2 * r - 1)]
        Fx[i] = u[i] * _weno_exact(G_, r, v, 1e-8)
    expect = -(np.roll(Fx, -1) - Fx) / 0.7
    assert np.abs(Gc - expect).max() < 1e-13 * np.abs(expect).max()


# ----------------------------------------------------------------------------- tau_7, tau_9 of WENO-Z (reading R20)
def _tau_of_h(G, t, coeffs, poly, h):
    """|sum_k coeffs[k] beta_k| in exact rationals on the cell averages of `poly` (ascending Fractions) on cells of width h
    centred at j h, j = -(r-1) .. r-1."""
    r = t["r"]

    def avg(j):
        lo, hi = (Fr(2 * j - 1, 2)) * h, (Fr(2 * j + 1, 2)) * h
        return sum(c * (hi ** (n + 1) - lo ** (n + 1)) / (n + 1) for n, c in enumerate(poly)) / h
    v = {j: avg(j) for j in range(-(r - 1), r)}
    tot = Fr(0)
    for k in range(r):
        Bk = G.beta_matrix(t, k)
        cells = list(range(k - (r - 1), k + 1))
        tot += coeffs[k] * sum(Bk[a][b] * v[cells[a]] * v[cells[b]] for a in range(r) for b in range(r))
    return abs(tot)


def _observed_order(G, t, coeffs, poly):
    import math
    a, b = _tau_of_h(G, t, coeffs, poly, Fr(1, 64)), _tau_of_h(G, t, coeffs, poly, Fr(1, 128))
    return math.log2(float(a / b))


@pytest.mark.parametrize("r,want,order,simple,simple_order", [(3, (1, 0, -1), 5, None, None),
                                                              (4, (1, 3, -3, -1), 7, (1, -1, -1, 1), 6),
                                                              (5, (1, 2, -6, 2, 1), 8, (1, 0, 0, 0, -1), 7)])
def test_tau_combination_cancels_to_the_highest_order(r, want, order, simple, simple_order):
    """DESIGN.md R20: tau_{2r-1} = |sum_k t_k beta_k| with the t that cancel the Taylor expansion to the highest order.
    (a) the table the oracle compiles (weno_tables.inc) holds (1,0,-1), (1,3,-3,-1), (1,2,-6,2,1);
    (b) measured in exact rationals on a generic degree-12 polynomial, tau shrinks like h^5, h^7, h^8 — and the simpler
        combinations (1,-1,-1,1), (1,0,0,0,-1) only like h^6, h^7, so typing those instead would fail here;
    (c) no other integer combination with |t_k| <= 6 reaches that order (uniqueness up to scale)."""
    import itertools
    import re
    G = _gen()
    t = G.tables(r)
    with open(os.path.join(ROOT, "oracle", "weno_tables.inc")) as f:
        line = next(l for l in f if l.startswith("static const long double WENO%d_TAU" % (2 * r - 1)))
    in_file = tuple(int(n) // int(d) for n, d in re.findall(r"Q\((-?\d+), (\d+)\)", line))
    assert in_file == want and tuple(int(x) for x in t["tau"]) == want
    rng = np.random.default_rng(100 + r)
    poly = [Fr(int(x), 7) for x in rng.integers(-9, 10, size=13)]
    poly[1] = Fr(5, 7); poly[2] = Fr(-3, 7); poly[3] = Fr(4, 7)          # generic: no low derivative vanishes at 0
    assert abs(_observed_order(G, t, want, poly) - order) < 0.15
    if simple is not None:
        assert abs(_observed_order(G, t, simple, poly) - simple_order) < 0.15 and simple_order < order
    if r <= 4:   # brute force over all small integer combinations: only multiples of `want` reach that order
        from math import gcd, log2
        unit = [tuple(int(a == k) for a in range(r)) for k in range(r)]
        # sum_k c_k beta_k is linear in c: evaluate the (signed) beta_k once per h
        def betas(h):
            out = []
            for k in range(r):
                Bk = G.beta_matrix(t, k)
                cells = list(range(k - (r - 1), k + 1))
                v = [sum(cf * (((Fr(2 * jj + 1, 2)) * h) ** (n + 1) - ((Fr(2 * jj - 1, 2)) * h) ** (n + 1)) / (n + 1)
                         for n, cf in enumerate(poly)) / h for jj in cells]
                out.append(sum(Bk[a][b] * v[a] * v[b] for a in range(r) for b in range(r)))
            return out
        b32, b64 = betas(Fr(1, 2 ** 14)), betas(Fr(1, 2 ** 15))
        assert abs(sum(u * b for u, b in zip(unit[0], b32))) == _tau_of_h(G, t, unit[0], poly, Fr(1, 2 ** 14))
        winners = []
        for c in itertools.product(range(-6, 7), repeat=r):
            if c[0] <= 0 or sum(c) != 0 or gcd(*c) != 1:
                continue
            t32, t64 = abs(sum(x * b for x, b in zip(c, b32))), abs(sum(x * b for x, b in zip(c, b64)))
            if t64 == 0 or log2(float(t32 / t64)) > order - 0.5:      # measured between h = 2^-14 and 2^-15
                winners.append(c)
        assert winners == [want]
    # the generator's own derivation (exact null space of the Taylor conditions) is one-dimensional and equals `want`
    assert G.derive_tau(r, [G.beta_matrix(t, k) for k in range(r)]) == list(want)
