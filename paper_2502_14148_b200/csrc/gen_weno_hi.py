"""gen_weno_hi.py — writes csrc/weno_hi.cuh: straight-line device code of WENO7-Z / WENO9-Z in DIFFERENCE form.

    python paper_2502_14148_b200/csrc/gen_weno_hi.py

Part of the product's build sources (the generated header is committed; nvcc never runs this).  It shares nothing with
oracle/: the derivation below goes through the PRIMITIVE function (Lagrange interpolation of the running sums of the cell
averages, then differentiation) and a change of basis to undivided differences, all in exact rationals.

What the emitted functions compute (PAPER.md:1030-1042 (B8)/(B9) generalised to r = 4, 5; R1, R2,
R20): for the 2r-1 cell values v[0..2r-2], v[r-1] the upwind cell of the face,
    p_k(face)      candidate k = 0..r-1 from the cells v[k..k+r-1]
    beta_k         = sum_{l=1}^{r-1} int_cell (d^l p_k / dx^l)^2 dx   (Jiang-Shu), the integral over the upwind cell
    tau            = |sum_k T_k beta_k|,  T = (1,3,-3,-1), (1,2,-6,2,1)
    alpha_k        = d_k (1 + (tau / (beta_k + eps))^2),  d = ideal weights
    result         = sum_k alpha_k (p_k - v[r-1]) / sum_k alpha_k        (the reconstruction MINUS the upwind cell value)
B200 notes: everything is expressed in the undivided differences D^l_j of the stencil (D^1_j = v[j+1]-v[j], D^l_j =
D^(l-1)_(j+1) - D^(l-1)_j), which (a) keeps a large field mean out of the arithmetic (H1), (b) makes beta_k a
quadratic form in r-1 variables (r(r-1)/2 coefficients instead of r(r+1)/2) that is well conditioned on smooth data, and
(c) shares the difference table between the r candidates.  fp64: product form with ONE reciprocal per reconstruction (see
emit_function); fp32: one reciprocal per candidate + one for the sum (fast_rcp).
INTEGER COEFFICIENTS: every rational coefficient is emitted multiplied by the least common denominator of its group (beta_k by
SB = 240 / 5040, the candidates by SX = 12 / 60, the ideal weights by 35 / 126, the centred weights by 60 / 840): the
scaled numbers are integers below 2^21, i.e. doubles whose low mantissa word is zero, which the FP64 / FP32 instructions take
as IMMEDIATE operands.  A non-integer literal costs two UMOV per use (ncu, WENO9 at C2: 1559 UMOV per cell-warp, 20 % of all
issued instructions).  The scaling is exact: tau and beta_k + eps carry the same factor SB (eps is multiplied by SB once),
the weights' common factor cancels between numerator and denominator, SX is folded into the final denominator.
"""
import os
from fractions import Fraction as F

HERE = os.path.dirname(os.path.abspath(__file__))
TAU = {4: [1, 3, -3, -1], 5: [1, 2, -6, 2, 1]}


# ---- tiny exact polynomial arithmetic (coefficient lists, lowest degree first)
def padd(a, b):
    n = max(len(a), len(b))
    return [(a[i] if i < len(a) else F(0)) + (b[i] if i < len(b) else F(0)) for i in range(n)]


def pmul(a, b):
    out = [F(0)] * (len(a) + len(b) - 1)
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            out[i + j] += x * y
    return out


def pscale(a, s):
    return [x * s for x in a]


def pder(a):
    return [a[i] * i for i in range(1, len(a))] or [F(0)]


def pint_def(a, lo, hi):
    return sum(c * (hi ** (i + 1) - lo ** (i + 1)) / (i + 1) for i, c in enumerate(a))


def peval(a, x):
    return sum(c * x ** i for i, c in enumerate(a))


def candidate_polys(r, k):
    """p_k as r polynomials, one per unit datum: cells j = k-(r-1) .. k, cell j = [j-1/2, j+1/2].  The primitive
    V(x_{j+1/2}) = sum_{i<=j} v_i is interpolated at the r+1 cell edges by Lagrange polynomials; p_k = dV/dx."""
    cells = list(range(k - (r - 1), k + 1))
    edges = [F(2 * c - 1, 2) for c in cells] + [F(2 * cells[-1] + 1, 2)]
    lag = []
    for a, xa in enumerate(edges):
        poly = [F(1)]
        for b, xb in enumerate(edges):
            if b != a:
                poly = pscale(pmul(poly, [-xb, F(1)]), 1 / (xa - xb))
        lag.append(poly)
    polys = []
    for jj in range(r):
        # datum jj contributes 1 to the primitive at every edge to its right: edges jj+1 .. r
        P = [F(0)]
        for a in range(jj + 1, r + 1):
            P = padd(P, lag[a])
        polys.append(pder(P))
    return polys


def value_tables(r):
    cand, beta = [], []
    for k in range(r):
        polys = candidate_polys(r, k)
        cand.append([peval(p, F(1, 2)) for p in polys])
        Bk = [[F(0)] * r for _ in range(r)]
        for a in range(r):
            for b in range(r):
                s, pa, pb = F(0), polys[a], polys[b]
                for l in range(1, r):
                    pa, pb = pder(pa), pder(pb)
                    s += pint_def(pmul(pa, pb), F(-1, 2), F(1, 2))
                Bk[a][b] = s
        beta.append(Bk)
    return cand, beta


def linear_weights(r, cand):
    """d_k: the combination of the candidates that is exact for the highest degree (2r-2): solve on monomial data."""
    cells = list(range(-(r - 1), r))
    rows, rhs = [], []
    for n in range(r, 2 * r - 1):       # degrees r .. 2r-2 fix r-1 equations; sum d = 1 is the r-th
        avg = [((F(2 * c + 1, 2)) ** (n + 1) - (F(2 * c - 1, 2)) ** (n + 1)) / (n + 1) for c in cells]
        rows.append([sum(cand[k][jj] * avg[k + jj] for jj in range(r)) for k in range(r)])
        rhs.append(F(1, 2) ** n)
    rows.append([F(1)] * r)
    rhs.append(F(1))
    return solve(rows, rhs)


def solve(A, b):
    n = len(A)
    M = [list(A[i]) + [b[i]] for i in range(n)]
    for c in range(n):
        p = next(i for i in range(c, n) if M[i][c] != 0)
        M[c], M[p] = M[p], M[c]
        M[c] = [x / M[c][c] for x in M[c]]
        for i in range(n):
            if i != c and M[i][c] != 0:
                f = M[i][c]
                M[i] = [x - f * y for x, y in zip(M[i], M[c])]
    return [M[i][n] for i in range(n)]


def inverse(A):
    n = len(A)
    cols = [solve(A, [F(int(i == j)) for i in range(n)]) for j in range(n)]
    return [[cols[j][i] for j in range(n)] for i in range(n)]


def difference_rows(r, k):
    """rows of the map (stencil values v[k..k+r-1]) -> (D^1_k, ..., D^(r-1)_k, v_c): leading differences of the stencil
    plus the upwind cell value (local index r-1-k)."""
    rows = []
    cur = [[F(int(a == b)) for b in range(r)] for a in range(r)]       # identity: D^0_j = v_j
    for l in range(1, r):
        cur = [[cur[j + 1][b] - cur[j][b] for b in range(r)] for j in range(len(cur) - 1)]
        rows.append(cur[0])
    rows.append([F(int(b == r - 1 - k)) for b in range(r)])
    return rows


def difference_tables(r):
    cand, beta = value_tables(r)
    d = linear_weights(r, cand)
    X, M = [], []
    for k in range(r):
        Tinv = inverse(difference_rows(r, k))                          # v = Tinv [y; v_c]
        cy = [sum(cand[k][a] * Tinv[a][col] for a in range(r)) for col in range(r)]
        assert cy[r - 1] == 1                                          # p_k = v_c + sum_l X_l y_l
        X.append(cy[:r - 1])
        Mk = [[sum(Tinv[a][i] * beta[k][a][b] * Tinv[b][j] for a in range(r) for b in range(r)) for j in range(r)] for i in range(r)]
        assert all(Mk[i][r - 1] == 0 and Mk[r - 1][i] == 0 for i in range(r))    # indicators do not see the mean
        M.append([row[:r - 1] for row in Mk[:r - 1]])
    return X, M, d


def lit(x):
    x = F(x)
    if x.denominator == 1:
        return "Real(%d.0)" % x.numerator
    return "Real(%d.0 / %d.0)" % (x.numerator, x.denominator)


def common_denominator(cs):
    from math import lcm
    out = 1
    for c in cs:
        out = lcm(out, F(c).denominator)
    return out


def is_immediate(n):
    """an integer-valued double whose low 32 mantissa bits are zero"""
    n = abs(int(n))
    while n and n % 2 == 0:
        n //= 2
    return n < 2 ** 21


def emit_function(r):
    X, M, d = difference_tables(r)
    n = 2 * r - 1
    SB = common_denominator([M[k][a][a] for k in range(r) for a in range(r - 1)] +
                            [2 * M[k][a][b] for k in range(r) for a in range(r - 1) for b in range(a + 1, r - 1)])
    SX = common_denominator([X[k][a] for k in range(r) for a in range(r - 1)])
    SD = common_denominator(d)
    L = []
    L.append("// WENO%d-Z minus the upwind cell value: v[0..%d], v[%d] = upwind cell of the face.  GENERATED (gen_weno_hi.py)." % (n, n - 1, r - 1))
    L.append("// xs_k = %d (p_k - v_c), bs_k = %d beta_k, as_k = %d alpha_k: integer coefficients = immediate operands." % (SX, SB, SD))
    L.append("template <class Real> __device__ __forceinline__ Real weno%dz_anom(const Real *v, Real eps) {" % n)
    for j in range(n - 1):
        L.append("  const Real d1_%d = v[%d] - v[%d];" % (j, j + 1, j))
    for l in range(2, r):
        for j in range(n - l):                 # D^l_j, j = 0 .. 2r-2-l (what stencil k does not use is dead code)
            L.append("  const Real d%d_%d = d%d_%d - d%d_%d;" % (l, j, l - 1, j + 1, l - 1, j))
    L.append("  const Real epss = eps * Real(%d.0);" % SB)

    def ilit(c):
        assert F(c).denominator == 1 and is_immediate(c), c
        return "Real(%d.0)" % int(c)
    for k in range(r):
        y = ["d%d_%d" % (l, k) for l in range(1, r)]
        terms = [(X[k][a] * SX, y[a]) for a in range(r - 1) if X[k][a] != 0]
        expr = "%s * %s" % (ilit(terms[-1][0]), terms[-1][1])
        for c, nm in reversed(terms[:-1]):
            expr = "fma(%s, %s, %s)" % (ilit(c), nm, expr)
        L.append("  const Real xs%d = %s;" % (k, expr))
        # bs_k = SB beta_k = sum_a y_a (SB M_aa y_a + 2 SB sum_{b>a} M_ab y_b)
        outer = None
        for a in reversed(range(r - 1)):
            inner = "%s * %s" % (ilit(M[k][a][a] * SB), y[a])
            for b in range(a + 1, r - 1):
                if M[k][a][b] != 0:
                    inner = "fma(%s, %s, %s)" % (ilit(2 * M[k][a][b] * SB), y[b], inner)
            outer = "%s * (%s)" % (y[a], inner) if outer is None else "fma(%s, %s, %s)" % (y[a], inner, outer)
        L.append("  const Real bs%d = %s;" % (k, outer))
    # tau: +-1 coefficients as plain adds
    terms = [(TAU[r][k], "bs%d" % k) for k in range(r) if TAU[r][k] != 0]
    expr = None
    for c, nm in terms:
        if expr is None:
            expr = nm if c == 1 else "%s * %s" % (ilit(c), nm)
        elif c == 1:
            expr = "(%s + %s)" % (expr, nm)
        elif c == -1:
            expr = "(%s - %s)" % (expr, nm)
        else:
            expr = "fma(%s, %s, %s)" % (ilit(c), nm, expr)
    L.append("  const Real tau = fabs(%s);" % expr)
    # ---- fp64: PRODUCT FORM, one reciprocal per reconstruction.  With b_k = bs_k + epss, P_k = prod_{j != k} b_j and
    # PI = prod_j b_j the weights alpha_k = d_k (1 + (tau / b_k)^2) are multiplied through by PI^2:
    #     alpha_k PI^2 = d_k (PI^2 + (tau P_k)^2),
    # so the r + 1 reciprocals (MUFU.RCP64H + 4 DFMA each) become 2r - 1 products and ONE quotient (num_over_den: MUFU +
    # 4 FP64); d_k and SX are folded into the integer coefficients of the candidates / the denominator at generation time.
    # r = 5: 54 -> 40 FP64 instructions and 6 -> 1 MUFU per reconstruction; r = 4: 44 -> 32 and 5 -> 1.
    # Valid while b^(2r) stays inside double range: |differences| within ~[1e-14, 1e+13] for eps = 1e-8 (fp32 would
    # underflow: the float instantiation keeps the reciprocal form below).
    L.append("  if constexpr (sizeof(Real) == 8) {")
    for k in range(r):
        L.append("    const Real b%d = bs%d + epss;" % (k, k))
    # prefix products pre[j] = b0..bj (j = 1..r-2), suffix products suf[j] = bj..b(r-1) (j = 1..r-2)
    pre = {0: "b0"}
    for j in range(1, r - 1):
        L.append("    const Real pre%d = %s * b%d;" % (j, pre[j - 1], j))
        pre[j] = "pre%d" % j
    suf = {r - 1: "b%d" % (r - 1)}
    for j in range(r - 2, 0, -1):
        L.append("    const Real suf%d = b%d * %s;" % (j, j, suf[j + 1]))
        suf[j] = "suf%d" % j
    for k in range(r):
        if k == 0:
            L.append("    const Real P0 = %s;" % suf[1])
        elif k == r - 1:
            L.append("    const Real P%d = %s;" % (k, pre[r - 2]))
        else:
            L.append("    const Real P%d = %s * %s;" % (k, pre[k - 1], suf[k + 1]))
    L.append("    const Real PI = %s * b%d;" % (pre[r - 2], r - 1))
    L.append("    const Real QQ = PI * PI;")
    for k in range(r):
        L.append("    const Real e%d = tau * P%d;" % (k, k))
    for k in range(r):
        L.append("    const Real a%d = fma(e%d, e%d, QQ);" % (k, k, k))
    # candidates carrying their ideal weight: xw_k = d_k SD xs_k (integer coefficients), denominator SX sum_k d_k SD a_k
    for k in range(r):
        y = ["d%d_%d" % (l, k) for l in range(1, r)]
        terms = [(X[k][a] * SX * d[k] * SD, y[a]) for a in range(r - 1) if X[k][a] != 0]
        expr2 = "%s * %s" % (ilit(terms[-1][0]), terms[-1][1])
        for c, nm in reversed(terms[:-1]):
            expr2 = "fma(%s, %s, %s)" % (ilit(c), nm, expr2)
        L.append("    const Real xw%d = %s;" % (k, expr2))
    num2 = "a%d * xw%d" % (r - 1, r - 1)
    den2 = "%s * a%d" % (ilit(d[r - 1] * SD * SX), r - 1)
    for k in reversed(range(r - 1)):
        num2 = "fma(a%d, xw%d, %s)" % (k, k, num2)
        den2 = "fma(%s, a%d, %s)" % (ilit(d[k] * SD * SX), k, den2)
    L.append("    return ocn::num_over_den(%s, %s);" % (num2, den2))
    L.append("  }")
    for k in range(r):
        L.append("  const Real q%d = tau * ocn::fast_rcp(bs%d + epss);" % (k, k))
    for k in range(r):
        c = d[k] * SD
        if c == 1:
            L.append("  const Real as%d = fma(q%d, q%d, Real(1.0));" % (k, k, k))
        else:
            L.append("  const Real as%d = %s * fma(q%d, q%d, Real(1.0));" % (k, ilit(c), k, k))
    num = "as%d * xs%d" % (r - 1, r - 1)
    den = "as%d" % (r - 1)
    for k in reversed(range(r - 1)):
        num = "fma(as%d, xs%d, %s)" % (k, k, num)
        den = "as%d + %s" % (k, den)
    L.append("  return (%s) * ocn::fast_rcp(%s * (%s));" % (num, ilit(SX), den))
    L.append("}")
    return "\n".join(L)


def centered_weights(order):
    """Centered(order) = symmetric part of the UpwindBiased(order-1) linear scheme (reading R4)."""
    r = order // 2
    cand, _ = value_tables(r) if r > 1 else ([[F(1)]], None)
    d = linear_weights(r, cand) if r > 1 else [F(1)]
    lin = [F(0)] * (2 * r - 1)
    for k in range(r):
        for jj in range(r):
            lin[k + jj] += d[k] * cand[k][jj]
    left, right = lin + [F(0)], [F(0)] + lin[::-1]
    return [(a + b) / 2 for a, b in zip(left, right)]


def emit():
    out = ["// weno_hi.cuh — GENERATED by gen_weno_hi.py; do not edit.  WENO7-Z / WENO9-Z in undivided-difference form and the",
           "// Centered(6) / Centered(8) advecting-velocity interpolation (SURVEY 8(f) N1; DESIGN.md R1, R2, R4, R20).",
           "#pragma once", '#include "recon.cuh"', "", "namespace ocn {", ""]
    for r in (4, 5):
        out.append(emit_function(r))
        out.append("")
    for order in (6, 8):
        w = centered_weights(order)
        half = order // 2
        # symmetric: sum_t w_t (q[m-1-t] + q[m+t]), t = 0 .. half-1, innermost pair first
        out.append("// Centered(%d) interpolation to the point between q[-1] and q[0] of a sequence with element stride s" % order)
        out.append("template <class Real> __device__ __forceinline__ Real centered%d(const Real *q, long long s) {" % order)
        S = common_denominator(w)
        expr = None
        for t in reversed(range(half)):
            pair = "(q[%d * s] + q[%d * s])" % (-1 - t, t)
            c = w[half + t] * S
            assert c.denominator == 1 and is_immediate(c)
            expr = "%s * %s" % (lit(c), pair) if expr is None else "fma(%s, %s, %s)" % (lit(c), pair, expr)
        out.append("  return (%s) * %s;      // integer weights x 1/%d" % (expr, lit(F(1, S)), S))
        out.append("}")
        out.append("")
    out.append("}  // namespace ocn")
    return "\n".join(out) + "\n"


if __name__ == "__main__":
    with open(os.path.join(HERE, "weno_hi.cuh"), "w") as f:
        f.write(emit())
    print("wrote csrc/weno_hi.cuh")
