"""oracle/gen_weno_tables.py — TEST INFRASTRUCTURE.  Exact (rational) tables of WENO(2r-1), r = 3, 4, 5, from the definition.

    python oracle/gen_weno_tables.py            # rewrites oracle/weno_tables.inc

Setting ((B8)/(B9)): finite-volume cells of width 1, cell j = [j-1/2, j+1/2]; the upwind
cell of the face is cell 0 and the face is at x = +1/2.  Candidate stencil k = 0..r-1 holds the r cells k-(r-1) .. k
(k = 0: the most upwind one; for r = 3 these are the paper's shifts s = +1, 0, -1).

  * candidate polynomial p_k (degree r-1): the unique polynomial whose CELL AVERAGES over the r cells of stencil k are
    the data ("finite volume", 1039).  AINV[k][n][j] = coefficient of x^n in p_k per unit of datum j,
    obtained by inverting the moment matrix  M[j][n] = average of x^n over cell j  in exact arithmetic.
  * candidate value  p_k(1/2) = sum_n (1/2)^n a_n                                    -> (B9) for r = 3.
  * smoothness indicator (Jiang & Shu's definition, reading R1):  beta_k = sum_{l=1}^{r-1} int_{-1/2}^{1/2} (d^l p_k/dx^l)^2 dx
    = sum_{n,n'>=1} IMAT[n][n'] a_n a_n'  with  IMAT[n][n'] = sum_l int d^l(x^n) d^l(x^n') dx.
  * ideal weights d_k: the convex combination of the candidates that equals the (2r-1)-cell linear reconstruction
    ("{c}^N ~ [c]^N when c is smooth").
  * WENO-Z global indicator tau_{2r-1} = |sum_k TAU[k] beta_k| — a READING (R20): the combination of the beta_k
    whose Taylor expansion on smooth data cancels to the highest order.  It is DERIVED here (derive_tau): beta_k on the cell
    averages of sum_m c_m x^m is sum_{m,n} E_k[m][n] c_m c_n with E_k[m][n] of order h^(m+n); the t with
    sum_k t_k (E_k[m][n] + E_k[n][m]) = 0 for every m+n <= P form a null space that shrinks as P grows; the last non-empty
    one is one-dimensional: (1,0,-1) (P = 4, tau_5 = O(h^5)), (1,3,-3,-1) (P = 6, tau_7 = O(h^7)), (1,2,-6,2,1) (P = 7,
    tau_9 = O(h^8)); scaled to coprime integers with a positive first entry.
Everything is a Fraction; the emitted file holds numerator/denominator pairs.  Nothing here is shared with the CUDA path.
"""
import os
from fractions import Fraction as F

HERE = os.path.dirname(os.path.abspath(__file__))


def mat_inv(A):
    n = len(A)
    M = [list(row) + [F(int(i == j)) for j in range(n)] for i, row in enumerate(A)]
    for c in range(n):
        p = next(r for r in range(c, n) if M[r][c] != 0)
        M[c], M[p] = M[p], M[c]
        piv = M[c][c]
        M[c] = [x / piv for x in M[c]]
        for r in range(n):
            if r != c and M[r][c] != 0:
                f = M[r][c]
                M[r] = [x - f * y for x, y in zip(M[r], M[c])]
    return [row[n:] for row in M]


def cell_average_of_monomial(n, j):
    """(1/1) * int_{j-1/2}^{j+1/2} x^n dx"""
    hi, lo = F(2 * j + 1, 2), F(2 * j - 1, 2)
    return (hi ** (n + 1) - lo ** (n + 1)) / (n + 1)


def monomial_coefficients(cells):
    """AINV[n][jj]: p(x) = sum_n (sum_jj AINV[n][jj] v[jj]) x^n has cell averages v over `cells`."""
    r = len(cells)
    M = [[cell_average_of_monomial(n, j) for n in range(r)] for j in cells]     # M a = v
    return mat_inv(M)                                                            # a = M^{-1} v


def deriv_coeff(n, l):
    """d^l/dx^l x^n = deriv_coeff * x^(n-l)"""
    c = 1
    for t in range(l):
        c *= (n - t)
    return c


def imat(r):
    """IMAT[n][n'] = sum_{l=1}^{r-1} int_{-1/2}^{1/2} d^l(x^n) d^l(x^n') dx"""
    I = [[F(0)] * r for _ in range(r)]
    for n in range(r):
        for m in range(r):
            s = F(0)
            for l in range(1, r):
                if n < l or m < l:
                    continue
                e = n + m - 2 * l
                integ = (F(1, 2) ** (e + 1) - F(-1, 2) ** (e + 1)) / (e + 1)
                s += deriv_coeff(n, l) * deriv_coeff(m, l) * integ
            I[n][m] = s
    return I


def nullspace(rows, n):
    """basis of {t : rows t = 0} by exact Gauss-Jordan elimination"""
    M = [list(row) for row in rows]
    piv, rr = [], 0
    for c in range(n):
        p = next((i for i in range(rr, len(M)) if M[i][c] != 0), None)
        if p is None:
            continue
        M[rr], M[p] = M[p], M[rr]
        M[rr] = [x / M[rr][c] for x in M[rr]]
        for i in range(len(M)):
            if i != rr and M[i][c] != 0:
                f = M[i][c]
                M[i] = [x - f * y for x, y in zip(M[i], M[rr])]
        piv.append(c)
        rr += 1
    basis = []
    for fc in (c for c in range(n) if c not in piv):
        v = [F(0)] * n
        v[fc] = F(1)
        for i, pc in enumerate(piv):
            v[pc] = -M[i][fc]
        basis.append(v)
    return basis


def derive_tau(r, betas):
    """the integer combination of the r indicators (value-form matrices `betas`) that cancels to the highest order in h"""
    from math import gcd, lcm

    def E(k, m, n):
        cells = range(k - (r - 1), k + 1)
        vm = [cell_average_of_monomial(m, j) for j in cells]
        vn = [cell_average_of_monomial(n, j) for j in cells]
        return sum(betas[k][a][b] * vm[a] * vn[b] for a in range(r) for b in range(r))
    rows, last = [], None
    for P in range(2, 4 * r):
        for m in range(0, P // 2 + 1):
            n = P - m
            rows.append([E(k, m, n) + (E(k, n, m) if m != n else 0) for k in range(r)])
        ns = nullspace(rows, r)
        if not ns:
            break
        last = ns
    assert last is not None and len(last) == 1, "the highest-order combination is not unique"
    t = last[0]
    den = 1
    for x in t:
        den = lcm(den, x.denominator)
    ints = [int(x * den) for x in t]
    g = 0
    for x in ints:
        g = gcd(g, abs(x))
    ints = [x // g for x in ints]
    if next(x for x in ints if x != 0) < 0:
        ints = [-x for x in ints]
    return ints


def tables(r):
    ainv, cand = [], []
    for k in range(r):
        cells = list(range(k - (r - 1), k + 1))
        A = monomial_coefficients(cells)
        ainv.append(A)
        cand.append([sum(A[n][jj] * F(1, 2) ** n for n in range(r)) for jj in range(r)])
    # (2r-1)-cell linear reconstruction at the face
    lin = linear_upwind(r)
    # ideal weights: sum_k d_k cand[k][jj] placed at global position k + jj must equal lin
    d = []
    for k in range(r):
        # global datum k (cell k-(r-1)) is touched by stencils 0..k only; solve forward
        acc = sum(d[kk] * cand[kk][k - kk] for kk in range(k) if 0 <= k - kk < r)
        d.append((lin[k] - acc) / cand[k][0])
    for gpos in range(2 * r - 1):
        tot = sum(d[k] * cand[k][gpos - k] for k in range(r) if 0 <= gpos - k < r)
        assert tot == lin[gpos], "ideal weights do not reproduce the linear scheme"
    assert sum(d) == 1 and all(x > 0 for x in d)
    tab = {"r": r, "ainv": ainv, "cand": cand, "imat": imat(r), "d": d, "lin": lin}
    tab["tau"] = [F(t) for t in derive_tau(r, [beta_matrix(tab, k) for k in range(r)])]
    return tab


def beta_matrix(tab, k):
    """B[jj][jj'] with beta_k = v^T B v in value form (used by the pins: Jiang-Shu's printed r = 3 indicators)."""
    r, A, I = tab["r"], tab["ainv"][k], tab["imat"]
    return [[sum(I[n][m] * A[n][a] * A[m][b] for n in range(1, r) for m in range(1, r)) for b in range(r)] for a in range(r)]


def linear_upwind(r):
    """weights of the (2r-1)-cell, order 2r-1, upwind-biased LINEAR reconstruction at the face: cells -(r-1) .. r-1"""
    full = list(range(-(r - 1), r))
    Af = monomial_coefficients(full)
    return [sum(Af[n][jj] * F(1, 2) ** n for n in range(2 * r - 1)) for jj in range(2 * r - 1)]


def centered_weights(order):
    """Centered(order), order = 2, 4, 6, 8: interpolation to the face from q[m-order/2] .. q[m+order/2-1] = the
    symmetric part of the UpwindBiased(order-1) linear scheme (PAPER.md:1013-1026 (B5)-(B7); reading R4: the
    advecting velocity of a WENO(N) flux uses Centered(N-1))."""
    lin = linear_upwind(order // 2)            # cells around the upwind cell 0, face at +1/2
    left = lin + [F(0)]                        # left-biased
    right = [F(0)] + lin[::-1]                 # its mirror image about the face (right-biased)
    return [(a + b) / 2 for a, b in zip(left, right)]


def emit():
    out = ["// oracle/weno_tables.inc — GENERATED by oracle/gen_weno_tables.py (exact rationals); do not edit.",
           "// Q(n, d) = (long double)n / (long double)d.  See the generator for the definitions and citations."]
    for r in (3, 4, 5):
        t = tables(r)
        q = lambda x: "Q(%d, %d)" % (x.numerator, x.denominator)
        out.append("static const long double WENO%d_AINV[%d][%d][%d] = {" % (2 * r - 1, r, r, r))
        for k in range(r):
            out.append("  {" + ", ".join("{" + ", ".join(q(x) for x in row) + "}" for row in t["ainv"][k]) + "},")
        out.append("};")
        out.append("static const long double WENO%d_IMAT[%d][%d] = {" % (2 * r - 1, r, r))
        for row in t["imat"]:
            out.append("  {" + ", ".join(q(x) for x in row) + "},")
        out.append("};")
        out.append("static const long double WENO%d_D[%d] = {%s};" % (2 * r - 1, r, ", ".join(q(x) for x in t["d"])))
        out.append("static const long double WENO%d_TAU[%d] = {%s};" % (2 * r - 1, r, ", ".join(q(x) for x in t["tau"])))
        cw = centered_weights(2 * r - 2)
        out.append("static const long double CENTERED%d_W[%d] = {%s};" % (2 * r - 2, 2 * r - 2, ", ".join(q(x) for x in cw)))
    return "\n".join(out) + "\n"


if __name__ == "__main__":
    with open(os.path.join(HERE, "weno_tables.inc"), "w") as f:
        f.write(emit())
    print("wrote oracle/weno_tables.inc")
