"""Exact (rational / big-integer) references used ONLY to pin the oracle.

They are the problem's definition written out in exact arithmetic -- no floating point,
no code from oracle/ or from the CUDA path:

* ``exact_h_by_definition``: the unique H (h33 = 1) with H*[src_k;1] ~ [dst_k;1], k = 0..3,
  by solving the 8 linear equations of Eq. 1-3 over the rationals.
* ``defining_property_holds``: dst_k x (H*src_k) == 0 exactly (Eq. 1).
* ``exact_inlier_count``: RANSAC inlier count by the definition (reading R9) with rational
  arithmetic: |pi(H s) - d|^2 <= t^2, W == 0 -> outlier.
"""
from fractions import Fraction
from itertools import combinations


def _solve_rational(A, b):
    n = len(A)
    M = [[Fraction(v) for v in row] + [Fraction(bv)] for row, bv in zip(A, b)]
    for col in range(n):
        piv = next((r for r in range(col, n) if M[r][col] != 0), None)
        if piv is None:
            raise ZeroDivisionError("singular system")
        M[col], M[piv] = M[piv], M[col]
        inv = 1 / M[col][col]
        M[col] = [v * inv for v in M[col]]
        for r in range(n):
            if r != col and M[r][col] != 0:
                f = M[r][col]
                M[r] = [vr - f * vc for vr, vc in zip(M[r], M[col])]
    return [M[r][n] for r in range(n)]


def exact_h_by_definition(src, dst):
    """src, dst: 4 (x,y) pairs of ints/Fractions.  Returns 3x3 list of Fractions with h33 = 1."""
    A, b = [], []
    for (x, y), (u, v) in zip(src, dst):
        x, y, u, v = Fraction(x), Fraction(y), Fraction(u), Fraction(v)
        # u = (h11 x + h12 y + h13) / (h31 x + h32 y + 1) and likewise v
        A.append([x, y, 1, 0, 0, 0, -u * x, -u * y]); b.append(u)
        A.append([0, 0, 0, x, y, 1, -v * x, -v * y]); b.append(v)
    h = _solve_rational(A, b)
    return [[h[0], h[1], h[2]], [h[3], h[4], h[5]], [h[6], h[7], Fraction(1)]]


def apply_exact(H, x, y):
    X = H[0][0] * x + H[0][1] * y + H[0][2]
    Y = H[1][0] * x + H[1][1] * y + H[1][2]
    W = H[2][0] * x + H[2][1] * y + H[2][2]
    return X, Y, W


def defining_property_holds(H, src, dst):
    """dst_k x (H src_k) == 0 exactly and H src_k != 0, for every k."""
    for (x, y), (u, v) in zip(src, dst):
        X, Y, W = apply_exact(H, x, y)
        if (X, Y, W) == (0, 0, 0):
            return False
        if (v * W - Y, X - u * W, u * Y - v * X) != (0, 0, 0):
            return False
    return True


def exact_inlier_count(H, src_xy, dst_xy, t):
    t2 = Fraction(t) ** 2
    c = 0
    for (x, y), (u, v) in zip(src_xy, dst_xy):
        X, Y, W = apply_exact(H, Fraction(x), Fraction(y))
        if W == 0:
            continue
        ex, ey = X / W - Fraction(u), Y / W - Fraction(v)
        if ex * ex + ey * ey <= t2:
            c += 1
    return c


def all_quads(n):
    return list(combinations(range(n), 4))
