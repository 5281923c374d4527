"""Prints the polynomial coefficients of pyro_math.cuh: p(r) ~ 2^r on [-1/2, 1/2].

Near-minimax by interpolation at Chebyshev nodes in 60-digit arithmetic, constant term
forced to 1 (so 2^0 = 1 exactly), coefficients rounded to double; the script then reports
the maximum relative error of the rounded polynomial evaluated exactly.  Usage:
    python gen_exp2_coeffs.py [degree ...]
"""
import sys

import mpmath as mp

mp.mp.dps = 60


def fit(deg):
    # interpolate q(r) = (2^r - 1)/r (degree deg-1) at Chebyshev nodes, p = 1 + r q(r)
    n = deg
    nodes = [mp.mpf(1) / 2 * mp.cos(mp.pi * (2 * i + 1) / (2 * n)) for i in range(n)]
    f = lambda r: mp.expm1(r * mp.log(2)) / r if abs(r) > mp.mpf("1e-40") else mp.log(2)
    A = mp.matrix(n, n)
    y = mp.matrix(n, 1)
    for i, r in enumerate(nodes):
        for j in range(n):
            A[i, j] = r**j
        y[i] = f(r)
    c = mp.lu_solve(A, y)
    coef = [1.0] + [float(c[j]) for j in range(n)]
    # max relative error of the double-rounded coefficients, exact evaluation
    worst = mp.mpf(0)
    for i in range(4001):
        r = mp.mpf(-1) / 2 + mp.mpf(i) / 4000
        p = mp.mpf(0)
        for cj in reversed(coef):
            p = p * r + mp.mpf(cj)
        worst = max(worst, abs(p / mp.mpf(2) ** r - 1))
    return coef, worst


if __name__ == "__main__":
    for deg in [int(a) for a in sys.argv[1:]] or [8, 9, 10, 11]:
        coef, worst = fit(deg)
        print(f"// degree {deg}: max relative error {mp.nstr(worst, 3)} (exact arithmetic)")
        for j, cj in enumerate(coef):
            print(f"//   c{j} = {cj!r}  ({float.hex(cj)})")
