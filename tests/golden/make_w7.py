"""Writes tests/golden/w7_transport.txt from the equations alone (50-digit mpmath).

    python tests/golden/make_w7.py

Calls neither the oracle nor the CUDA path.  Pins the mixture-averaged transport formulas (A.18)-(A.24)
PAPER.md:968-996 on a hand-written three-species mixture at T = 900 K: species
viscosities (A.22), Wilke factors (A.21), mixture viscosity (A.20), species and mixture conductivity (A.24), (A.23),
binary (A.19) and mixture-averaged (A.18) diffusivities, mole fractions from (A.3).
"""
import os

import mpmath as mp

mp.mp.dps = 50
T = mp.mpf(900)
WEIGHT = (mp.mpf("2.016"), mp.mpf("31.998"), mp.mpf("28.014"))
Y = (mp.mpf("0.05"), mp.mpf("0.25"), mp.mpf("0.70"))
VISC = ((mp.mpf("-2e-4"), mp.mpf("3e-4"), mp.mpf("-2e-5"), mp.mpf("1e-6"), mp.mpf("-2e-8")),
        (mp.mpf("-4e-4"), mp.mpf("5e-4"), mp.mpf("-4e-5"), mp.mpf("2e-6"), mp.mpf("-5e-8")),
        (mp.mpf("-3e-4"), mp.mpf("4e-4"), mp.mpf("-3e-5"), mp.mpf("1.5e-6"), mp.mpf("-3e-8")))
COND = ((mp.mpf("1e-3"), mp.mpf("5e-4"), mp.mpf("1e-4"), mp.mpf("-5e-6"), mp.mpf("2e-7")),
        (mp.mpf("-2e-4"), mp.mpf("1e-4"), mp.mpf("2e-5"), mp.mpf("-1e-6"), mp.mpf("5e-8")),
        (mp.mpf("-1e-4"), mp.mpf("8e-5"), mp.mpf("3e-5"), mp.mpf("-2e-6"), mp.mpf("6e-8")))
# symmetric pair table, m = 0..4
DIFF = {(0, 1): (mp.mpf("-6e-6"), mp.mpf("2e-6"), mp.mpf("1e-7"), mp.mpf("2e-9"), mp.mpf("1e-10")),
        (0, 2): (mp.mpf("-5e-6"), mp.mpf("1.8e-6"), mp.mpf("1.2e-7"), mp.mpf("1e-9"), mp.mpf("2e-10")),
        (1, 2): (mp.mpf("-1.5e-6"), mp.mpf("5e-7"), mp.mpf("3e-8"), mp.mpf("5e-10"), mp.mpf("4e-11"))}


def poly(c, x):
    return sum(cm * x ** m for m, cm in enumerate(c))


def compute():
    lnT, sq = mp.log(T), mp.sqrt(T)
    W = 1 / sum(y / w for y, w in zip(Y, WEIGHT))
    X = [W * y / w for y, w in zip(Y, WEIGHT)]
    mu = [sq * poly(VISC[k], lnT) ** 2 for k in range(3)]
    ka = [sq * poly(COND[k], lnT) for k in range(3)]
    phi = [[(1 + mp.sqrt(mu[k] / mu[j] * mp.sqrt(WEIGHT[j] / WEIGHT[k]))) ** 2 / mp.sqrt(8 * (1 + WEIGHT[k] / WEIGHT[j]))
            for j in range(3)] for k in range(3)]
    mu_mix = sum(X[k] * mu[k] / sum(phi[k][j] * X[j] for j in range(3)) for k in range(3))
    ka_mix = (sum(x * k for x, k in zip(X, ka)) + 1 / sum(x / k for x, k in zip(X, ka))) / 2
    D = lambda k, j: sq * poly(DIFF[(min(k, j), max(k, j))], lnT)
    Dkm = [(W - X[k] * WEIGHT[k]) / W / sum(X[j] / D(k, j) for j in range(3) if j != k) for k in range(3)]
    out = [("W", W)] + [(f"X_{k}", X[k]) for k in range(3)] + [(f"mu_{k}", mu[k]) for k in range(3)]
    out += [(f"kappa_{k}", ka[k]) for k in range(3)] + [(f"phi_{k}{j}", phi[k][j]) for k in range(3) for j in range(3)]
    out += [("D_01", D(0, 1)), ("D_02", D(0, 2)), ("D_12", D(1, 2)), ("mu_mix", mu_mix), ("kappa_mix", ka_mix)]
    out += [(f"D_{k}m", Dkm[k]) for k in range(3)]
    return out


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "w7_transport.txt")
    with open(path, "w") as f:
        f.write("# W7: mixture-averaged transport (A.18)-(A.24) PAPER.md:968-996 of a hand-written three-species mixture at 900 K,\n"
                "# Y = (0.05, 0.25, 0.70), W = (2.016, 31.998, 28.014); fits in make_w7.py.  50-digit mpmath, equations only.\n")
        for key, val in compute():
            f.write(f"{key} {mp.nstr(val, 20)}\n")
    print(path)


if __name__ == "__main__":
    main()
