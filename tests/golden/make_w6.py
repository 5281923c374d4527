"""Writes tests/golden/w6_reaction_derivatives.txt from the equations alone (50-digit mpmath).

    python tests/golden/make_w6.py

Calls neither the oracle nor the CUDA path.  Pins the analytic chemical Jacobian (
PAPER.md:697-714 eq. (6), (A.36) PAPER.md:1057): partial derivatives of the rate of progress R = q_f - q_r of the
reaction A + B (+M) <=> AB of W2/W5 with respect to the three concentrations and to temperature, for the four
reaction types.  The elementary case has the closed forms dR/dC_A = k C_B, dR/dC_B = k C_A,
dR/dC_AB = -k/K_c; the other types are differentiated numerically by mpmath at 50 digits (mp.diff of the rate
function written from (A.7), (A.9), (A.10)-(A.13) and the third-body / falloff forms of readings G6, G8) -- a route
that shares nothing with the oracle's hand-derived chain rule.  Also the pieces of the (rho, e) form (reading G26):
e_k and c_v of the constant-c_p species, dT/dY_k|_e = -e_k/c_v from (A.25)-(A.29).
"""
import os

import mpmath as mp

mp.mp.dps = 50
R, p0 = mp.mpf("8314.46261815324"), mp.mpf(101325)
A, b, th = mp.mpf("35127309770106.477"), mp.mpf("-0.7"), mp.mpf(8590)
A0, b0, th0 = mp.mpf("1e12"), mp.mpf("-1.5"), mp.mpf(2000)              # W3 low-pressure limit
TROE = (mp.mpf("0.6"), mp.mpf(100), mp.mpf(1500), mp.mpf(5000))         # W3
# (a1, a6, a7): the W2 species, except a6 of AB = 45000 K (W2: -5000 K) so that K_c = 201 m^3/kmol at 1350 K and the
# reverse rate is of the size of the forward rate -- every term of the derivatives is visible in the values
SPECIES = ((mp.mpf("2.5"), 25000, mp.mpf("0.5")), (mp.mpf("2.5"), 30000, 1), (mp.mpf("3.5"), 45000, 4))
WEIGHT = (mp.mpf(10), mp.mpf(15), mp.mpf(25))
EFF = (mp.mpf("2.5"), mp.mpf(1), mp.mpf(12))   # third-body efficiencies of W5 (A 2.5, AB 12, default 1)
STATE = (mp.mpf(1350), (mp.mpf("0.004"), mp.mpf("0.005"), mp.mpf("0.003")))   # T, C


def k_arr(T, A=A, b=b, th=th):
    return A * T ** b * mp.e ** (-th / T)


def g_RT(sp, T):
    a1, a6, a7 = sp
    return (a1 + a6 / T) - (a1 * mp.log(T) + a7)


def Kc(T):   # A + B <=> AB, sum(nu) = -1   (A.10)
    dg = g_RT(SPECIES[2], T) - g_RT(SPECIES[0], T) - g_RT(SPECIES[1], T)
    return (p0 / (R * T)) ** (-1) * mp.e ** (-dg)


def rate(kind, T, C):
    """R = q_f - q_r of A + B (+M) <=> AB.  kind: elementary, three_body, lindemann, troe."""
    M = sum(e * c for e, c in zip(EFF, C))
    k = k_arr(T)
    if kind in ("lindemann", "troe"):
        Pr = k_arr(T, A0, b0, th0) * M / k
        F = mp.mpf(1)
        if kind == "troe":
            al, T3, T1, T2 = TROE
            Fc = (1 - al) * mp.e ** (-T / T3) + al * mp.e ** (-T / T1) + mp.e ** (-T2 / T)
            lFc = mp.log10(Fc)
            c, n = mp.mpf("-0.4") - mp.mpf("0.67") * lFc, mp.mpf("0.75") - mp.mpf("1.27") * lFc
            f1 = (mp.log10(Pr) + c) / (n - mp.mpf("0.14") * (mp.log10(Pr) + c))
            F = mp.mpf(10) ** (lFc / (1 + f1 ** 2))
        k = k * Pr / (1 + Pr) * F
    Rj = k * C[0] * C[1] - k / Kc(T) * C[2]
    return M * Rj if kind == "three_body" else Rj


def compute():
    """[(key, value)] of the fixture."""
    T, C = STATE
    out = [("T", T), ("C_A", C[0]), ("C_B", C[1]), ("C_AB", C[2])]
    for kind in ("elementary", "three_body", "lindemann", "troe"):
        out.append((f"{kind}_R", rate(kind, T, C)))
        for i, name in enumerate(("A", "B", "AB")):
            f = lambda c, i=i: rate(kind, T, tuple(c if q == i else C[q] for q in range(3)))
            out.append((f"{kind}_dR_dC_{name}", mp.diff(f, C[i])))
        out.append((f"{kind}_dR_dT", mp.diff(lambda t: rate(kind, t, C), T)))
    # closed forms of the elementary case (dR/dC_A = k C_B)
    k = k_arr(T)
    out += [("closed_dR_dC_A", k * C[1]), ("closed_dR_dC_B", k * C[0]), ("closed_dR_dC_AB", -k / Kc(T))]
    # (rho, e) form: e_k = ((a1 - 1) T + a6) R / W_k for constant-c_p species (A.26), c_v = sum_k Y_k (a1 - 1) R / W_k
    rho = sum(c * w for c, w in zip(C, WEIGHT))
    Y = [c * w / rho for c, w in zip(C, WEIGHT)]
    e = [((sp[0] - 1) * T + sp[1]) * R / w for sp, w in zip(SPECIES, WEIGHT)]
    cv = sum(y * (sp[0] - 1) * R / w for y, sp, w in zip(Y, SPECIES, WEIGHT))
    out += [("rho", rho), ("e_A", e[0]), ("e_B", e[1]), ("e_AB", e[2]), ("cv", cv)]
    return out


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "w6_reaction_derivatives.txt")
    with open(path, "w") as f:
        f.write("# W6: derivatives of the rate of progress of A + B (+M) <=> AB (W2 species with a6 of AB = 45000 K, W1 Arrhenius triple\n"
                "# PAPER.md:205-208, W3 falloff parameters, W5 efficiencies) at T = 1350 K, C = (0.004, 0.005, 0.003) kmol/m^3.\n"
                "# Written by tests/golden/make_w6.py: 50-digit mpmath, numerical differentiation (mp.diff) of the rate written\n"
                "# from (A.7), (A.9)-(A.13) and readings G6, G8; closed_* are the closed forms of the elementary case\n"
                "# (PAPER.md:315).  e_k, c_v: (A.26), (A.29) for the (rho, e) form of the Jacobian (reading G26).\n")
        for key, val in compute():
            f.write(f"{key} {mp.nstr(val, 20)}\n")
    print(path)


if __name__ == "__main__":
    main()
