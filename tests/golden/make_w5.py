"""Writes tests/golden/w5_three_body_and_falloff_rates.txt from the equations alone (50-digit mpmath).

    python tests/golden/make_w5.py

Calls neither the oracle nor the CUDA path.  Pins reading G8: a three-body
reaction has R = [M] (q_f - q_r); a falloff reaction has [M] only inside P_r, and its reverse rate
uses the same effective rate coefficient, q_r = k_eff / K_c * prod C^nu''.
Equations: (A.7) PAPER.md:916, (A.9) :925, (A.10)-(A.13) :932-943; third-body / falloff forms per
reading G6 (the paper only cites them).
"""
import os

import mpmath as mp

mp.mp.dps = 50
R, p0 = mp.mpf("8314.46261815324"), mp.mpf(101325)
A, b, th = mp.mpf("35127309770106.477"), mp.mpf("-0.7"), mp.mpf(8590)
SPECIES = ((mp.mpf("2.5"), 25000, mp.mpf("0.5")), (mp.mpf("2.5"), 30000, 1), (mp.mpf("3.5"), -5000, 4))   # (a1, a6, a7)


def k_arr(T):
    return A * T ** b * mp.e ** (-th / T)


def g_RT(sp, T):
    a1, a6, a7 = sp
    return (a1 + a6 / T) - (a1 * mp.log(T) + a7)


def Kc(T):   # A + B <=> AB, sum(nu) = -1
    dg = g_RT(SPECIES[2], T) - g_RT(SPECIES[0], T) - g_RT(SPECIES[1], T)
    return (p0 / (R * T)) ** (-1) * mp.e ** (-dg)


def main():
    out = []
    # three-body at 1500 K, C = (2e-3, 3e-3, 1e-3), efficiencies A: 2.5, AB: 12, default 1
    T = mp.mpf(1500)
    C = (mp.mpf("2e-3"), mp.mpf("3e-3"), mp.mpf("1e-3"))
    M = mp.mpf("2.5") * C[0] + 1 * C[1] + 12 * C[2]
    kf = k_arr(T)
    qf = M * kf * C[0] * C[1]
    qr = M * kf / Kc(T) * C[2]
    out += [("tb_M", M), ("tb_kf", kf), ("tb_qf", qf), ("tb_qr", qr), ("tb_omega_AB", qf - qr)]
    # falloff at 1200 K (the W3 state): C = (0.004, 0.005, 0.001), unit efficiencies, [M] = 0.01
    T = mp.mpf(1200)
    C = (mp.mpf("0.004"), mp.mpf("0.005"), mp.mpf("0.001"))
    M = C[0] + C[1] + C[2]
    k0 = mp.mpf("1e12") * T ** mp.mpf("-1.5") * mp.e ** (-mp.mpf(2000) / T)
    Pr = k0 * M / k_arr(T)
    k_lind = k_arr(T) * Pr / (1 + Pr)
    Fc = mp.mpf("0.4") * mp.e ** (-T / 100) + mp.mpf("0.6") * mp.e ** (-T / 1500) + mp.e ** (-mp.mpf(5000) / T)
    lFc = mp.log10(Fc)
    c, n = mp.mpf("-0.4") - mp.mpf("0.67") * lFc, mp.mpf("0.75") - mp.mpf("1.27") * lFc
    f1 = (mp.log10(Pr) + c) / (n - mp.mpf("0.14") * (mp.log10(Pr) + c))
    k_troe = k_lind * mp.mpf(10) ** (lFc / (1 + f1 ** 2))
    out += [("fo_M", M), ("fo_Kc", Kc(T))]
    for name, k in (("lindemann", k_lind), ("troe", k_troe)):
        out += [(f"fo_qf_{name}", k * C[0] * C[1]), (f"fo_qr_{name}", k / Kc(T) * C[2])]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "w5_three_body_and_falloff_rates.txt")
    with open(path, "w") as f:
        f.write("# W5: where [M] multiplies (reading G8).  Written by tests/golden/make_w5.py (50-digit mpmath, equations only).\n"
                "# Reaction A + B (+M) <=> AB with the W2 species and the W1 Arrhenius triple (PAPER.md:205-208).\n"
                "# tb_*: three-body at 1500 K, C = (2e-3, 3e-3, 1e-3) kmol/m^3, efficiencies A 2.5, AB 12, default 1:\n"
                "#       q_f = [M] k_f C_A C_B, q_r = [M] k_f/K_c C_AB   ((A.7) PAPER.md:916 times [M]).\n"
                "# fo_*: falloff at 1200 K, the W3 state C = (0.004, 0.005, 0.001), [M] = 0.01, low-pressure and Troe\n"
                "#       parameters of W3: q_f = k_eff C_A C_B with NO extra [M]; q_r = k_eff/K_c C_AB.\n")
        for key, val in out:
            f.write(f"{key} {mp.nstr(val, 20)}\n")
    print(path)


if __name__ == "__main__":
    main()
