"""Pins of the CPU oracle (no GPU): what the paper and the mathematics fix.

P1-P16 and W1-W4 of SURVEY.md section 8(c); each test names the passage it pins.
"""
import os

import mpmath as mp
import numpy as np
import pytest

from conftest import read_golden
from oracle import oracle
from paper_2503_24286_b200 import inputs
from paper_2503_24286_b200.inputs import (ELEMENTARY, FALLOFF_LINDEMANN, FALLOFF_TROE, THREE_BODY,
                                          P_ATM, R_UNIVERSAL, simple_mechanism)

W1 = dict(A=35127309770106.477, b=-0.7, theta=8590.0)


def _w2_species():
    z = [0.0] * 4
    return [
        dict(W=10.0, lo=[2.5, *z, 25000.0, 0.5]),
        dict(W=15.0, lo=[2.5, *z, 30000.0, 1.0]),
        dict(W=25.0, lo=[3.5, *z, -5000.0, 4.0]),
    ]


def _w2_mech(**rx):
    r = dict(reac={0: 1, 1: 1}, prod={2: 1}, **W1)
    r.update(rx)
    return simple_mechanism(_w2_species(), [r])


def _state_from_C(mech, C):
    """rho, Y giving the concentrations C (A.8): rho = sum C_k W_k, Y_k = C_k W_k / rho."""
    C = np.asarray(C, dtype=np.float64)
    rho = float((C * mech.mol_weight).sum())
    return rho, C * mech.mol_weight / rho


# ---------------------------------------------------------------- fixtures are what the equations give
def test_golden_values_recomputed_with_mpmath(golden_dir):
    mp.mp.dps = 50
    A, b, th = mp.mpf("35127309770106.477"), mp.mpf("-0.7"), mp.mpf(8590)
    k = lambda T: A * mp.mpf(T) ** b * mp.e ** (-th / T)
    for line in open(os.path.join(golden_dir, "w1_arrhenius.txt")):
        if line.startswith("#") or not line.strip():
            continue
        T, val = line.split()
        assert abs(k(int(T)) / mp.mpf(val) - 1) < mp.mpf("1e-16")
    g = read_golden(os.path.join(golden_dir, "w2_single_reaction.txt"))
    T = mp.mpf(1500)
    R, p0 = mp.mpf("8314.46261815324"), mp.mpf(101325)
    gk = lambda a1, a6, a7: (a1 + a6 / T) - (a1 * mp.log(T) + a7)
    gA, gB, gAB = gk(mp.mpf("2.5"), 25000, mp.mpf("0.5")), gk(mp.mpf("2.5"), 30000, 1), gk(mp.mpf("3.5"), -5000, 4)
    lnKc = -1 * mp.log(p0 / (R * T)) - (gAB - gA - gB)
    Kc = mp.e ** lnKc
    rf = k(1500) * mp.mpf("2e-3") * mp.mpf("3e-3")
    rr = k(1500) / Kc * mp.mpf("1e-3")
    for key, val in (("g_RT_A", gA), ("g_RT_B", gB), ("g_RT_AB", gAB), ("sum_nu_g", gAB - gA - gB),
                     ("ln_p0_RT", mp.log(p0 / (R * T))), ("ln_Kc", lnKc), ("Kc", Kc), ("kf", k(1500)),
                     ("rf", rf), ("rr", rr), ("R", rf - rr), ("C_AB_eq", Kc * mp.mpf("2e-3") * mp.mpf("3e-3"))):
        assert abs(val / mp.mpf(g[key]) - 1) < mp.mpf("1e-15"), key
    g = read_golden(os.path.join(golden_dir, "w3_falloff.txt"))
    T = mp.mpf(1200)
    k0 = mp.mpf("1e12") * T ** mp.mpf("-1.5") * mp.e ** (-mp.mpf(2000) / T)
    Pr = k0 * mp.mpf("0.01") / k(1200)
    Fc = mp.mpf("0.4") * mp.e ** (-T / 100) + mp.mpf("0.6") * mp.e ** (-T / 1500) + mp.e ** (-mp.mpf(5000) / T)
    lFc = mp.log10(Fc)
    c, n = mp.mpf("-0.4") - mp.mpf("0.67") * lFc, mp.mpf("0.75") - mp.mpf("1.27") * lFc
    f1 = (mp.log10(Pr) + c) / (n - mp.mpf("0.14") * (mp.log10(Pr) + c))
    F = mp.mpf(10) ** (lFc / (1 + f1**2))
    for key, val in (("k_inf", k(1200)), ("k0", k0), ("Pr", Pr), ("k_lindemann", k(1200) * Pr / (1 + Pr)),
                     ("Fcent", Fc), ("log10_Fcent", lFc), ("c", c), ("n", n), ("f1", f1), ("F", F),
                     ("k_troe", k(1200) * Pr / (1 + Pr) * F)):
        assert abs(val / mp.mpf(g[key]) - 1) < mp.mpf("1e-15"), key
    g = read_golden(os.path.join(golden_dir, "w4_newton.txt"))
    assert abs(((mp.mpf("2.5") * mp.mpf("1234.5") - 1000) * R / mp.mpf("28.014")) / mp.mpf(g["e"]) - 1) < 1e-16
    assert abs((mp.mpf("2.5") * R / mp.mpf("28.014")) / mp.mpf(g["cv"]) - 1) < 1e-16


# ---------------------------------------------------------------- W1-W4
@pytest.mark.parametrize("real", ["f64", "f80"])
def test_w1_arrhenius_value_paper_triple(golden_dir, real):
    """(A.9) PAPER.md:925 with the triple printed at PAPER.md:205-208."""
    mech = simple_mechanism(_w2_species(), [dict(reac={0: 1}, prod={1: 1}, reversible=0, **W1)])
    o = oracle.Oracle(mech, real)
    for line in open(os.path.join(golden_dir, "w1_arrhenius.txt")):
        if line.startswith("#") or not line.strip():
            continue
        T, val = line.split()
        d = o.reaction_detail(0, 1.0, float(T), [1.0, 0.0, 0.0])
        assert abs(float(d["kf"]) / float(val) - 1) < 4e-15


def test_w2_single_reaction_hand_computation(golden_dir):
    """(A.7), (A.10)-(A.13): hand-computed g/RT, Kc, r_f, r_r, R of A + B <=> AB."""
    g = {k: float(v) for k, v in read_golden(os.path.join(golden_dir, "w2_single_reaction.txt")).items()}
    mech = _w2_mech()
    o = oracle.Oracle(mech)
    T = 1500.0
    for k, key in enumerate(("g_RT_A", "g_RT_B", "g_RT_AB")):
        assert abs(o.species_thermo(k, T)[3] / g[key] - 1) < 1e-14
    rho, Y = _state_from_C(mech, [2e-3, 3e-3, 1e-3])
    d = o.reaction_detail(0, rho, T, Y)
    assert abs(d["Kc"] / g["Kc"] - 1) < 1e-13
    assert abs(d["kf"] / g["kf"] - 1) < 4e-15
    assert abs(d["qf"] / g["rf"] - 1) < 1e-14
    assert abs(d["qr"] / g["rr"] - 1) < 1e-13
    om, bd = o.get_net_production_rates([rho], [T], Y[:, None])
    assert abs(om[2, 0] / g["R"] - 1) < 1e-14 and om[0, 0] == -om[2, 0] and om[1, 0] == -om[2, 0]
    assert abs(bd[0, 0] / (g["rf"] + g["rr"]) - 1) < 1e-14
    # equilibrium concentration of AB makes the net rate vanish (P6, elementary)
    rho, Y = _state_from_C(mech, [2e-3, 3e-3, g["C_AB_eq"]])
    d = o.reaction_detail(0, rho, T, Y)
    assert abs(d["qf"] - d["qr"]) <= 1e-13 * d["qf"]


def test_w3_falloff_hand_computation(golden_dir):
    """Lindemann and Troe (reading G6) against the hand computation."""
    g = {k: float(v) for k, v in read_golden(os.path.join(golden_dir, "w3_falloff.txt")).items()}
    low = dict(A0=1e12, b0=-1.5, theta0=2000.0)
    T = 1200.0
    for rtype, troe, kkey in ((FALLOFF_LINDEMANN, None, "k_lindemann"), (FALLOFF_TROE, (0.6, 100.0, 1500.0, 5000.0), "k_troe")):
        rx = dict(type=rtype, **low)
        if troe:
            rx["troe"] = troe
        mech = _w2_mech(**rx)
        o = oracle.Oracle(mech)
        # [M] = 0.01 with unit efficiencies: total concentration 0.01
        rho, Y = _state_from_C(mech, [0.004, 0.005, 0.001])
        d = o.reaction_detail(0, rho, T, Y)
        assert abs(d["M"] / 0.01 - 1) < 1e-14
        assert abs(d["k_inf"] / g["k_inf"] - 1) < 4e-15
        assert abs(d["k0"] / g["k0"] - 1) < 4e-15
        assert abs(d["Pr"] / g["Pr"] - 1) < 1e-14
        assert abs(d["kf"] / g[kkey] - 1) < 1e-13
        if troe:
            assert abs(d["F"] / g["F"] - 1) < 1e-13


def test_w4_newton_constant_cp_one_step(golden_dir):
    """(A.25)-(A.30): e, c_v closed form; Newton converges in one step when e is linear in T (P8)."""
    g = {k: float(v) for k, v in read_golden(os.path.join(golden_dir, "w4_newton.txt")).items()}
    mech = simple_mechanism([dict(W=28.014, lo=[3.5, 0, 0, 0, 0, -1000.0, 0.0])], [])
    o = oracle.Oracle(mech)
    assert abs(o.mixture_e(1234.5, [1.0]) / g["e"] - 1) < 1e-15
    assert abs(o.mixture_cv(1234.5, [1.0]) / g["cv"] - 1) < 1e-15
    for Tg in (300.0, 1234.5 * 0.9, 2999.0):
        T, it, cv = o.get_temperature([g["e"]], np.array([[1.0]]), [Tg], tol=1e-6, max_iter=10)
        assert abs(T[0] / 1234.5 - 1) < 1e-14
        assert it[0] <= 2 and cv[0] == 1   # step 1 lands on T*, step 2 only confirms |dT| < tol
        T1, it1, _ = o.get_temperature([g["e"]], np.array([[1.0]]), [Tg], tol=1e-6, max_iter=1)
        assert abs(T1[0] / 1234.5 - 1) < 1e-14


def test_w5_three_body_factor_and_no_extra_factor_on_falloff(golden_dir):
    """Reading G8: a three-body reaction has q_f = [M] k_f C_A C_B and q_r = [M] k_f/K_c C_AB; a falloff
    reaction has [M] only inside P_r (q_f = k_eff C_A C_B, no extra factor) and its reverse rate uses the
    same effective coefficient.  Closed-form values from the equations (make_w5.py), cross-checked here
    against the W2 / W3 fixtures of SURVEY.md section 8(c)."""
    g = {k: float(v) for k, v in read_golden(os.path.join(golden_dir, "w5_three_body_and_falloff_rates.txt")).items()}
    g2 = {k: float(v) for k, v in read_golden(os.path.join(golden_dir, "w2_single_reaction.txt")).items()}
    g3 = {k: float(v) for k, v in read_golden(os.path.join(golden_dir, "w3_falloff.txt")).items()}
    # the fixture is consistent with the survey's hand computations
    assert abs(g["tb_qf"] / (0.02 * g2["rf"]) - 1) < 1e-15 and abs(g["tb_qr"] / (0.02 * g2["rr"]) - 1) < 1e-15
    assert abs(g["fo_qf_lindemann"] / (g3["k_lindemann"] * 0.004 * 0.005) - 1) < 1e-15
    assert abs(g["fo_qf_troe"] / (g3["k_troe"] * 0.004 * 0.005) - 1) < 1e-15
    assert abs(g["fo_qr_troe"] / (g3["k_troe"] / g["fo_Kc"] * 0.001) - 1) < 1e-15
    # three-body
    mech = _w2_mech(type=THREE_BODY, eff={0: 2.5, 2: 12.0})
    for real, tol in (("f64", 2e-14), ("f80", 2e-15)):
        o = oracle.Oracle(mech, real)
        rho, Y = _state_from_C(mech, [2e-3, 3e-3, 1e-3])
        d = o.reaction_detail(0, rho, 1500.0, Y)
        assert abs(float(d["M"]) / g["tb_M"] - 1) < 1e-14
        assert abs(float(d["kf"]) / g["tb_kf"] - 1) < 4e-15
        assert abs(float(d["qf"]) / g["tb_qf"] - 1) < tol
        assert abs(float(d["qr"]) / g["tb_qr"] - 1) < 50 * tol   # K_c carries exp(33): conditioning
        om, bd = o.get_net_production_rates([rho], [1500.0], Y[:, None])
        assert abs(float(om[2, 0]) / g["tb_omega_AB"] - 1) < tol
        assert om[0, 0] == -om[2, 0] and om[1, 0] == -om[2, 0]
        assert abs(float(bd[2, 0]) / (g["tb_qf"] + g["tb_qr"]) - 1) < tol
    # falloff: no extra [M] on the rate of progress, reverse rate from the same effective coefficient
    low = dict(A0=1e12, b0=-1.5, theta0=2000.0)
    for rtype, troe, name in ((FALLOFF_LINDEMANN, None, "lindemann"), (FALLOFF_TROE, (0.6, 100.0, 1500.0, 5000.0), "troe")):
        rx = dict(type=rtype, **low)
        if troe:
            rx["troe"] = troe
        mech = _w2_mech(**rx)
        o = oracle.Oracle(mech)
        rho, Y = _state_from_C(mech, [0.004, 0.005, 0.001])
        d = o.reaction_detail(0, rho, 1200.0, Y)
        assert abs(d["M"] / g["fo_M"] - 1) < 1e-14
        assert abs(d["Kc"] / g["fo_Kc"] - 1) < 1e-13
        assert abs(d["qf"] / g["fo_qf_" + name] - 1) < 1e-13
        assert abs(d["qr"] / g["fo_qr_" + name] - 1) < 2e-13
        om, _ = o.get_net_production_rates([rho], [1200.0], Y[:, None])
        assert abs(om[2, 0] / (g["fo_qf_" + name] - g["fo_qr_" + name]) - 1) < 1e-13


def test_third_body_efficiency_lists_in_any_order():
    """[M] = sum_k eff_k C_k (G6) does not depend on the order in which the non-default efficiencies are
    listed (include/pyro.h: any order, each species at most once)."""
    mech = _w2_mech(type=THREE_BODY, eff={0: 2.5, 2: 12.0})
    rev = _w2_mech(type=THREE_BODY, eff={0: 2.5, 2: 12.0})
    rev.eff_species = rev.eff_species[::-1].copy()
    rev.eff_value = rev.eff_value[::-1].copy()
    assert list(rev.eff_species) == [2, 0]
    rho, Y = _state_from_C(mech, [2e-3, 3e-3, 1e-3])
    a = oracle.Oracle(mech).reaction_detail(0, rho, 1500.0, Y)
    b = oracle.Oracle(rev).reaction_detail(0, rho, 1500.0, Y)
    assert a["M"] == b["M"] and abs(a["M"] / 0.02 - 1) < 1e-14 and a["qf"] == b["qf"]


# ---------------------------------------------------------------- P1-P4 thermodynamics
@pytest.fixture(scope="module")
def cfg0():
    mech = inputs.config_mechanism(0)
    return mech, oracle.Oracle(mech), oracle.Oracle(mech, "f80")


def test_p1_nasa_continuity_at_tmid(cfg0):
    """Generated high range matches the low range at T_mid (H1); branch is T < T_mid ? lo : hi (G10)."""
    mech, o, _ = cfg0
    Tm = 1000.0
    below, above = np.nextafter(Tm, 0.0), np.nextafter(Tm, 2 * Tm)
    for k in range(mech.n_species):
        lo = np.array(o.species_thermo(k, below))
        at = np.array(o.species_thermo(k, Tm))
        hi = np.array(o.species_thermo(k, above))
        scale = np.abs(at[:3]).max()
        assert np.all(np.abs(lo - at) <= 1e-11 * scale)
        assert np.all(np.abs(hi - at) <= 1e-12 * scale)
    # the branch really switches coefficient sets: make a species discontinuous on purpose
    sp = [dict(W=1.0, lo=[3, 0, 0, 0, 0, 0, 0], hi=[5, 0, 0, 0, 0, 0, 0])]
    o2 = oracle.Oracle(simple_mechanism(sp, []))
    assert o2.species_thermo(0, below)[0] == 3.0
    assert o2.species_thermo(0, Tm)[0] == 5.0
    assert o2.species_thermo(0, above)[0] == 5.0


@pytest.mark.parametrize("T", [350.0, 900.0, 1400.0, 2800.0])
def test_p2_p3_cp_is_dh_dT_and_ds_dT(cfg0, T):
    """c_p = dh/dT (G3, (A.12)) and c_p/T = ds/dT (G2), by central differences in long double."""
    mech, _, o80 = cfg0
    L = np.longdouble
    dT = L(T) * L(1e-5)
    for k in range(mech.n_species):
        cp, h, s, g = o80.species_thermo(k, L(T))
        _, hp, sp, gp = o80.species_thermo(k, L(T) + dT)
        _, hm, sm, gm = o80.species_thermo(k, L(T) - dT)
        dh = (hp * (L(T) + dT) - hm * (L(T) - dT)) / (2 * dT)   # d(h/R)/dT
        ds = (sp - sm) / (2 * dT)
        assert abs(dh / cp - 1) < 1e-8
        assert abs(ds * L(T) / cp - 1) < 1e-8
        # d(g/RT)/dT = -h/(R T^2)
        dg = (gp - gm) / (2 * dT)
        assert abs(dg / (-h / L(T)) - 1) < 1e-7 or abs(dg + h / L(T)) < 1e-10
        assert g == h - s   # (A.11)


def test_p4_cv_is_de_dT(cfg0):
    """(A.29) per unit mass (G4): c_v = d e/dT of (A.25)-(A.26)."""
    mech, _, o80 = cfg0
    st = inputs.config_states(0, n=16)
    L = np.longdouble
    for p in range(16):
        T = L(st["T"][p])
        if abs(float(T) - 1000.0) < 1.0:
            continue
        Y = st["Y"][:, p]
        dT = T * L(1e-5)
        de = (o80.mixture_e(T + dT, Y) - o80.mixture_e(T - dT, Y)) / (2 * dT)
        assert abs(de / o80.mixture_cv(T, Y) - 1) < 1e-8


# ---------------------------------------------------------------- P5 conservation, P15 brute force
@pytest.mark.parametrize("cfg", [0, 2])
def test_p5_mass_and_element_conservation_and_p15_dense(cfg):
    mech = inputs.config_mechanism(cfg)
    o = oracle.Oracle(mech)
    n = 256 if cfg == 0 else 64
    st = inputs.config_states(cfg, n=n)
    om, bd, rf, rr = o.get_net_production_rates(st["rho"], st["T"], st["Y"], want_rates=True)
    assert np.isfinite(om).all() and np.isfinite(rf).all() and np.isfinite(rr).all()
    W = mech.mol_weight[:, None]
    assert np.all(np.abs((W * om).sum(0)) <= 1e-13 * (W * bd).sum(0))
    for e in range(mech.n_elements):
        ne = mech.elem_comp[:, e][:, None].astype(np.float64)
        assert np.all(np.abs((ne * om).sum(0)) <= 1e-13 * (ne * bd).sum(0) + 1e-300)
    # P15: dense nu (N_s x N_r) mat-vec equals the sparse accumulation; bound likewise
    nup, nupp = mech.nu_dense()
    nu = (nupp - nup).astype(np.float64)
    dense = nu @ (rf - rr)
    assert np.all(np.abs(dense - om) <= 1e-13 * bd + 1e-300)
    assert np.allclose(np.abs(nu) @ (np.abs(rf) + np.abs(rr)), bd, rtol=1e-13, atol=0)
    # the generator's reactions are element balanced
    assert np.all(mech.elem_comp.T.astype(np.int64) @ (nupp - nup) == 0)


# ---------------------------------------------------------------- P6 detailed balance, P7
@pytest.mark.parametrize("rtype", [ELEMENTARY, THREE_BODY, FALLOFF_LINDEMANN, FALLOFF_TROE])
def test_p6_detailed_balance_every_reaction_type(rtype):
    """Zero net rate at equilibrium concentrations, whatever [M] and F are (G1, G8)."""
    rx = dict(type=rtype, A0=1e12, b0=-1.5, theta0=2000.0, eff={0: 2.5, 2: 0.7})
    if rtype == FALLOFF_TROE:
        rx["troe"] = (0.6, 100.0, 1500.0, 5000.0)
    # 2A + B <=> AB + C-like: use coefficients > 1 to pin the integer powers too
    sp = _w2_species() + [dict(W=5.0, lo=[3.0, 1e-3, 0, 0, 0, -1000.0, 2.0])]
    r = dict(reac={0: 2, 1: 1}, prod={2: 1, 3: 2}, **W1)
    r.update(rx)
    mech = simple_mechanism(sp, [r])
    o = oracle.Oracle(mech, "f80")
    for T in (800.0, 1500.0, 2500.0):
        C = np.array([2e-3, 3e-3, 1e-3, 1.0], dtype=np.longdouble)
        rho, Y = _state_from_C(mech, C.astype(np.float64))
        Kc = o.reaction_detail(0, rho, T, Y)["Kc"]
        # choose C_3 so that C_AB C_3^2 = Kc C_A^2 C_B
        C[3] = np.sqrt(Kc * C[0] ** 2 * C[1] / C[2])
        od = oracle.Oracle(mech)
        rho, Y = _state_from_C(mech, C.astype(np.float64))
        d = od.reaction_detail(0, rho, T, Y)
        assert d["qf"] > 0 and abs(d["qf"] - d["qr"]) <= 2e-13 * d["qf"]
        if rtype == THREE_BODY:
            assert abs(d["M"] / (2.5 * C[0] + C[1] + 0.7 * C[2] + C[3]) - 1) < 1e-14


def test_p7_kc_forward_times_backward_is_one_and_p0_independence():
    """(A.10; G1): exponent of p0/RT is sum(nu)."""
    sp = _w2_species()
    fwd = simple_mechanism(sp, [dict(reac={0: 1, 1: 1}, prod={2: 1}, **W1)])
    bwd = simple_mechanism(sp, [dict(reac={2: 1}, prod={0: 1, 1: 1}, **W1)])
    Y = [0.3, 0.3, 0.4]
    for T in (500.0, 1500.0, 2900.0):
        k1 = oracle.Oracle(fwd, "f80").reaction_detail(0, 1.0, T, Y)["Kc"]
        k2 = oracle.Oracle(bwd, "f80").reaction_detail(0, 1.0, T, Y)["Kc"]
        assert abs(k1 * k2 - 1) < 1e-15
    # sum(nu) = 0: Kc = exp(-sum nu g/RT), no p0/RT factor
    iso = simple_mechanism(sp[:2], [dict(reac={0: 1}, prod={1: 1}, **W1)])
    o = oracle.Oracle(iso)
    T = 1300.0
    gA, gB = o.species_thermo(0, T)[3], o.species_thermo(1, T)[3]
    assert abs(o.reaction_detail(0, 1.0, T, [0.5, 0.5])["Kc"] / np.exp(-(gB - gA)) - 1) < 1e-14
    # sum(nu) = -1: Kc * (p0/RT) = exp(-sum nu g/RT)
    d = oracle.Oracle(fwd).reaction_detail(0, 1.0, T, Y)
    o3 = oracle.Oracle(fwd)
    dg = o3.species_thermo(2, T)[3] - o3.species_thermo(0, T)[3] - o3.species_thermo(1, T)[3]
    assert abs(d["Kc"] * (P_ATM / (R_UNIVERSAL * T)) / np.exp(-dg) - 1) < 1e-13


# ---------------------------------------------------------------- P8 Newton
@pytest.mark.parametrize("cfg", [0, 2])
def test_p8_newton_recovers_generating_temperature(cfg):
    mech = inputs.config_mechanism(cfg)
    o = oracle.Oracle(mech)
    st = inputs.config_states(cfg, n=512)   # e evaluated by the generator in long double (H9)
    T, it, conv = o.get_temperature(st["e"], st["Y"], st["T_guess"], tol=1e-6, max_iter=10)
    assert conv.all() and it.max() <= 6
    assert np.max(np.abs(T - st["T"]) / st["T"]) < 1e-12


def test_p8_newton_cap_and_nonconvergence_report():
    mech = inputs.config_mechanism(0)
    o = oracle.Oracle(mech)
    st = inputs.config_states(0, n=8)
    T, it, conv = o.get_temperature(st["e"], st["Y"], st["T_guess"], tol=1e-300, max_iter=3)
    assert (it == 3).all() and (conv == 0).all() and np.isfinite(T).all()


# ---------------------------------------------------------------- P9-P11 third body and falloff
def test_p9_unit_efficiencies_give_total_concentration():
    mech = _w2_mech(type=THREE_BODY)
    o = oracle.Oracle(mech)
    T, P = 1100.0, 3 * P_ATM
    Y = np.array([0.2, 0.5, 0.3])
    Wbar = 1.0 / (Y / mech.mol_weight).sum()
    rho = P * Wbar / (R_UNIVERSAL * T)
    assert abs(o.reaction_detail(0, rho, T, Y)["M"] / (P / (R_UNIVERSAL * T)) - 1) < 1e-14


def test_p10_lindemann_limits():
    T = 1200.0
    hi = oracle.Oracle(_w2_mech(type=FALLOFF_LINDEMANN, A0=1e40, b0=0.0, theta0=0.0))
    d = hi.reaction_detail(0, 1.0, T, [0.3, 0.3, 0.4])
    assert d["Pr"] > 1e20 and abs(d["kf"] / d["k_inf"] - 1) < 1e-15
    lo = oracle.Oracle(_w2_mech(type=FALLOFF_LINDEMANN, A0=1e-10, b0=0.0, theta0=0.0))
    d = lo.reaction_detail(0, 1.0, T, [0.3, 0.3, 0.4])
    assert d["Pr"] < 1e-10 and abs(d["kf"] / (d["k0"] * d["M"]) - 1) < 1e-9


def test_p11_troe_reduces_to_lindemann_and_three_vs_four_parameters():
    low = dict(A0=1e12, b0=-1.5, theta0=2000.0)
    T, Y = 1200.0, [0.3, 0.3, 0.4]
    lind = oracle.Oracle(_w2_mech(type=FALLOFF_LINDEMANN, **low)).reaction_detail(0, 1.0, T, Y)
    # alpha = 1, T* = +inf, T** = +inf: Fcent = exp(-T/inf) = 1, so F = 1
    troe1 = oracle.Oracle(_w2_mech(type=FALLOFF_TROE, troe=(1.0, 100.0, np.inf, np.inf), **low)).reaction_detail(0, 1.0, T, Y)
    assert troe1["F"] == 1.0 and troe1["kf"] == lind["kf"]
    # 3- vs 4-parameter forms differ exactly by the exp(-T**/T) term of Fcent (G7):
    # with T** = 5000 the 4-parameter Fcent is larger by exp(-5000/1200)
    p3 = oracle.Oracle(_w2_mech(type=FALLOFF_TROE, troe=(0.6, 100.0, 1500.0, np.inf), **low)).reaction_detail(0, 1.0, T, Y)
    p4 = oracle.Oracle(_w2_mech(type=FALLOFF_TROE, troe=(0.6, 100.0, 1500.0, 5000.0), **low)).reaction_detail(0, 1.0, T, Y)

    def F_of(Fc, Pr):
        lFc = np.log10(Fc)
        c, n = -0.4 - 0.67 * lFc, 0.75 - 1.27 * lFc
        f1 = (np.log10(Pr) + c) / (n - 0.14 * (np.log10(Pr) + c))
        return 10.0 ** (lFc / (1 + f1 * f1))
    Fc3 = 0.4 * np.exp(-T / 100.0) + 0.6 * np.exp(-T / 1500.0)
    assert abs(p3["F"] / F_of(Fc3, p3["Pr"]) - 1) < 1e-13
    assert abs(p4["F"] / F_of(Fc3 + np.exp(-5000.0 / T), p4["Pr"]) - 1) < 1e-13
    assert p3["F"] != p4["F"]


# ---------------------------------------------------------------- P12 scaling, P16 irreversible
def test_p12_scaling_with_density_and_prefactor():
    sp = _w2_species()
    r = dict(reac={0: 2, 1: 1}, prod={2: 1}, **W1)
    mech = simple_mechanism(sp, [r])
    o = oracle.Oracle(mech)
    Y, T = np.array([0.2, 0.5, 0.3]), 1400.0
    d1 = o.reaction_detail(0, 0.7, T, Y)
    d2 = o.reaction_detail(0, 1.4, T, Y)
    assert abs(d2["qf"] / d1["qf"] / 8.0 - 1) < 1e-14      # lambda^(sum nu') = 2^3
    assert abs(d2["qr"] / d1["qr"] / 2.0 - 1) < 1e-14      # lambda^(sum nu'') = 2^1
    r2 = dict(r)
    r2["A"] = 2 * r["A"]
    o2 = oracle.Oracle(simple_mechanism(sp, [r2]))
    om1, _ = o.get_net_production_rates([0.7], [T], Y[:, None])
    om2, _ = o2.get_net_production_rates([0.7], [T], Y[:, None])
    assert np.allclose(om2, 2 * om1, rtol=1e-15, atol=0)
    # stoichiometric signs and magnitudes: omega = nu R
    R = d1["qf"] - d1["qr"]
    assert np.allclose(om1[:, 0], np.array([-2.0, -1.0, 1.0]) * R, rtol=1e-15)


def test_p16_irreversible_flag():
    mech = _w2_mech(reversible=0)
    o = oracle.Oracle(mech)
    rho, Y = _state_from_C(mech, [2e-3, 3e-3, 1e-3])
    d = o.reaction_detail(0, rho, 1500.0, Y)
    assert d["qr"] == 0.0 and d["Kc"] == 0.0
    rho2, Y2 = _state_from_C(mech, [2e-3, 3e-3, 5.0])
    d2 = o.reaction_detail(0, rho2, 1500.0, Y2)
    assert abs(d2["qf"] / d["qf"] - 1) < 1e-14   # products do not enter


# ---------------------------------------------------------------- P14 double vs long double
@pytest.mark.parametrize("cfg", [0, 2])
def test_p14_double_oracle_agrees_with_long_double(cfg):
    mech = inputs.config_mechanism(cfg)
    n = 512 if cfg == 0 else 64
    st = inputs.config_states(cfg, n=n)
    om, bd = oracle.Oracle(mech).get_net_production_rates(st["rho"], st["T"], st["Y"])
    om80, bd80 = oracle.Oracle(mech, "f80").get_net_production_rates(st["rho"], st["T"], st["Y"])
    err = np.abs(om - om80.astype(np.float64))
    assert np.all(err <= 1e-13 * bd)
    T, _, _ = oracle.Oracle(mech).get_temperature(st["e"], st["Y"], st["T_guess"])
    T80, _, _ = oracle.Oracle(mech, "f80").get_temperature(st["e"], st["Y"], st["T_guess"])
    assert np.max(np.abs(T - T80.astype(np.float64)) / T) < 1e-13


# ---------------------------------------------------------------- paper's toy inputs
def test_paper_toy_inputs_forward_rate_closed_form():
    """R_f = k(T) C_m C_n for the toy of listings 10/15: T = linspace(1000, 2100, 10), C = (0.2, 0.8);
    T = 300, C = 0.5; and the gradient structure of eq (3) PAPER.md:315 by finite differences."""
    sp = _w2_species()
    mech = simple_mechanism(sp, [dict(reac={0: 1, 1: 1}, prod={2: 1}, reversible=0, **W1)])
    o = oracle.Oracle(mech, "f80")
    L = np.longdouble
    for T in list(np.linspace(1000, 2100, 10)) + [300.0]:
        Cm, Cn = (0.2, 0.8) if T != 300.0 else (0.5, 0.5)
        rho, Y = _state_from_C(mech, [Cm, Cn, 0.0])
        d = o.reaction_detail(0, rho, T, Y)
        k = L(W1["A"]) * L(T) ** L(W1["b"]) * np.exp(-L(W1["theta"]) / L(T))
        assert abs(d["qf"] / (k * L(Cm) * L(Cn)) - 1) < 1e-15
        # dR/dT = R (b/T + theta/T^2)
        h = L(T) * L(1e-6)
        dp = o.reaction_detail(0, rho, L(T) + h, Y)["qf"]
        dm = o.reaction_detail(0, rho, L(T) - h, Y)["qf"]
        assert abs((dp - dm) / (2 * h) / (d["qf"] * (L(W1["b"]) / L(T) + L(W1["theta"]) / L(T) ** 2)) - 1) < 1e-9


# ---------------------------------------------------------------- N1-N7: SURVEY.md 8(f) NEXT-1 (EOS, enthalpy form)
def test_n1_n2_n3_enthalpy_identities(cfg0):
    """h - e = R T sum_k Y_k/W_k (h_k = e_k + R T/W_k, A.26); c_p = dh/dT; c_p - c_v = R sum_k Y_k/W_k (A.29, G4)."""
    mech, o, o80 = cfg0
    st = inputs.config_states(0, n=16)
    L = np.longdouble
    for p in range(16):
        T, Y = float(st["T"][p]), st["Y"][:, p]
        rw = R_UNIVERSAL * float((Y / mech.mol_weight).sum())
        assert abs((o.mixture_h(T, Y) - o.mixture_e(T, Y)) / (rw * T) - 1) < 1e-11   # h, e are ~1e3 x R T/W here
        assert abs((o.mixture_cp(T, Y) - o.mixture_cv(T, Y)) / rw - 1) < 1e-12
        if abs(T - 1000.0) < 1.0:
            continue
        dT = L(T) * L(1e-5)
        dh = (o80.mixture_h(L(T) + dT, Y) - o80.mixture_h(L(T) - dT, Y)) / (2 * dT)
        assert abs(dh / o80.mixture_cp(L(T), Y) - 1) < 1e-8


def test_n4_newton_on_enthalpy_recovers_temperature_and_closed_form():
    """Enthalpy form of the inversion: constant-c_p species h = (a1 T + a6) R/W gives T in
    one step; on configs[0] the solve recovers the T that generated h."""
    mech1 = simple_mechanism([dict(W=28.014, lo=[3.5, 0, 0, 0, 0, -1000.0, 0.0])], [])
    o1 = oracle.Oracle(mech1)
    h = (3.5 * 1234.5 - 1000.0) * R_UNIVERSAL / 28.014
    assert abs(o1.mixture_h(1234.5, [1.0]) / h - 1) < 1e-15
    assert abs(o1.mixture_cp(1234.5, [1.0]) / (3.5 * R_UNIVERSAL / 28.014) - 1) < 1e-15
    for Tg in (300.0, 1111.0, 2999.0):
        T, it, cv = o1.get_temperature_from_enthalpy([h], np.array([[1.0]]), [Tg])
        assert abs(T[0] / 1234.5 - 1) < 1e-14 and it[0] <= 2 and cv[0] == 1
    mech = inputs.config_mechanism(0)
    o = oracle.Oracle(mech)
    st = inputs.config_states(0, n=256)
    hh = np.array([o.mixture_h(float(st["T"][p]), st["Y"][:, p]) for p in range(256)])
    T, it, conv = o.get_temperature_from_enthalpy(hh, st["Y"], st["T_guess"])
    assert conv.all() and it.max() <= 6
    assert np.max(np.abs(T - st["T"]) / st["T"]) < 1e-12
    # it is a different equation from the energy form: feeding e instead of h lands elsewhere
    T_e, _, _ = o.get_temperature_from_enthalpy(st["e"][:256], st["Y"], st["T_guess"])
    assert np.min(np.abs(T_e - st["T"]) / st["T"]) > 1e-3


def test_n5_n6_n7_equation_of_state():
    """(A.2), (A.3): single species rho = p W/(R T); p(rho(p)) = p; sum_k C_k = p/(R T) with C_k of (A.8)."""
    mech1 = simple_mechanism([dict(W=28.014, lo=[3.5, 0, 0, 0, 0, -1000.0, 0.0])], [])
    o1 = oracle.Oracle(mech1)
    rho = o1.get_density([2 * P_ATM], [750.0], np.array([[1.0]]))
    assert abs(rho[0] / (2 * P_ATM * 28.014 / (R_UNIVERSAL * 750.0)) - 1) < 1e-15
    mech = inputs.config_mechanism(2)
    o = oracle.Oracle(mech)
    st = inputs.config_states(2, n=64)
    p = np.full(64, P_ATM) * np.linspace(0.1, 50.0, 64)
    rho = o.get_density(p, st["T"], st["Y"])
    assert np.max(np.abs(o.get_pressure(rho, st["T"], st["Y"]) / p - 1)) < 1e-14
    C = rho[None, :] * st["Y"] / mech.mol_weight[:, None]
    assert np.max(np.abs(C.sum(axis=0) / (p / (R_UNIVERSAL * st["T"])) - 1)) < 1e-13
    # the generator's own density (ideal gas at 1 atm, H7) is the same function
    assert np.max(np.abs(o.get_density(np.full(64, P_ATM), st["T"], st["Y"]) / st["rho"] - 1)) < 1e-13
