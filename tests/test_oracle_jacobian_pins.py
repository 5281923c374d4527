"""Pins of the oracle's analytic chemical Jacobian (no GPU): SURVEY.md 8(f) NEXT-2.

J = dS/dY, S_i = W_i omega_i   (eq. (6); (A.1) PAPER.md:888; (A.36) PAPER.md:1057).
  J1  finite differences of the oracle's own omega in long double: one-sided differences converge linearly in
      delta as in eq. (7) / fig. 8, central differences agree to 1e-8
  J2  W6: closed forms of the single reaction (dR/dC_A = k C_B) and 50-digit numerical
      derivatives of the three-body / Lindemann / Troe rate (tests/golden/make_w6.py)
  J3  mass and element conservation per column: sum_i J_ik = 0, sum_i n_e,i J_ik / W_i = 0
  J4  the (rho, e) form (reading G26) against differences through the oracle's own temperature inversion
  J5  dS/dT by central differences, every reaction type
"""
import importlib.util
import os

import mpmath as mp
import numpy as np
import pytest

from conftest import read_golden
from hand_cases import all_paths_mechanism, random_states
from oracle import oracle
from paper_2503_24286_b200 import inputs
from paper_2503_24286_b200.inputs import (FALLOFF_LINDEMANN, FALLOFF_TROE, THREE_BODY, simple_mechanism)

W1 = dict(A=35127309770106.477, b=-0.7, theta=8590.0)
LD = np.longdouble


def _fd_jacobian(o, mech, rho, T, Y, delta, central):
    """dS_i/dY_k at fixed (rho, T) from differences of the oracle's omega: Y_k -> Y_k +- delta."""
    ns = mech.n_species
    W = mech.mol_weight.astype(o.dtype)
    J = np.zeros((ns, ns), dtype=o.dtype)
    base = None
    if not central:
        base, _ = o.get_net_production_rates([rho], [T], np.asarray(Y, dtype=o.dtype)[:, None])
    for k in range(ns):
        Yp = np.array(Y, dtype=o.dtype)
        Yp[k] += o.dtype(delta)
        wp, _ = o.get_net_production_rates([rho], [T], Yp[:, None])
        if central:
            Ym = np.array(Y, dtype=o.dtype)
            Ym[k] -= o.dtype(delta)
            wm, _ = o.get_net_production_rates([rho], [T], Ym[:, None])
            J[:, k] = W * (wp[:, 0] - wm[:, 0]) / (2 * o.dtype(delta))
        else:
            J[:, k] = W * (wp[:, 0] - base[:, 0]) / o.dtype(delta)
    return J


def _mechs():
    return [("all_paths", all_paths_mechanism()), ("cfg0", inputs.config_mechanism(0))]


@pytest.mark.parametrize("name,mech", _mechs(), ids=[m[0] for m in _mechs()])
def test_j1_finite_differences_converge_linearly_and_central_agrees(name, mech):
    """Eq. (7): eps(delta) = ||J - J_FD(delta)||_F / ||J||_F falls linearly with delta for
    first-order differences; central differences in long double agree with the analytic Jacobian to 1e-8."""
    o80 = oracle.Oracle(mech, "f80")
    rho, T, Y = random_states(mech, 6, seed=11)
    for p in range(6):
        y = Y[:, p].astype(LD) + LD(1e-3)   # keep every species away from zero so that all terms are exercised
        J, dSdT, bJ, bT = o80.get_jacobian([rho[p]], [T[p]], y[:, None], mode=0)
        J = J[:, :, 0]
        nrm = np.sqrt(float((J * J).sum()))
        eps = []
        for delta in (1e-3, 1e-4, 1e-5):
            Jfd = _fd_jacobian(o80, mech, rho[p], T[p], y, delta, central=False)
            eps.append(np.sqrt(float(((J - Jfd) ** 2).sum())) / nrm)
        assert eps[0] > 0 and 5 < eps[0] / eps[1] < 20, (name, p, eps)
        assert eps[2] < 1e-13 or 5 < eps[1] / eps[2] < 20, (name, p, eps)   # until rounding takes over (fig. 8)
        Jc = _fd_jacobian(o80, mech, rho[p], T[p], y, 1e-5, central=True)
        assert np.sqrt(float(((J - Jc) ** 2).sum())) / nrm < 1e-8
        # element by element against the sum of absolute terms (what the parity tolerance is scaled with), plus
        # the rounding noise of the difference quotient itself: long double rounding of omega_i over 2 delta
        _, bw = o80.get_net_production_rates([rho[p]], [T[p]], y[:, None])
        noise = (LD(1e-18) / LD(1e-5)) * (mech.mol_weight.astype(LD) * bw[:, 0])[:, None]
        assert np.all(np.abs(J - Jc) <= 1e-7 * bJ[:, :, 0] + noise)
        assert np.all(bJ[:, :, 0] >= np.abs(J) * (1 - 1e-12))


def _w6_mech(**rx):
    z = [0.0] * 4
    sp = [dict(W=10.0, lo=[2.5, *z, 25000.0, 0.5]), dict(W=15.0, lo=[2.5, *z, 30000.0, 1.0]),
          dict(W=25.0, lo=[3.5, *z, 45000.0, 4.0])]
    r = dict(reac={0: 1, 1: 1}, prod={2: 1}, **W1)
    r.update(rx)
    return simple_mechanism(sp, [r])


def test_j2_w6_closed_forms_and_high_precision_derivatives(golden_dir):
    """W6: dR/dC_k and dR/dT of A + B (+M) <=> AB for the four reaction types.  J_ik = W_i nu_i (rho/W_k) dR/dC_k
    at fixed (rho, T); dS_i/dT = W_i nu_i dR/dT; (rho, e) form: J_ik - dS_i/dT e_k/c_v (reading G26)."""
    spec = importlib.util.spec_from_file_location("make_w6", os.path.join(golden_dir, "make_w6.py"))
    mk = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mk)
    g = read_golden(os.path.join(golden_dir, "w6_reaction_derivatives.txt"))
    for key, val in mk.compute():   # the fixture is what the equations give (50-digit re-evaluation)
        assert abs(val / mp.mpf(g[key]) - 1) < mp.mpf("1e-18"), key
    for k in ("A", "B", "AB"):      # mp.diff reproduces the closed forms of the elementary case
        assert abs(mp.mpf(g[f"elementary_dR_dC_{k}"]) / mp.mpf(g[f"closed_dR_dC_{k}"]) - 1) < mp.mpf("1e-18")
    g = {k: float(v) for k, v in g.items()}
    C = np.array([g["C_A"], g["C_B"], g["C_AB"]])
    low = dict(A0=1e12, b0=-1.5, theta0=2000.0)
    eff = {0: 2.5, 2: 12.0}
    kinds = dict(elementary=dict(eff=eff), three_body=dict(type=THREE_BODY, eff=eff),
                 lindemann=dict(type=FALLOFF_LINDEMANN, eff=eff, **low),
                 troe=dict(type=FALLOFF_TROE, eff=eff, troe=(0.6, 100.0, 1500.0, 5000.0), **low))
    nu = np.array([-1.0, -1.0, 1.0])
    for kind, rx in kinds.items():
        mech = _w6_mech(**rx)
        W = mech.mol_weight
        rho = float((C * W).sum())
        assert abs(rho / g["rho"] - 1) < 1e-15
        Y = C * W / rho
        dRdC = np.array([g[f"{kind}_dR_dC_A"], g[f"{kind}_dR_dC_B"], g[f"{kind}_dR_dC_AB"]])
        J_ref = (W * nu)[:, None] * (rho / W)[None, :] * dRdC[None, :]
        sT_ref = W * nu * g[f"{kind}_dR_dT"]
        ek = np.array([g["e_A"], g["e_B"], g["e_AB"]])
        Je_ref = J_ref - sT_ref[:, None] * ek[None, :] / g["cv"]
        for real, tol in (("f64", 2e-12), ("f80", 2e-15)):
            o = oracle.Oracle(mech, real)
            om, _ = o.get_net_production_rates([rho], [g["T"]], Y[:, None])
            assert abs(float(om[2, 0]) / g[f"{kind}_R"] - 1) < tol
            J, sT, bJ, bT = o.get_jacobian([rho], [g["T"]], Y[:, None], mode=0)
            assert np.all(np.abs(J[:, :, 0].astype(np.float64) - J_ref) <= tol * np.abs(bJ[:, :, 0].astype(np.float64))), kind
            assert np.all(np.abs(sT[:, 0].astype(np.float64) - sT_ref) <= 50 * tol * np.abs(bT[:, 0].astype(np.float64))), kind
            Je, _, bJe, _ = o.get_jacobian([rho], [g["T"]], Y[:, None], mode=1)
            assert np.all(np.abs(Je[:, :, 0].astype(np.float64) - Je_ref) <= 50 * tol * np.abs(bJe[:, :, 0].astype(np.float64))), kind
            # the bound is not vacuous: it is of the size of the entries' own terms
            assert np.all(bJ[:, :, 0] <= 4 * (np.abs((W * nu)[:, None] * (rho / W)[None, :]) *
                                              (np.abs(dRdC)[None, :] + 2 * abs(g["closed_dR_dC_AB"]) + 2 * g["closed_dR_dC_A"])))


@pytest.mark.parametrize("cfg", [0, 2])
def test_j3_mass_and_element_conservation_per_column(cfg):
    """sum_i J_ik = sum_i W_i d omega_i/dY_k = 0 (mass) and sum_i n_e,i d omega_i/dY_k = 0 (elements) for every
    column k and for dS/dT: every reaction conserves them ((A.5), element-balanced reactions, H2/H4)."""
    mech = inputs.config_mechanism(cfg)
    st = inputs.config_states(cfg, n=8)
    o = oracle.Oracle(mech)
    for mode in (0, 1):
        J, sT, bJ, bT = o.get_jacobian(st["rho"], st["T"], st["Y"], mode=mode)
        assert np.all(np.isfinite(J)) and np.all(np.isfinite(sT))
        assert np.all(np.abs(J.sum(axis=0)) <= 1e-13 * bJ.sum(axis=0) + 1e-300)
        assert np.all(np.abs(sT.sum(axis=0)) <= 1e-13 * bT.sum(axis=0))
        w = J / mech.mol_weight[:, None, None]           # d omega_i / dY_k
        bw = bJ / mech.mol_weight[:, None, None]
        for e in range(mech.n_elements):
            ne = mech.elem_comp[:, e].astype(np.float64)
            assert np.all(np.abs((ne[:, None, None] * w).sum(axis=0)) <= 1e-13 * (ne[:, None, None] * bw).sum(axis=0) + 1e-300)


def test_j4_fixed_energy_form_against_differences_through_the_newton_solve():
    """Reading G26 / listing 23: at fixed (rho, e) the temperature follows Y through the
    inversion (A.25)-(A.28); J_ik = d/dY_k [W_i omega_i(rho, T(e, Y), Y)].  Central differences through the
    oracle's own get_temperature in long double."""
    mech = all_paths_mechanism()
    o = oracle.Oracle(mech, "f80")
    rho, T, Y = random_states(mech, 4, seed=5)
    W = mech.mol_weight.astype(LD)
    for p in range(4):
        y = Y[:, p].astype(LD) + LD(1e-3)
        Tp = LD(T[p])
        e = o.mixture_e(Tp, y)
        J, _, bJ, _ = o.get_jacobian([rho[p]], [Tp], y[:, None], mode=1)

        def S(yy):
            Tn, _, conv = o.get_temperature([e], yy[:, None], [Tp], tol=LD(1e-9), max_iter=50)   # quadratic convergence: the returned iterate is exact to rounding
            assert conv[0] == 1
            w, _ = o.get_net_production_rates([rho[p]], Tn, yy[:, None])
            return W * w[:, 0]

        d = LD(1e-7)   # dT/dY_k ~ e_k/c_v ~ 1e4 K: keeps the temperature excursion at 1e-3 K
        for k in range(mech.n_species):
            yp, ym = y.copy(), y.copy()
            yp[k] += d
            ym[k] -= d
            col = (S(yp) - S(ym)) / (2 * d)
            assert np.all(np.abs(col - J[:, k, 0]) <= 1e-6 * bJ[:, k, 0]), (p, k)


@pytest.mark.parametrize("name,mech", _mechs(), ids=[m[0] for m in _mechs()])
def test_j5_temperature_derivative_by_central_differences(name, mech):
    """dS_i/dT at fixed (rho, Y) = W_i sum_j nu_ij dR_j/dT: Arrhenius (A.9), van't Hoff from (A.10)-(A.13),
    falloff forms (G6).  Points are kept away from T_mid, where the NASA ranges switch (G10)."""
    o = oracle.Oracle(mech, "f80")
    rho, T, Y = random_states(mech, 8, seed=3)
    T = np.where(np.abs(T - 1000.0) < 5.0, T + 20.0, T)
    W = mech.mol_weight.astype(LD)
    for p in range(8):
        y = Y[:, p].astype(LD)
        _, sT, _, bT = o.get_jacobian([rho[p]], [T[p]], y[:, None], mode=0)
        h = LD(T[p]) * LD(1e-6)
        wp, _ = o.get_net_production_rates([rho[p]], [LD(T[p]) + h], y[:, None])
        wm, _ = o.get_net_production_rates([rho[p]], [LD(T[p]) - h], y[:, None])
        fd = W * (wp[:, 0] - wm[:, 0]) / (2 * h)
        assert np.all(np.abs(fd - sT[:, 0]) <= 1e-8 * bT[:, 0]), (name, p)


def test_double_jacobian_agrees_with_long_double():
    """Conditioning of the parity tolerance: the double oracle against the long double one, relative to the
    sums of absolute terms."""
    mech = inputs.config_mechanism(0)
    st = inputs.config_states(0, n=64)
    for mode in (0, 1):
        J, sT, bJ, bT = oracle.Oracle(mech).get_jacobian(st["rho"], st["T"], st["Y"], mode=mode)
        J8, sT8, _, _ = oracle.Oracle(mech, "f80").get_jacobian(st["rho"], st["T"], st["Y"], mode=mode)
        assert np.all(np.abs(J - J8.astype(np.float64)) <= 1e-12 * bJ + 1e-300)
        assert np.all(np.abs(sT - sT8.astype(np.float64)) <= 1e-12 * bT + 1e-300)
