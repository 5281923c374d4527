"""Pins of the oracle's reactor march (no GPU): SURVEY.md 8(f) NEXT-4.

Adiabatic isochoric reactors (A.1) PAPER.md:886-888, rho dY_k/dt = W_k omega_k, marched with classical RK4 at a fixed
step.
  R1  one irreversible reaction A -> B with a constant rate coefficient: dY_A/dt = -k Y_A, and one RK4 step of a
      linear equation is the degree-4 Taylor polynomial of exp(-k dt) exactly -- fixes the stage abscissae and weights
  R2  fourth-order convergence in dt on a real mechanism (long double)
  R3  mass and element conservation
  R4  energy: e(T_final, Y_final) = e, the returned temperature is that of the final state
  R5  an equilibrium composition is a fixed point
"""
import numpy as np
import pytest

from hand_cases import all_paths_mechanism, random_states
from oracle import oracle
from paper_2503_24286_b200 import inputs
from paper_2503_24286_b200.inputs import simple_mechanism

LD = np.longdouble


def test_r1_linear_decay_step_is_the_taylor_polynomial():
    z4 = [0.0] * 4
    sp = [dict(W=20.0, lo=[3.5, *z4, -1000.0, 2.0]), dict(W=20.0, lo=[3.0, *z4, -3000.0, 3.0])]
    k = 2.5e5
    mech = simple_mechanism(sp, [dict(reac={0: 1}, prod={1: 1}, A=k, b=0.0, theta=0.0, reversible=0)])
    for real, tol in (("f64", 1e-14), ("f80", 1e-17)):
        o = oracle.Oracle(mech, real)
        Y0 = np.array([[0.7], [0.3]])
        T0, rho = 1100.0, 0.4
        e = o.mixture_e(T0, Y0[:, 0])
        for dt, steps in ((1e-6, 1), (2e-6, 7), (4e-7, 40)):
            z = LD(k) * LD(dt)
            P = 1 - z + z * z / 2 - z ** 3 / 6 + z ** 4 / 24
            Y, T, Yb, bad = o.reactor_rk4([rho], [e], Y0, [T0], dt, steps)
            yA = LD(Y0[0, 0]) * P ** steps
            yB = LD(Y0[1, 0]) + (LD(Y0[0, 0]) - yA)
            assert bad == 0
            assert abs(LD(Y[0, 0]) - yA) <= tol * steps and abs(LD(Y[1, 0]) - yB) <= tol * steps
            assert abs(float(o.mixture_e(T[0], Y[:, 0])) / float(e) - 1) < 1e-12                      # R4
            assert Yb[0, 0] > 0 and abs(float(Yb[0, 0]) - float(Yb[1, 0])) <= 1e-12 * float(Yb[0, 0])


def stable_dt(o, st, safety=0.05):
    """A step that resolves the fastest chemical time scale of every state in `st`: the largest row sum of the
    Jacobian of dY/dt = S/rho at fixed (rho, e) bounds its spectral radius (the synthetic mechanisms are far
    stiffer than the paper's 10 ns would allow)."""
    J, _, _, _ = o.get_jacobian(st["rho"], st["T"], st["Y"], mode=1)
    rate = np.max(np.abs(J.astype(np.float64)).sum(axis=1) / st["rho"][None, :])
    return safety / float(rate)


def _run(o, st, p, dt, steps):
    Y, T, Yb, bad = o.reactor_rk4(st["rho"][p:p + 1], st["e"][p:p + 1].astype(o.dtype), st["Y"][:, p:p + 1],
                                  st["T"][p:p + 1], dt, steps, tol=o.dtype(1e-9), max_iter=30)
    assert bad == 0
    return Y[:, 0], T[0]


def test_r2_fourth_order_convergence():
    """Error against a 16-times finer march falls by 2^4 when dt is halved (long double, configs[0] mechanism)."""
    mech = inputs.config_mechanism(0)
    o = oracle.Oracle(mech, "f80")
    st = inputs.config_states(0, n=64)
    st["e"] = np.array([o.mixture_e(LD(st["T"][p]), st["Y"][:, p].astype(LD)) for p in range(64)], dtype=LD)
    checked = 0
    for p in range(64):
        if not 1200.0 < st["T"][p] < 2500.0:
            continue
        # a step that resolves the fastest time scale of this state: the largest row sum of the Jacobian of
        # dY/dt = S/rho at fixed (rho, e) bounds its spectral radius
        J, _, _, _ = o.get_jacobian(st["rho"][p:p + 1], st["T"][p:p + 1], st["Y"][:, p:p + 1], mode=1)
        rate = float(np.max(np.abs(J[:, :, 0].astype(np.float64)).sum(axis=1)) / st["rho"][p])
        dt = 0.05 / rate
        t_end = 8 * dt
        ref, _ = _run(o, st, p, dt / 16, 128)
        e1 = np.max(np.abs(_run(o, st, p, dt, 8)[0] - ref))
        e2 = np.max(np.abs(_run(o, st, p, dt / 2, 16)[0] - ref))
        if e2 < 1e-17:      # already at rounding level
            continue
        assert 9.0 < float(e1 / e2) < 25.0, (p, float(e1), float(e2), t_end)
        checked += 1
    assert checked >= 5


@pytest.mark.parametrize("cfg", [0, 2])
def test_r3_r4_conservation_of_mass_elements_and_energy(cfg):
    mech = inputs.config_mechanism(cfg)
    o = oracle.Oracle(mech)
    st = inputs.config_states(cfg, n=16)
    dt = stable_dt(o, st)
    Y, T, Yb, bad = o.reactor_rk4(st["rho"], st["e"], st["Y"], st["T_guess"], dt, 20)
    assert bad == 0 and np.all(np.isfinite(Y)) and np.all(np.isfinite(T))
    assert np.any(np.abs(Y - st["Y"]) > 1e-3 * np.abs(st["Y"]))      # something happened
    scale = Yb.sum(axis=0) + 1.0
    assert np.all(np.abs(Y.sum(axis=0) - st["Y"].sum(axis=0)) <= 1e-13 * scale)
    for el in range(mech.n_elements):
        w = mech.elem_comp[:, el] / mech.mol_weight
        assert np.all(np.abs((w[:, None] * (Y - st["Y"])).sum(axis=0)) <= 1e-13 * (w[:, None] * (Yb + np.abs(Y))).sum(axis=0))
    for p in range(16):
        assert abs(o.mixture_e(T[p], Y[:, p]) / st["e"][p] - 1) < 1e-11


def test_r5_equilibrium_composition_is_a_fixed_point():
    z4 = [0.0] * 4
    sp = [dict(W=10.0, lo=[2.5, *z4, 25000.0, 0.5]), dict(W=15.0, lo=[2.5, *z4, 30000.0, 1.0]),
          dict(W=25.0, lo=[3.5, *z4, 45000.0, 4.0])]
    mech = simple_mechanism(sp, [dict(reac={0: 1, 1: 1}, prod={2: 1}, A=35127309770106.477, b=-0.7, theta=8590.0)])
    o = oracle.Oracle(mech, "f80")
    T0 = LD(1350.0)
    CA, CB = LD(0.004), LD(0.005)
    Y_probe = np.array([0.3, 0.3, 0.4], dtype=LD)
    Kc = o.reaction_detail(0, 1.0, T0, Y_probe)["Kc"]
    C = np.array([CA, CB, Kc * CA * CB], dtype=LD)
    W = mech.mol_weight.astype(LD)
    rho = (C * W).sum()
    Y0 = (C * W / rho)[:, None]
    e = o.mixture_e(T0, Y0[:, 0])
    Y, T, Yb, bad = o.reactor_rk4([rho], [e], Y0, [T0], 1e-9, 50)
    assert bad == 0
    assert np.all(np.abs(Y - Y0) <= 1e-15 * (Yb + 1.0)) and abs(T[0] - T0) < 1e-9
    # and away from equilibrium it moves
    Y1 = Y0.copy()
    Y1[0, 0] *= 1.2
    Y2, _, _, _ = o.reactor_rk4([rho], [e], Y1, [T0], 1e-9, 50)
    assert abs(Y2[0, 0] - Y1[0, 0]) > 1e-9


def test_double_reactor_agrees_with_long_double():
    mech = all_paths_mechanism()
    rho, T, Y = random_states(mech, 32, seed=2)
    o, o8 = oracle.Oracle(mech), oracle.Oracle(mech, "f80")
    e = np.array([o.mixture_e(T[p], Y[:, p]) for p in range(32)])
    dt = stable_dt(o, dict(rho=rho, T=T, Y=Y))
    a = o.reactor_rk4(rho, e, Y, T, dt, 10)
    b = o8.reactor_rk4(rho, e, Y, T, dt, 10)
    assert np.isfinite(a[0]).all() and a[3] == 0
    assert np.all(np.abs(a[0] - b[0].astype(np.float64)) <= 1e-12 * (a[2] + np.abs(a[0])))


# ---------------------------------------------------------------- Crank-Nicolson march (A.32)-(A.36) PAPER.md:1043-1062
def _decay_mech(k):
    z4 = [0.0] * 4
    sp = [dict(W=20.0, lo=[3.5, *z4, -1000.0, 2.0]), dict(W=20.0, lo=[3.0, *z4, -3000.0, 3.0])]
    return simple_mechanism(sp, [dict(reac={0: 1}, prod={1: 1}, A=k, b=0.0, theta=0.0, reversible=0)])


def test_c1_linear_decay_step_and_c4_stability_where_rk4_diverges():
    """dY_A/dt = -k Y_A: one Crank-Nicolson step is y (1 - z/2)/(1 + z/2), z = k dt, reached by ONE Newton iteration
    (the problem is linear and the Jacobian exact).  At z = 20 RK4 grows by |P(z)| = 5e3 per step, CN stays bounded
    (the implicit scheme allows larger steps)."""
    k = 2.5e5
    mech = _decay_mech(k)
    for real, tol in (("f64", 1e-14), ("f80", 1e-17)):
        o = oracle.Oracle(mech, real)
        Y0 = np.array([[0.7], [0.3]])
        T0, rho = 1100.0, 0.4
        e = o.mixture_e(T0, Y0[:, 0])
        for dt, steps, iters in ((1e-6, 1, 1), (2e-6, 7, 1), (4e-7, 40, 3), (8e-5, 5, 2)):
            z = LD(k) * LD(dt)
            g = (1 - z / 2) / (1 + z / 2)
            Y, T, Yb, lu, bad = o.reactor_cn([rho], [e], Y0, [T0], dt, steps, newton_iters=iters)
            yA = LD(Y0[0, 0]) * g ** steps
            assert bad == 0
            assert abs(LD(Y[0, 0]) - yA) <= tol * steps * 4 and abs(LD(Y[1, 0]) - (LD(Y0[1, 0]) + LD(Y0[0, 0]) - yA)) <= tol * steps * 4
            if iters > 1:
                assert float(lu[0]) <= 1e-15          # the second Newton update of a linear problem is rounding
            assert abs(float(o.mixture_e(T[0], Y[:, 0])) / float(e) - 1) < 1e-12
    # z = 20: RK4 diverges, CN does not
    o = oracle.Oracle(mech)
    Yr, _, _, _ = o.reactor_rk4([rho], [e], Y0, [T0], 8e-5, 5)
    Yc, _, _, _, _ = o.reactor_cn([rho], [e], Y0, [T0], 8e-5, 5, newton_iters=1)
    assert abs(Yr[0, 0]) > 1e10 and abs(Yc[0, 0]) <= 0.7


def test_c2_second_order_convergence_and_c3_conservation():
    mech = inputs.config_mechanism(0)
    o = oracle.Oracle(mech, "f80")
    st = inputs.config_states(0, n=64)
    st["e"] = np.array([o.mixture_e(LD(st["T"][p]), st["Y"][:, p].astype(LD)) for p in range(64)], dtype=LD)
    checked = 0
    for p in range(64):
        if not 1200.0 < st["T"][p] < 2500.0:
            continue
        s1 = {k: v[..., p:p + 1] for k, v in st.items() if k in ("rho", "T", "Y", "e")}
        dt = stable_dt(o, s1, safety=0.2)
        ref, _ = _run(o, st, p, dt / 16, 128)                         # RK4, 16 times finer
        run = lambda h, n: o.reactor_cn(s1["rho"], s1["e"], s1["Y"], s1["T"], h, n, newton_iters=6, tol=LD(1e-9), max_iter=30)
        Y1, _, Yb, lu1, bad1 = run(dt, 8)
        Y2, _, _, lu2, bad2 = run(dt / 2, 16)
        assert bad1 == bad2 == 0 and float(lu1[0]) < 1e-12 and float(lu2[0]) < 1e-12   # Newton converged
        e1, e2 = np.max(np.abs(Y1[:, 0] - ref)), np.max(np.abs(Y2[:, 0] - ref))
        if e2 < 1e-16:
            continue
        assert 3.0 < float(e1 / e2) < 5.5, (p, float(e1), float(e2))
        # C3: linear invariants are kept by every Newton update
        assert abs(float(Y1[:, 0].sum() - s1["Y"][:, 0].astype(LD).sum())) <= 1e-16 * float(Yb[:, 0].sum() + 1)
        for el in range(mech.n_elements):
            w = (mech.elem_comp[:, el] / mech.mol_weight).astype(LD)
            assert abs(float((w * (Y1[:, 0] - s1["Y"][:, 0].astype(LD))).sum())) <= 1e-16 * float((w * (Yb[:, 0] + 1)).sum())
        checked += 1
    assert checked >= 5
