"""Hand-written mechanisms that exercise every packer path (inputs only, no arithmetic)."""
import numpy as np

from paper_2503_24286_b200.inputs import (ELEMENTARY, FALLOFF_LINDEMANN, FALLOFF_TROE, THREE_BODY,
                                          simple_mechanism)

W1 = dict(A=35127309770106.477, b=-0.7, theta=8590.0)


def species5():
    """Five species with smooth two-range NASA sets (continuous at 1000 K by construction)."""
    sp = []
    base = [
        (2.0, [2.5, 1.0e-4, 0.0, 0.0, 0.0, 25000.0, 0.5]),
        (16.0, [3.0, 5.0e-4, -1.0e-7, 0.0, 0.0, 30000.0, 1.0]),
        (18.0, [3.5, 1.0e-3, 2.0e-7, -1.0e-11, 0.0, -5000.0, 4.0]),
        (34.0, [4.0, 2.0e-3, -3.0e-7, 2.0e-11, -1.0e-15, -12000.0, 3.0]),
        (28.0, [3.5, 2.0e-4, 0.0, 0.0, 0.0, -1000.0, 2.5]),
    ]
    for W, lo in base:
        hi = list(lo)
        hi[2] = lo[2] * 0.5
        # keep cp, h, s continuous at 1000 K: adjust a2 (cp), a6 (h), a7 (s)
        Tm = 1000.0
        hi[1] = lo[1] + (lo[2] - hi[2]) * Tm
        hi[0] = lo[0] + (lo[1] - hi[1]) * Tm + (lo[2] - hi[2]) * Tm**2
        hi[5] = lo[5] + sum((lo[m] - hi[m]) * Tm ** (m + 1) / (m + 1) for m in range(5))
        hi[6] = lo[6] + (lo[0] - hi[0]) * np.log(Tm) + sum((lo[m] - hi[m]) * Tm**m / m for m in range(1, 5))
        sp.append(dict(W=W, lo=lo, hi=hi))
    return sp


def all_paths_mechanism():
    """Every reaction class of the packer in one mechanism:
    plain reversible/irreversible with 1-3 molecules per side and coefficients 2 and 3,
    three-body, Lindemann, Troe with 3 and 4 parameters, non-unit default efficiency,
    and a species on both sides (net coefficient zero)."""
    low = dict(A0=1e12, b0=-1.5, theta0=2000.0)
    rx = [
        dict(reac={0: 1, 1: 1}, prod={2: 1}, **W1),
        dict(reac={0: 2}, prod={4: 1}, A=3e8, b=0.5, theta=1200.0),
        dict(reac={3: 1}, prod={1: 2, 0: 1}, A=5e10, b=0.0, theta=15000.0),
        dict(reac={0: 3}, prod={2: 1, 4: 1}, A=2e9, b=-1.0, theta=500.0),
        dict(reac={2: 1, 1: 1}, prod={3: 1}, A=4e7, b=1.2, theta=-300.0, reversible=0),
        dict(reac={0: 1, 1: 1}, prod={2: 1}, type=THREE_BODY, eff={0: 2.5, 2: 12.0, 4: 0.3}, eff_order=[2, 4, 0],
             A=1e10, b=-1.0, theta=0.0),   # efficiencies listed out of order
        dict(reac={1: 2}, prod={3: 1}, type=THREE_BODY, eff_default=0.5, eff={4: 1.5}, A=6e9, b=0.0, theta=100.0,
             reversible=0),
        dict(reac={2: 1}, prod={0: 1, 1: 1}, type=FALLOFF_LINDEMANN, eff={3: 6.0}, A=1e13, b=0.0, theta=20000.0,
             A0=1e14, b0=-0.5, theta0=18000.0),
        dict(reac={0: 1, 1: 1}, prod={2: 1}, type=FALLOFF_TROE, troe=(0.6, 100.0, 1500.0, 5000.0), eff={0: 2.0},
             **W1, **low),
        dict(reac={4: 1, 0: 1}, prod={3: 1}, type=FALLOFF_TROE, troe=(0.3, 250.0, 2500.0, np.inf), A=2e10, b=0.3,
             theta=900.0, **low),
        dict(reac={0: 1, 1: 1, 4: 1}, prod={2: 1, 4: 1}, A=7e11, b=-0.8, theta=0.0),   # species 4 on both sides
    ]
    return simple_mechanism(species5(), rx)


def random_states(mech, n, seed=7):
    rng = np.random.default_rng(seed)
    T = rng.uniform(300.0, 3000.0, size=n)
    T[:3] = [1000.0, np.nextafter(1000.0, 0.0), np.nextafter(1000.0, 2000.0)]   # the branch point (G10)
    Y = rng.dirichlet(np.full(mech.n_species, 0.7), size=n).T.copy()
    rho = rng.uniform(0.05, 5.0, size=n)
    return rho, T, Y


def degenerate_mechanisms():
    """Degenerate cases the packer and the kernels must take: no reaction at all (omega = 0), a single
    species, and a mechanism whose reactions are all in the extended class (nothing in the plain loops)."""
    sp = species5()
    none = simple_mechanism(sp, [])
    one = simple_mechanism(sp[:1], [])
    low = dict(A0=1e12, b0=-1.5, theta0=2000.0)
    ext = simple_mechanism(sp, [
        dict(reac={0: 2}, prod={1: 1, 2: 1}, A=3e9, b=0.5, theta=4000.0),                      # repeated species
        dict(reac={1: 1, 3: 1}, prod={4: 1}, A=5e8, b=0.0, theta=1500.0, reversible=0),         # irreversible
        dict(reac={2: 1, 3: 1}, prod={0: 1, 4: 1}, A=2e10, b=-0.3, theta=6000.0, type=1, eff={0: 2.5, 4: 0.4}),
        dict(reac={0: 1, 1: 1}, prod={2: 1}, A=4e9, b=0.2, theta=900.0, type=3, troe=(0.6, 100.0, 1500.0, 5000.0),
             eff={3: 6.0}, **low),
    ])
    return dict(none=none, one=one, ext=ext)


def fuzz_mechanisms():
    """Seeded synthetic mechanisms of other shapes than the configs: reaction counts that leave ragged
    lockstep groups, many / few special reactions, both sides of the 64-reaction packing switch."""
    from paper_2503_24286_b200 import inputs
    specs = [("h2", 13, 2, (1, 5), 2, 1, 11), ("h2", 40, 6, (2, 7), 3, 2, 12), ("gri", 63, 9, (4, 9), 5, 4, 13),
             ("gri", 65, 0, (1, 1), 0, 0, 14), ("gri", 150, 40, (5, 12), 30, 10, 15), ("large", 90, 10, (6, 8), 7, 3, 16)]
    return [inputs.make_mechanism(k, nr, ntb, ne, nt, nl, seed=sd, name=f"fuzz{sd}") for k, nr, ntb, ne, nt, nl, sd in specs]


def extreme_thermo_mechanisms(a6):
    """Species whose a6 (formation enthalpy / R) is `a6` for every species: |g/RT| ~ |a6|/T is far beyond what a
    product of per-species factors exp(g/RT) can hold in FP64, while the Gibbs-energy DIFFERENCES that the
    equilibrium constants see are small or moderate.
      "balanced":  A + B <=> C + D in all four reaction types (sum nu = 0: the common a6 cancels in K_c)
      "assoc":     A + B <=> AB, A + AB <=> B + A2-like ... (sum nu != 0: K_c keeps one a6/T)"""
    def sp(W, a1, a7, dh=0.0):
        lo = [a1, 4.0e-4, -5.0e-8, 0.0, 0.0, a6 + dh, a7]
        return dict(W=W, lo=lo)   # one range
    low = dict(A0=1e12, b0=-1.5, theta0=2000.0)
    four = [sp(10.0, 3.5, 2.0), sp(12.0, 3.0, 4.0, 800.0), sp(9.0, 3.2, 3.0, -600.0), sp(13.0, 3.3, 2.5, 300.0)]
    balanced = simple_mechanism(four, [
        dict(reac={0: 1, 1: 1}, prod={2: 1, 3: 1}, A=3e9, b=0.3, theta=2500.0),
        dict(reac={0: 1, 1: 1}, prod={2: 1, 3: 1}, type=THREE_BODY, eff={0: 2.0, 3: 5.0}, A=1e10, b=-0.5, theta=500.0),
        dict(reac={2: 1, 3: 1}, prod={0: 1, 1: 1}, type=FALLOFF_TROE, troe=(0.6, 100.0, 1500.0, 5000.0), eff={1: 3.0},
             A=2e10, b=0.0, theta=1500.0, **low),
        dict(reac={0: 1, 1: 1}, prod={2: 1, 3: 1}, A=4e8, b=0.0, theta=1000.0, reversible=0),
    ], name=f"balanced{a6:g}")
    three = [sp(10.0, 3.5, 2.0), sp(12.0, 3.0, 4.0, 800.0), sp(22.0, 4.2, 5.0, -900.0)]
    assoc = simple_mechanism(three, [
        dict(reac={0: 1, 1: 1}, prod={2: 1}, A=3e9, b=0.3, theta=2500.0),
        dict(reac={2: 1}, prod={0: 1, 1: 1}, type=FALLOFF_LINDEMANN, eff={0: 2.0}, A=1e13, b=0.0, theta=20000.0,
             A0=1e14, b0=-0.5, theta0=18000.0),
    ], name=f"assoc{a6:g}")
    return dict(balanced=balanced, assoc=assoc)


def troe_sentinel_mechanism():
    """Troe parameter sets with the sentinel temperatures real mechanism files carry (T*** = 1e-30, T* = 1e30,
    T** = 1e30): the exponents -T/T***, -T**/T are astronomically large, the terms themselves exactly 0 or 1."""
    low = dict(A0=1e12, b0=-1.5, theta0=2000.0)
    return simple_mechanism(species5(), [
        dict(reac={0: 1, 1: 1}, prod={2: 1}, type=FALLOFF_TROE, troe=(0.7, 1e-30, 1e30, np.inf), **W1, **low),
        dict(reac={4: 1, 0: 1}, prod={3: 1}, type=FALLOFF_TROE, troe=(0.5, 120.0, 1800.0, 1e30), A=2e10, b=0.3, theta=900.0, **low),
        dict(reac={1: 2}, prod={3: 1}, type=FALLOFF_TROE, troe=(0.4, 1e-8, 900.0, 1e30), A=6e9, b=0.0, theta=100.0, **low),
        dict(reac={2: 1}, prod={0: 1, 1: 1}, type=FALLOFF_TROE, troe=(0.62, 1e-30, 1e30, 4000.0), A=1e13, b=0.0,
             theta=20000.0, A0=1e14, b0=-0.5, theta0=18000.0),
    ], name="troe_sentinels")
