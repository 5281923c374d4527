"""Seeded synthetic mechanisms and states (the only module shared by oracle and CUDA path).

This module draws *inputs*: species tables, reaction tables and thermodynamic
states shaped like the workloads of BASELINE.json `configs[0..4]` (rules H0-H9
of SURVEY.md section 8(d), restated in DESIGN.md "Input recipe").  It holds no
part of the method that is being tested: nothing here computes a rate, a
production rate or a Newton iterate.  The few closed-form evaluations it needs
to make inputs *valid* (c_p range check of a drawn NASA-7 set, |ln K_c| guard
that keeps (A.10) finite, ideal-gas density, and the internal energy that is
handed to the temperature solve) are written out locally in numpy and are used
by neither the oracle nor the CUDA library.

The paper measures on the San Diego H2-air mechanism, a 10-species H2 subset
of GRI-3.0 and verifies on GRI-3.0.  Those
files are not available; these synthetic mechanisms take their shapes only.

Units: SI with kmol (W kg/kmol, C kmol/m^3, R = 8314.46261815324 J/(kmol K)).
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

import numpy as np

R_UNIVERSAL = 8314.46261815324  # J/(kmol K)
P_ATM = 101325.0  # Pa
T_MID = 1000.0

ATOMIC_WEIGHT = {"H": 1.008, "C": 12.011, "N": 14.007, "O": 15.999, "Ar": 39.948}

# reaction types (same numbering as include/pyro.h; plain data, not arithmetic)
ELEMENTARY, THREE_BODY, FALLOFF_LINDEMANN, FALLOFF_TROE = 0, 1, 2, 3


@dataclass
class Mechanism:
    """Flat host description of a mechanism (numpy arrays, C-contiguous)."""

    elements: list
    elem_comp: np.ndarray  # [n_species][n_elements] int32
    mol_weight: np.ndarray  # [n_species]
    nasa_lo: np.ndarray  # [n_species][7]
    nasa_hi: np.ndarray  # [n_species][7]
    t_mid: np.ndarray  # [n_species]
    reac_ptr: np.ndarray
    reac_species: np.ndarray
    reac_coeff: np.ndarray
    prod_ptr: np.ndarray
    prod_species: np.ndarray
    prod_coeff: np.ndarray
    A: np.ndarray
    b: np.ndarray
    theta: np.ndarray
    rtype: np.ndarray  # uint8
    reversible: np.ndarray  # uint8
    eff_default: np.ndarray
    eff_ptr: np.ndarray
    eff_species: np.ndarray
    eff_value: np.ndarray
    A0: np.ndarray
    b0: np.ndarray
    theta0: np.ndarray
    troe: np.ndarray  # [n_reactions][4] alpha, T***, T*, T**
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def n_species(self) -> int:
        return int(self.mol_weight.shape[0])

    @property
    def n_reactions(self) -> int:
        return int(self.A.shape[0])

    @property
    def n_elements(self) -> int:
        return int(self.elem_comp.shape[1])

    def nu_dense(self):
        """Dense (nu', nu'') as int arrays [n_species][n_reactions] (for brute-force tests)."""
        ns, nr = self.n_species, self.n_reactions
        nup = np.zeros((ns, nr), dtype=np.int64)
        nupp = np.zeros((ns, nr), dtype=np.int64)
        for j in range(nr):
            for q in range(self.reac_ptr[j], self.reac_ptr[j + 1]):
                nup[self.reac_species[q], j] += self.reac_coeff[q]
            for q in range(self.prod_ptr[j], self.prod_ptr[j + 1]):
                nupp[self.prod_species[q], j] += self.prod_coeff[q]
        return nup, nupp


# --------------------------------------------------------------------------
# helpers that only serve input validity
# --------------------------------------------------------------------------
def _cp_R(a, T):
    return a[0] + T * (a[1] + T * (a[2] + T * (a[3] + T * a[4])))


def _g_RT(a, T):
    h = a[0] + a[1] / 2 * T + a[2] / 3 * T**2 + a[3] / 4 * T**3 + a[4] / 5 * T**4 + a[5] / T
    s = a[0] * np.log(T) + a[1] * T + a[2] / 2 * T**2 + a[3] / 3 * T**3 + a[4] / 4 * T**4 + a[6]
    return h - s


def _draw_nasa(rng):
    """Rule H1: low range from the config-0 distributions, high range matched in value
    and first derivative of c_p at T_mid (h and s continuous), both redrawn until
    1.5 <= c_p/R <= 60 on their validity range."""
    Tlo = np.linspace(200.0, T_MID, 33)
    Thi = np.linspace(T_MID, 3600.0, 53)
    while True:
        lo = np.array(
            [
                rng.uniform(2.5, 4.5),
                rng.uniform(-5e-3, 5e-3),
                rng.uniform(-1e-5, 1e-5),
                rng.uniform(-1e-8, 1e-8),
                rng.uniform(-1e-12, 1e-12),
                rng.uniform(-5e4, 5e4),
                rng.uniform(-10.0, 10.0),
            ]
        )
        c = _cp_R(lo, Tlo)
        if c.min() >= 1.5 and c.max() <= 60.0:
            break
    Tm = T_MID
    for _ in range(10000):
        hi = np.zeros(7)
        hi[2] = rng.uniform(-1e-6, 1e-6)
        hi[3] = rng.uniform(-3e-10, 3e-10)
        hi[4] = rng.uniform(-3e-14, 3e-14)
        # d(cp/R)/dT equal at T_mid -> a2'; cp/R equal -> a1'
        dlo = lo[1] + 2 * lo[2] * Tm + 3 * lo[3] * Tm**2 + 4 * lo[4] * Tm**3
        hi[1] = dlo - (2 * hi[2] * Tm + 3 * hi[3] * Tm**2 + 4 * hi[4] * Tm**3)
        hi[0] = _cp_R(lo, Tm) - (hi[1] * Tm + hi[2] * Tm**2 + hi[3] * Tm**3 + hi[4] * Tm**4)
        # h continuous: a6' ; s continuous: a7'
        hi[5] = lo[5] + sum((lo[m] - hi[m]) * Tm ** (m + 1) / (m + 1) for m in range(5))
        hi[6] = lo[6] + (lo[0] - hi[0]) * np.log(Tm) + sum(
            (lo[m] - hi[m]) * Tm**m / m for m in range(1, 5)
        )
        c = _cp_R(hi, Thi)
        if c.min() >= 1.5 and c.max() <= 60.0:
            return lo, hi
    return _draw_nasa(rng)


def _species_compositions(cfg_kind, rng):
    """Rule H2: distinct small-integer element compositions; returns (elements, comp, diluent, inert)."""
    if cfg_kind == "h2":
        elements = ["H", "O", "N"]
        comp = [(h, o, 0) for h in range(3) for o in range(3) if (h, o) != (0, 0)]
        comp.append((0, 0, 2))
        return elements, np.array(comp, dtype=np.int32), len(comp) - 1, []
    if cfg_kind == "gri":
        elements = ["C", "H", "O", "N", "Ar"]
        comp = [(0, 0, 0, 0, 1), (0, 0, 0, 2, 0)]
        caps = (3, 6, 3, 1)
        n_total = 53
    elif cfg_kind == "large":
        elements = ["C", "H", "O", "N"]
        comp = [(0, 0, 0, 2)]
        caps = (8, 18, 4, 2)
        n_total = 120
    else:
        raise ValueError(cfg_kind)
    seen = set(comp)
    ne = len(elements)
    while len(comp) < n_total:
        v = tuple(int(rng.integers(0, c + 1)) for c in caps) + (0,) * (ne - 4)
        if sum(v) == 0 or v in seen:
            continue
        seen.add(v)
        comp.append(v)
    comp = np.array(comp, dtype=np.int32)
    if cfg_kind == "gri":
        return elements, comp, 1, [0]
    return elements, comp, 0, []


def _multisets(n_species, comp, size):
    """All multisets of `size` species with their element totals."""
    idx = np.array(list(itertools.combinations_with_replacement(range(n_species), size)), dtype=np.int32)
    totals = comp[idx].sum(axis=1)
    return idx, totals


def make_mechanism(
    kind,
    n_reactions,
    n_three_body,
    n_eff,
    n_troe,
    n_lindemann,
    seed,
    name="",
):
    """Rules H1-H6.  `kind` in {"h2", "gri", "large"}; `n_eff` = (min, max) listed efficiencies."""
    rng = np.random.default_rng(seed)
    elements, comp, diluent, inert = _species_compositions(kind, rng)
    ns, ne = comp.shape
    aw = np.array([ATOMIC_WEIGHT[e] for e in elements])
    W = comp @ aw

    nasa_lo = np.zeros((ns, 7))
    nasa_hi = np.zeros((ns, 7))
    for k in range(ns):
        nasa_lo[k], nasa_hi[k] = _draw_nasa(rng)
    t_mid = np.full(ns, T_MID)

    # ---- reactions (H4): element-balanced pairs of disjoint multisets of 1-3 species
    by_size = {}
    for size in (1, 2, 3):
        idx, tot = _multisets(ns, comp, size)
        # positional hash of the element totals
        key = np.zeros(len(idx), dtype=np.int64)
        for e in range(ne):
            key = key * 64 + tot[:, e]
        order = np.argsort(key, kind="stable")
        by_size[size] = (idx[order], key[order])
    Tchk = np.array([250.0, 300.0, 400.0, 600.0, 800.0, 999.0, 1001.0, 1500.0, 2000.0, 2500.0, 3000.0, 3600.0])
    gtab = np.zeros((ns, len(Tchk)))
    for k in range(ns):
        for i, T in enumerate(Tchk):
            gtab[k, i] = _g_RT(nasa_lo[k] if T < T_MID else nasa_hi[k], T)
    ln_c0 = np.log(P_ATM / (R_UNIVERSAL * Tchk))

    reactions = []
    seen = set()
    size_p = np.array([0.2, 0.6, 0.2])
    guard = 0
    while len(reactions) < n_reactions:
        guard += 1
        if guard > 2_000_000:
            raise RuntimeError("reaction search did not terminate")
        nr_, np_ = (int(rng.choice(3, p=size_p)) + 1 for _ in range(2))
        ridx, rkey = by_size[nr_]
        pidx, pkey = by_size[np_]
        i = int(rng.integers(0, len(ridx)))
        lo = int(np.searchsorted(pkey, rkey[i], side="left"))
        hi = int(np.searchsorted(pkey, rkey[i], side="right"))
        if hi <= lo:
            continue
        j = int(rng.integers(lo, hi))
        reac = tuple(int(x) for x in ridx[i])
        prod = tuple(int(x) for x in pidx[j])
        if set(reac) & set(prod):
            continue
        if (reac, prod) in seen or (prod, reac) in seen:
            continue
        # G21 guard: |ln Kc| <= 600 over the whole temperature range used
        dnu = len(prod) - len(reac)
        ln_kc = dnu * ln_c0 - (gtab[list(prod)].sum(axis=0) - gtab[list(reac)].sum(axis=0))
        if np.abs(ln_kc).max() > 600.0:
            continue
        seen.add((reac, prod))
        reactions.append((reac, prod))

    nr = n_reactions
    sum_nu = np.array([len(p) - len(r) for r, p in reactions])
    rtype = np.zeros(nr, dtype=np.uint8)
    # falloff (H6): among reactions with sum(nu) != 0 when available
    n_fall = n_troe + n_lindemann
    cand = [j for j in range(nr) if sum_nu[j] != 0]
    if len(cand) < n_fall:
        cand = cand + [j for j in range(nr) if sum_nu[j] == 0]
    fall = rng.choice(np.array(cand), size=n_fall, replace=False) if n_fall else np.array([], dtype=int)
    for q, j in enumerate(fall):
        rtype[j] = FALLOFF_TROE if q < n_troe else FALLOFF_LINDEMANN
    rest = np.array([j for j in range(nr) if rtype[j] == ELEMENTARY])
    tb = rng.choice(rest, size=n_three_body, replace=False) if n_three_body else np.array([], dtype=int)
    rtype[tb] = THREE_BODY

    # Arrhenius (H3): A cgs log-uniform, converted once to SI-kmol
    A_cgs = 10.0 ** rng.uniform(6.0, 14.0, size=nr)
    b = rng.uniform(-2.0, 3.0, size=nr)
    theta = rng.uniform(0.0, 3.0e4, size=nr)
    order = np.array([len(r) for r, _ in reactions]) + (rtype == THREE_BODY)
    A = A_cgs * 10.0 ** (-3.0 * (order - 1))

    A0 = np.ones(nr)
    b0 = np.zeros(nr)
    theta0 = np.zeros(nr)
    troe = np.zeros((nr, 4))
    troe[:, 0] = 1.0
    troe[:, 1:] = np.inf
    for j in range(nr):
        if rtype[j] >= FALLOFF_LINDEMANN:
            A0[j] = A[j] * 10.0 ** rng.uniform(0.0, 4.0)
            b0[j] = b[j] + rng.uniform(-1.0, 1.0)
            theta0[j] = theta[j] * rng.uniform(0.5, 1.5)
        if rtype[j] == FALLOFF_TROE:
            troe[j] = [
                rng.uniform(0.1, 0.9),
                rng.uniform(50.0, 300.0),
                rng.uniform(500.0, 3000.0),
                rng.uniform(2000.0, 8000.0),
            ]

    # efficiencies (H5, G9): three-body and falloff reactions list non-default species
    eff_ptr = [0]
    eff_species = []
    eff_value = []
    for j in range(nr):
        if rtype[j] != ELEMENTARY:
            n_list = int(rng.integers(n_eff[0], n_eff[1] + 1))
            sp = rng.choice(ns, size=n_list, replace=False)
            for k in np.sort(sp):
                eff_species.append(int(k))
                eff_value.append(float(rng.uniform(0.5, 12.0)))
        eff_ptr.append(len(eff_species))

    def csr(side):
        ptr, sp, co = [0], [], []
        for rx in reactions:
            ms = rx[side]
            for k in sorted(set(ms)):
                sp.append(k)
                co.append(ms.count(k))
            ptr.append(len(sp))
        return (np.array(ptr, dtype=np.int32), np.array(sp, dtype=np.int32), np.array(co, dtype=np.int32))

    rp, rs, rc = csr(0)
    pp, ps, pc = csr(1)
    return Mechanism(
        elements=elements,
        elem_comp=np.ascontiguousarray(comp, dtype=np.int32),
        mol_weight=np.ascontiguousarray(W, dtype=np.float64),
        nasa_lo=nasa_lo,
        nasa_hi=nasa_hi,
        t_mid=t_mid,
        reac_ptr=rp,
        reac_species=rs,
        reac_coeff=rc,
        prod_ptr=pp,
        prod_species=ps,
        prod_coeff=pc,
        A=A,
        b=b,
        theta=theta,
        rtype=rtype,
        reversible=np.ones(nr, dtype=np.uint8),
        eff_default=np.ones(nr),
        eff_ptr=np.array(eff_ptr, dtype=np.int32),
        eff_species=np.array(eff_species, dtype=np.int32),
        eff_value=np.array(eff_value, dtype=np.float64),
        A0=A0,
        b0=b0,
        theta0=theta0,
        troe=troe,
        name=name,
        meta={"kind": kind, "seed": seed, "diluent": diluent, "inert": inert},
    )


# --------------------------------------------------------------------------
# the five configurations of BASELINE.json
# --------------------------------------------------------------------------
_MECH_SPEC = {
    # cfg: (kind, n_reactions, n_three_body, (eff_min, eff_max), n_troe, n_lindemann)
    0: ("h2", 21, 3, (3, 3), 1, 0),
    1: ("h2", 21, 3, (3, 3), 1, 0),
    2: ("gri", 325, 28, (6, 8), 22, 7),
    3: ("large", 700, 60, (6, 8), 50, 0),
    4: ("gri", 325, 28, (6, 8), 22, 7),
}

CONFIG_POINTS = {0: 4096, 1: 1 << 24, 2: 1 << 22, 3: 1 << 20, 4: 256**3}

_mech_cache = {}


def config_mechanism(cfg):
    """Mechanism of `configs[cfg]` (H0: seed 1000 + cfg; cfg 4 reuses cfg 2's)."""
    key = 2 if cfg == 4 else cfg
    if key not in _mech_cache:
        kind, nr, ntb, neff, ntroe, nlind = _MECH_SPEC[key]
        _mech_cache[key] = make_mechanism(kind, nr, ntb, neff, ntroe, nlind, seed=1000 + key, name=f"cfg{key}")
    return _mech_cache[key]


def _mean_weight(mech, Y):
    """(A.3): W = 1 / sum(Y_k / W_k); Y is [n_species][n]."""
    acc = np.zeros(Y.shape[1])
    for k in range(mech.n_species):   # no [n_species][n] temporary (7 GB at 256^3 x 53)
        acc += Y[k] / mech.mol_weight[k]
    return 1.0 / acc


def mixture_energy(mech, T, Y, dtype=np.longdouble):
    """e = sum_k Y_k (h_k - R T)/W_k (A.25, A.26), evaluated in `dtype`, rounded to double.

    Used only to produce the input `e` of the temperature solve (rule H9).  In
    numpy.longdouble (the default for small n) "Newton recovers T" tests the solve and
    not this generator; at bench sizes float64 is used because e is then just an input."""
    ld = dtype
    Ts = T.astype(ld)
    acc = np.zeros(T.shape[0], dtype=ld)
    for tm in np.unique(mech.t_mid):   # each species on its own range (reading G10); one mask per break temperature
        low = T < tm
        for mask, coef in ((low, mech.nasa_lo), (~low, mech.nasa_hi)):
            idx = np.nonzero(mask)[0]
            if idx.size == 0:
                continue
            Tk = Ts[idx]
            part = np.zeros(idx.size, dtype=ld)
            for k in np.nonzero(mech.t_mid == tm)[0]:
                a = coef[k].astype(ld)
                # (h/(R T) - 1) T = (a1-1) T + a2/2 T^2 + ... + a5/5 T^5 + a6
                poly = a[4] / 5
                poly = poly * Tk + a[3] / 4
                poly = poly * Tk + a[2] / 3
                poly = poly * Tk + a[1] / 2
                poly = poly * Tk + (a[0] - 1)
                poly = poly * Tk + a[5]
                part += Y[k, idx].astype(ld) * poly / ld(mech.mol_weight[k])
            acc[idx] += part
    return (acc * ld(R_UNIVERSAL)).astype(np.float64)


def with_species_break_temperatures(mech, t_mids):
    """A copy of `mech` whose species k switches NASA range at t_mids[k % len(t_mids)] instead of T_MID.  The
    high range keeps its a3..a5; a1, a2, a6, a7 are solved again so that c_p, dc_p/dT, h and s are continuous
    at the species' own break temperature (rule H1 at another T_mid).  Real NASA-7 files carry one break
    temperature per species; the configs use 1000 K throughout."""
    import copy
    out = copy.deepcopy(mech)
    out.t_mid = np.array([t_mids[k % len(t_mids)] for k in range(mech.n_species)], dtype=np.float64)
    out.nasa_hi = mech.nasa_hi.copy()
    for k in range(mech.n_species):
        lo, hi, Tm = mech.nasa_lo[k], out.nasa_hi[k], out.t_mid[k]
        dlo = lo[1] + 2 * lo[2] * Tm + 3 * lo[3] * Tm**2 + 4 * lo[4] * Tm**3
        hi[1] = dlo - (2 * hi[2] * Tm + 3 * hi[3] * Tm**2 + 4 * hi[4] * Tm**3)
        hi[0] = _cp_R(lo, Tm) - (hi[1] * Tm + hi[2] * Tm**2 + hi[3] * Tm**3 + hi[4] * Tm**4)
        hi[5] = lo[5] + sum((lo[m] - hi[m]) * Tm ** (m + 1) / (m + 1) for m in range(5))
        hi[6] = lo[6] + (lo[0] - hi[0]) * np.log(Tm) + sum((lo[m] - hi[m]) * Tm**m / m for m in range(1, 5))
    out.name = mech.name + "_tmids"
    return out


def _dirichlet(rng, alpha, ns, n):
    g = rng.standard_gamma(alpha, size=(ns, n))
    g = np.maximum(g, 1e-300)
    return g / g.sum(axis=0, keepdims=True)


def _diluted(rng, mech, alpha, n):
    """Rule H8: other species ~ Dirichlet(alpha), diluent fixed at d ~ U(0.6, 0.9)."""
    ns = mech.n_species
    dil = mech.meta["diluent"]
    Y = np.zeros((ns, n))
    others = [k for k in range(ns) if k != dil]
    d = rng.uniform(0.6, 0.9, size=n)
    Y[others] = _dirichlet(rng, alpha, ns - 1, n) * (1.0 - d)
    Y[dil] = d
    return Y


def config_states(cfg, n=None, seed=None, e_dtype=None):
    """States of `configs[cfg]` (H7-H9).  Returns a dict of float64 arrays:
    rho[n], T[n], Y[n_species][n], P[n]; for every cfg also e[n] and T_guess[n]
    (e by `mixture_energy`, in longdouble when n <= 2^18 unless `e_dtype` says otherwise;
    T_guess = T (1 + U(-0.1, 0.1)))."""
    mech = config_mechanism(cfg)
    n = CONFIG_POINTS[cfg] if n is None else int(n)
    rng = np.random.default_rng(2000 + cfg if seed is None else seed)
    ns = mech.n_species
    if e_dtype is None:
        e_dtype = np.longdouble if n <= (1 << 18) else np.float64
    if cfg == 4:
        return _flame_states(mech, rng, n, e_dtype)
    T = rng.uniform(300.0, 3000.0, size=n)
    if cfg in (0, 2):
        P = np.full(n, P_ATM)
    elif cfg == 1:
        P = P_ATM * np.exp(rng.uniform(np.log(0.1), np.log(50.0), size=n))
    else:
        P = P_ATM * np.exp(rng.uniform(np.log(1.0), np.log(40.0), size=n))
    if cfg == 2:
        Y = _diluted(rng, mech, 0.3, n)
    else:
        Y = _dirichlet(rng, 0.5 if cfg in (0, 1) else 0.3, ns, n)
    return _finish_states(mech, rng, T, P, Y, e_dtype)


def _finish_states(mech, rng, T, P, Y, e_dtype):
    n = T.shape[0]
    rho = P * _mean_weight(mech, Y) / (R_UNIVERSAL * T)
    e = np.empty(n)
    chunk = 1 << 20
    for s in range(0, n, chunk):
        e[s : s + chunk] = mixture_energy(mech, T[s : s + chunk], Y[:, s : s + chunk], e_dtype)
    T_guess = T * (1.0 + rng.uniform(-0.1, 0.1, size=n))
    return {
        "rho": np.ascontiguousarray(rho),
        "T": np.ascontiguousarray(T),
        "Y": np.ascontiguousarray(Y),
        "P": np.ascontiguousarray(P),
        "e": e,
        "T_guess": np.ascontiguousarray(T_guess),
    }


def _flame_states(mech, rng, n, e_dtype):
    """Rule H9: tanh flame front along x on a cubic grid with low-wavenumber perturbations.

    `n` must be a cube (256^3 at full size; smaller cubes for tests)."""
    m = round(n ** (1.0 / 3.0))
    if m**3 != n:
        raise ValueError("cfg 4 needs a cubic number of points")
    x = np.arange(m) / max(m - 1, 1)
    c1 = 0.5 * (1.0 + np.tanh((x - 0.5) / 0.05))
    # phi: seeded Fourier modes with max|k_i| <= 4, via an inverse FFT of a sparse spectrum
    spec = np.zeros((m, m, m), dtype=np.complex128)
    kmax = min(4, (m - 1) // 2)
    ks = range(-kmax, kmax + 1)
    for kz in ks:
        for ky in ks:
            for kx in ks:
                if (kx, ky, kz) == (0, 0, 0):
                    continue
                amp = rng.uniform(0.0, 1.0)
                ph = rng.uniform(0.0, 2 * np.pi)
                spec[kz % m, ky % m, kx % m] += amp * np.exp(1j * ph)
    phi = np.fft.ifftn(spec).real
    phi /= np.abs(phi).max()
    c = np.broadcast_to(c1[None, None, :], (m, m, m))
    T = ((300.0 + 2100.0 * c) * (1.0 + 0.05 * phi)).reshape(-1)
    cflat = np.ascontiguousarray(c).reshape(-1)
    Yu = _diluted(rng, mech, 0.3, 1)[:, 0]
    Yb = _diluted(rng, mech, 0.3, 1)[:, 0]
    Y = np.empty((mech.n_species, n))
    for k in range(mech.n_species):
        Y[k] = (1.0 - cflat) * Yu[k] + cflat * Yb[k]
    P = np.full(n, P_ATM)
    return _finish_states(mech, rng, np.ascontiguousarray(T), P, Y, e_dtype)


def simple_mechanism(species, reactions, elements=(), name="hand"):
    """Hand-written mechanism for pins and edge cases (no random numbers).

    species:   list of dicts {W, lo: [a1..a7], hi: [a1..a7] (default = lo), t_mid (default 1000),
               comp (optional element composition)}
    reactions: list of dicts {reac: {species: coeff}, prod: {species: coeff}, A, b, theta,
               type (default ELEMENTARY), reversible (default 1), eff_default (default 1),
               eff: {species: value}, eff_order: [species...] (default ascending), A0, b0, theta0,
               troe: (alpha, T3, T1, T2)}
    """
    ns = len(species)
    ne = len(elements)
    comp = np.zeros((ns, ne), dtype=np.int32)
    lo = np.zeros((ns, 7))
    hi = np.zeros((ns, 7))
    tm = np.zeros(ns)
    W = np.zeros(ns)
    for k, s in enumerate(species):
        W[k] = s["W"]
        lo[k] = s["lo"]
        hi[k] = s.get("hi", s["lo"])
        tm[k] = s.get("t_mid", T_MID)
        if ne:
            comp[k] = s["comp"]
    nr = len(reactions)

    def csr(key):
        ptr, sp, co = [0], [], []
        for r in reactions:
            for k in sorted(r[key]):
                sp.append(k)
                co.append(r[key][k])
            ptr.append(len(sp))
        return np.array(ptr, dtype=np.int32), np.array(sp, dtype=np.int32), np.array(co, dtype=np.int32)

    rp, rs, rc = csr("reac")
    pp, ps, pc = csr("prod")
    eptr, esp, eval_ = [0], [], []
    troe = np.zeros((nr, 4))
    troe[:, 0] = 1.0
    troe[:, 1:] = np.inf
    for j, r in enumerate(reactions):
        for k in r.get("eff_order", sorted(r.get("eff", {}))):   # eff_order: list the efficiencies in that order
            esp.append(k)
            eval_.append(r["eff"][k])
        eptr.append(len(esp))
        if "troe" in r:
            troe[j] = r["troe"]
    f = lambda key, default: np.array([r.get(key, default) for r in reactions], dtype=np.float64)
    return Mechanism(
        elements=list(elements), elem_comp=comp, mol_weight=W, nasa_lo=lo, nasa_hi=hi, t_mid=tm,
        reac_ptr=rp, reac_species=rs, reac_coeff=rc, prod_ptr=pp, prod_species=ps, prod_coeff=pc,
        A=f("A", 1.0), b=f("b", 0.0), theta=f("theta", 0.0),
        rtype=np.array([r.get("type", ELEMENTARY) for r in reactions], dtype=np.uint8),
        reversible=np.array([r.get("reversible", 1) for r in reactions], dtype=np.uint8),
        eff_default=f("eff_default", 1.0),
        eff_ptr=np.array(eptr, dtype=np.int32), eff_species=np.array(esp, dtype=np.int32),
        eff_value=np.array(eval_, dtype=np.float64),
        A0=f("A0", 1.0), b0=f("b0", 0.0), theta0=f("theta0", 0.0), troe=troe, name=name,
        meta={"kind": "hand"},
    )


# --------------------------------------------------------------------------
# transport fits: inputs of the mixture-averaged transport path (A.18)-(A.24)
# --------------------------------------------------------------------------
@dataclass
class Transport:
    """Polynomial fits in ln T of the species transport properties, in the forms the paper prints:
    mu_k = sqrt(T) (sum_m visc[k,m] (ln T)^m)^2 (A.22), kappa_k = sqrt(T) sum_m cond[k,m] (ln T)^m (A.24),
    D_kj = sqrt(T) sum_m diff[k,j,m] (ln T)^m (A.19).  SI units (Pa s, W/(m K), m^2/s)."""

    mol_weight: np.ndarray  # [n_species]
    visc: np.ndarray        # [n_species][5]
    cond: np.ndarray        # [n_species][5]
    diff: np.ndarray        # [n_species][n_species][5], symmetric in the species pair
    name: str = ""

    @property
    def n_species(self) -> int:
        return int(self.mol_weight.shape[0])


def make_transport(mol_weight, seed, name="transport"):
    """Synthetic fits shaped like those a kinetic-theory code produces (the paper takes them from Cantera,
    which is not available here): per species a Lennard-Jones diameter sigma ~ U(2.5, 5.5) Angstrom and well depth
    eps/k ~ U(30, 600) K; Chapman-Enskog viscosity, an Eucken-like conductivity and binary diffusivities at 1 atm from
    the textbook collision-integral fits (Neufeld), sampled at 32 temperatures over 250-3500 K and least-squares
    fitted in ln T in the printed forms.  These are input DATA: neither the oracle nor the CUDA path uses this code."""
    rng = np.random.default_rng(seed)
    W = np.asarray(mol_weight, dtype=np.float64)
    ns = W.shape[0]
    sigma = rng.uniform(2.5, 5.5, size=ns)
    eps = rng.uniform(30.0, 600.0, size=ns)
    eucken = rng.uniform(1.0, 2.0, size=ns)
    T = np.geomspace(250.0, 3500.0, 32)
    lnT = np.log(T)
    V = np.vander(lnT, 5, increasing=True)
    om22 = lambda ts: 1.16145 * ts ** -0.14874 + 0.52487 * np.exp(-0.7732 * ts) + 2.16178 * np.exp(-2.43787 * ts)
    om11 = lambda ts: 1.06036 * ts ** -0.1561 + 0.193 * np.exp(-0.47635 * ts) + 1.03587 * np.exp(-1.52996 * ts) \
        + 1.76474 * np.exp(-3.89411 * ts)
    visc = np.zeros((ns, 5))
    cond = np.zeros((ns, 5))
    diff = np.zeros((ns, ns, 5))
    for k in range(ns):
        mu = 2.6693e-6 * np.sqrt(W[k] * T) / (sigma[k] ** 2 * om22(T / eps[k]))           # Pa s
        visc[k] = np.linalg.lstsq(V, np.sqrt(mu / np.sqrt(T)), rcond=None)[0]
        ka = mu * 3.75 * R_UNIVERSAL / W[k] * eucken[k]                                     # W/(m K)
        cond[k] = np.linalg.lstsq(V, ka / np.sqrt(T), rcond=None)[0]
    for k in range(ns):
        for j in range(k, ns):
            s_kj = 0.5 * (sigma[k] + sigma[j])
            e_kj = np.sqrt(eps[k] * eps[j])
            d = 2.6628e-7 * np.sqrt(T ** 3 * (W[k] + W[j]) / (2.0 * W[k] * W[j])) / (s_kj ** 2 * om11(T / e_kj))   # m^2/s at 1 atm
            diff[k, j] = diff[j, k] = np.linalg.lstsq(V, d / np.sqrt(T), rcond=None)[0]
    return Transport(mol_weight=W.copy(), visc=visc, cond=cond, diff=diff, name=name)


def config_transport(cfg):
    """Transport fits for the species of configs[cfg] (seed 3000 + cfg; cfg 4 shares cfg 2's)."""
    c = 2 if cfg == 4 else cfg
    return make_transport(config_mechanism(cfg).mol_weight, 3000 + c, name=f"cfg{c}")
