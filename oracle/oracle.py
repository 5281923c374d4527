"""ctypes front end of the CPU oracle (oracle/pyro_oracle.cpp).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from the CUDA path; the mechanism arrives as
a `paper_2503_24286_b200.inputs.Mechanism` (plain numpy arrays) or any object with the
same attributes.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pyro_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force=False):
    """g++ -O2 -ffp-contract=off -fopenmp: the plain definition, no contraction, no fast-math."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared",
               "-fPIC", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


class _Mech(C.Structure):
    _fields_ = [
        ("n_species", C.c_int32), ("n_reactions", C.c_int32),
        ("mol_weight", C.c_void_p), ("nasa_lo", C.c_void_p), ("nasa_hi", C.c_void_p), ("t_mid", C.c_void_p),
        ("reac_ptr", C.c_void_p), ("reac_species", C.c_void_p), ("reac_coeff", C.c_void_p),
        ("prod_ptr", C.c_void_p), ("prod_species", C.c_void_p), ("prod_coeff", C.c_void_p),
        ("A", C.c_void_p), ("b", C.c_void_p), ("theta", C.c_void_p),
        ("type", C.c_void_p), ("reversible", C.c_void_p),
        ("eff_default", C.c_void_p), ("eff_ptr", C.c_void_p), ("eff_species", C.c_void_p),
        ("eff_value", C.c_void_p),
        ("A0", C.c_void_p), ("b0", C.c_void_p), ("theta0", C.c_void_p), ("troe", C.c_void_p),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_num_threads.restype = C.c_int
        _lib.oracle_sizeof_real80.restype = C.c_int
        for sfx, real in (("f64", C.c_double), ("f80", C.c_longdouble)):
            getattr(_lib, f"oracle_mixture_e_{sfx}").restype = real
            getattr(_lib, f"oracle_mixture_cv_{sfx}").restype = real
            for nm in ("mixture_h", "mixture_cp"):
                getattr(_lib, f"oracle_{nm}_{sfx}").restype = real
                getattr(_lib, f"oracle_{nm}_{sfx}").argtypes = [C.c_void_p, real, C.c_void_p]
            getattr(_lib, f"oracle_get_temperature_h_{sfx}").argtypes = [
                C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, real, C.c_int,
                C.c_void_p, C.c_void_p, C.c_void_p]
            for nm in ("get_density", "get_pressure"):
                getattr(_lib, f"oracle_{nm}_{sfx}").argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p,
                                                                C.c_void_p, C.c_void_p, C.c_void_p]
            getattr(_lib, f"oracle_mixture_e_{sfx}").argtypes = [C.c_void_p, real, C.c_void_p]
            getattr(_lib, f"oracle_mixture_cv_{sfx}").argtypes = [C.c_void_p, real, C.c_void_p]
            getattr(_lib, f"oracle_species_thermo_{sfx}").argtypes = [C.c_void_p, C.c_int, real, C.c_void_p]
            getattr(_lib, f"oracle_reaction_detail_{sfx}").argtypes = [
                C.c_void_p, C.c_int, real, real, C.c_void_p, C.c_void_p]
            getattr(_lib, f"oracle_get_temperature_{sfx}").argtypes = [
                C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, real, C.c_int,
                C.c_void_p, C.c_void_p, C.c_void_p]
            getattr(_lib, f"oracle_get_net_production_rates_{sfx}").argtypes = [
                C.c_void_p, C.c_int64, C.c_int64] + [C.c_void_p] * 7
            getattr(_lib, f"oracle_get_transport_{sfx}").argtypes = [C.c_void_p, C.c_int64, C.c_int64] + [C.c_void_p] * 5
            getattr(_lib, f"oracle_reactor_cn_{sfx}").argtypes = [
                C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, real, C.c_int, C.c_int,
                real, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
            getattr(_lib, f"oracle_reactor_rk4_{sfx}").argtypes = [
                C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, real, C.c_int, real,
                C.c_int, C.c_void_p, C.c_void_p]
            getattr(_lib, f"oracle_get_jacobian_{sfx}").argtypes = [
                C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int] + [C.c_void_p] * 4
    return _lib


def num_threads():
    return int(_load().oracle_num_threads())


def set_num_threads(n):
    _load().oracle_set_num_threads(int(n))


_DETAIL_FIELDS = ("kf", "k_inf", "k0", "M", "Pr", "F", "Kc", "qf", "qr")


class Oracle:
    """The oracle bound to one mechanism.  `real` = "f64" (the oracle) or "f80" (long double arbiter)."""

    def __init__(self, mech, real="f64"):
        lib = _load()
        if real == "f80" and lib.oracle_sizeof_real80() != np.dtype(np.longdouble).itemsize:
            raise RuntimeError("long double layout mismatch between g++ and numpy")
        self.real = real
        self.dtype = np.float64 if real == "f64" else np.longdouble
        self._creal = C.c_double if real == "f64" else C.c_longdouble
        self.n_species = int(mech.n_species)
        self.n_reactions = int(mech.n_reactions)
        keep = {}

        def arr(x, dt):
            a = np.ascontiguousarray(np.asarray(x), dtype=dt)
            keep[id(a)] = a
            return a.ctypes.data

        m = _Mech()
        m.n_species, m.n_reactions = self.n_species, self.n_reactions
        for name in ("mol_weight", "nasa_lo", "nasa_hi", "t_mid", "A", "b", "theta", "eff_default",
                     "eff_value", "A0", "b0", "theta0", "troe"):
            setattr(m, name, arr(getattr(mech, name), np.float64))
        for name in ("reac_ptr", "reac_species", "reac_coeff", "prod_ptr", "prod_species", "prod_coeff",
                     "eff_ptr", "eff_species"):
            setattr(m, name, arr(getattr(mech, name), np.int32))
        m.type = arr(mech.rtype, np.uint8)
        m.reversible = arr(mech.reversible, np.uint8)
        self._keep = keep
        self._m = m
        self._lib = lib

    def _fn(self, name):
        return getattr(self._lib, f"oracle_{name}_{self.real}")

    def _vec(self, x):
        return np.ascontiguousarray(np.asarray(x), dtype=self.dtype)

    # ---- single-point pieces (pins) ----
    def species_thermo(self, k, T):
        """(cp/R, h/RT, s/R, g/RT) of species k at T   [(A.11)-(A.13), (A.31)]."""
        out = np.zeros(4, dtype=self.dtype)
        self._fn("species_thermo")(C.byref(self._m), int(k), self._creal(T), out.ctypes.data)
        return tuple(out)

    def mixture_e(self, T, Y):
        Y = self._vec(Y)
        return self._fn("mixture_e")(C.byref(self._m), self._creal(T), Y.ctypes.data)

    def mixture_cv(self, T, Y):
        Y = self._vec(Y)
        return self._fn("mixture_cv")(C.byref(self._m), self._creal(T), Y.ctypes.data)

    def mixture_h(self, T, Y):
        """Mixture enthalpy per unit mass (enthalpy form of the inversion)."""
        Y = self._vec(Y)
        return self._fn("mixture_h")(C.byref(self._m), self._creal(T), Y.ctypes.data)

    def mixture_cp(self, T, Y):
        Y = self._vec(Y)
        return self._fn("mixture_cp")(C.byref(self._m), self._creal(T), Y.ctypes.data)

    def reaction_detail(self, j, rho, T, Y):
        Y = self._vec(Y)
        out = np.zeros(9, dtype=self.dtype)
        self._fn("reaction_detail")(C.byref(self._m), int(j), self._creal(rho), self._creal(T),
                                    Y.ctypes.data, out.ctypes.data)
        return dict(zip(_DETAIL_FIELDS, out))

    # ---- field calls (SoA [species][points], leading dimension = n) ----
    def get_temperature(self, e, Y, T_guess, tol=1e-6, max_iter=10):
        e = self._vec(e)
        Y = self._vec(Y)
        Tg = self._vec(T_guess)
        n = e.shape[0]
        assert Y.shape == (self.n_species, n)
        T = np.empty(n, dtype=self.dtype)
        iters = np.empty(n, dtype=np.int32)
        conv = np.empty(n, dtype=np.int32)
        self._fn("get_temperature")(C.byref(self._m), n, n, e.ctypes.data, Y.ctypes.data, Tg.ctypes.data,
                                    self._creal(tol), int(max_iter), T.ctypes.data, iters.ctypes.data,
                                    conv.ctypes.data)
        return T, iters, conv

    def get_temperature_from_enthalpy(self, h, Y, T_guess, tol=1e-6, max_iter=10):
        h = self._vec(h)
        Y = self._vec(Y)
        Tg = self._vec(T_guess)
        n = h.shape[0]
        assert Y.shape == (self.n_species, n)
        T = np.empty(n, dtype=self.dtype)
        iters = np.empty(n, dtype=np.int32)
        conv = np.empty(n, dtype=np.int32)
        self._fn("get_temperature_h")(C.byref(self._m), n, n, h.ctypes.data, Y.ctypes.data, Tg.ctypes.data,
                                      self._creal(tol), int(max_iter), T.ctypes.data, iters.ctypes.data,
                                      conv.ctypes.data)
        return T, iters, conv

    def _eos(self, name, a, T, Y):
        a = self._vec(a)
        T = self._vec(T)
        Y = self._vec(Y)
        n = a.shape[0]
        assert Y.shape == (self.n_species, n)
        out = np.empty(n, dtype=self.dtype)
        self._fn(name)(C.byref(self._m), n, n, a.ctypes.data, T.ctypes.data, Y.ctypes.data, out.ctypes.data)
        return out

    def get_density(self, p, T, Y):
        """rho = p W / (R T), W = 1 / sum_k Y_k/W_k   (A.2), (A.3) PAPER.md:892-899."""
        return self._eos("get_density", p, T, Y)

    def get_pressure(self, rho, T, Y):
        return self._eos("get_pressure", rho, T, Y)

    def get_net_production_rates(self, rho, T, Y, want_rates=False, want_bound=True):
        rho = self._vec(rho)
        T = self._vec(T)
        Y = self._vec(Y)
        n = rho.shape[0]
        assert Y.shape == (self.n_species, n)
        omega = np.empty((self.n_species, n), dtype=self.dtype)
        bound = np.empty((self.n_species, n), dtype=self.dtype) if want_bound else None
        rf = np.empty((self.n_reactions, n), dtype=self.dtype) if want_rates else None
        rr = np.empty((self.n_reactions, n), dtype=self.dtype) if want_rates else None
        self._fn("get_net_production_rates")(
            C.byref(self._m), n, n, rho.ctypes.data, T.ctypes.data, Y.ctypes.data, omega.ctypes.data,
            bound.ctypes.data if want_bound else None, rf.ctypes.data if want_rates else None,
            rr.ctypes.data if want_rates else None)
        if want_rates:
            return omega, bound, rf, rr
        return omega, bound

    def get_jacobian(self, rho, T, Y, mode=0):
        """Chemical Jacobian J[i, k, p] = dS_i/dY_k (S_i = W_i omega_i, eq. (6), (A.36)) and
        dSdT[i, p] = dS_i/dT at fixed (rho, Y).  mode 0: Y-derivatives at fixed (rho, T); mode 1: at fixed
        (rho, e), i.e. through the temperature inversion as the paper's listing 23 (reading G26).
        Returns J, dSdT and the sums of absolute terms boundJ, bounddSdT that scale the parity tolerance."""
        rho = self._vec(rho)
        T = self._vec(T)
        Y = self._vec(Y)
        n = rho.shape[0]
        ns = self.n_species
        assert Y.shape == (ns, n)
        J = np.empty((ns, ns, n), dtype=self.dtype)
        bJ = np.empty((ns, ns, n), dtype=self.dtype)
        dSdT = np.empty((ns, n), dtype=self.dtype)
        bT = np.empty((ns, n), dtype=self.dtype)
        self._fn("get_jacobian")(C.byref(self._m), n, n, rho.ctypes.data, T.ctypes.data, Y.ctypes.data, int(mode),
                                 J.ctypes.data, dSdT.ctypes.data, bJ.ctypes.data, bT.ctypes.data)
        return J, dSdT, bJ, bT

    def reactor_rk4(self, rho, e, Y, T_guess, dt, n_steps, tol=1e-6, max_iter=10):
        """n_steps classical Runge-Kutta steps of size dt of the adiabatic isochoric reactors (A.1) PAPER.md:886-888
        (PAPER.md:616), one reactor per point.  Returns (Y, T, Ybound, n_not_converged): final mass fractions,
        temperature of the final state, the accumulated size of the terms added into each Y_k."""
        rho = self._vec(rho)
        e = self._vec(e)
        Y = self._vec(Y).copy()
        T = self._vec(T_guess).copy()
        n = rho.shape[0]
        assert Y.shape == (self.n_species, n)
        Yb = np.empty_like(Y)
        bad = C.c_int64(0)
        self._fn("reactor_rk4")(C.byref(self._m), n, n, rho.ctypes.data, e.ctypes.data, Y.ctypes.data, T.ctypes.data,
                                self._creal(dt), int(n_steps), self._creal(tol), int(max_iter), Yb.ctypes.data,
                                C.byref(bad))
        return Y, T, Yb, int(bad.value)

    def reactor_cn(self, rho, e, Y, T_guess, dt, n_steps, newton_iters=4, tol=1e-6, max_iter=10):
        """n_steps Crank-Nicolson steps (A.32)-(A.36) PAPER.md:1043-1062 of the reactors, `newton_iters` Newton
        iterations each.  Returns (Y, T, Ybound, last_update, n_not_converged)."""
        rho = self._vec(rho)
        e = self._vec(e)
        Y = self._vec(Y).copy()
        T = self._vec(T_guess).copy()
        n = rho.shape[0]
        assert Y.shape == (self.n_species, n)
        Yb = np.empty_like(Y)
        lu = np.empty(n, dtype=self.dtype)
        bad = C.c_int64(0)
        self._fn("reactor_cn")(C.byref(self._m), n, n, rho.ctypes.data, e.ctypes.data, Y.ctypes.data, T.ctypes.data,
                               self._creal(dt), int(n_steps), int(newton_iters), self._creal(tol), int(max_iter),
                               Yb.ctypes.data, lu.ctypes.data, C.byref(bad))
        return Y, T, Yb, lu, int(bad.value)


class _Transport(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("mol_weight", C.c_void_p), ("visc", C.c_void_p), ("cond", C.c_void_p),
                ("diff", C.c_void_p)]


class TransportOracle:
    """Mixture-averaged transport properties (A.18)-(A.24) PAPER.md:968-996 for a table of polynomial fits
    (`paper_2503_24286_b200.inputs.Transport` or any object with mol_weight [ns], visc [ns,5], cond [ns,5],
    diff [ns,ns,5])."""

    def __init__(self, tr, real="f64"):
        self._lib = _load()
        self.real = real
        self.dtype = np.float64 if real == "f64" else np.longdouble
        self.n_species = int(np.asarray(tr.mol_weight).shape[0])
        self._keep = [np.ascontiguousarray(np.asarray(getattr(tr, k)), dtype=np.float64)
                      for k in ("mol_weight", "visc", "cond", "diff")]
        assert self._keep[1].shape == (self.n_species, 5) and self._keep[3].shape == (self.n_species, self.n_species, 5)
        self._t = _Transport(self.n_species, *[a.ctypes.data for a in self._keep])

    def get_transport(self, T, Y):
        """Returns (mu [n], kappa [n], D_km [n_species, n])."""
        T = np.ascontiguousarray(np.asarray(T), dtype=self.dtype)
        Y = np.ascontiguousarray(np.asarray(Y), dtype=self.dtype)
        n = T.shape[0]
        assert Y.shape == (self.n_species, n)
        mu = np.empty(n, dtype=self.dtype)
        ka = np.empty(n, dtype=self.dtype)
        D = np.empty((self.n_species, n), dtype=self.dtype)
        getattr(self._lib, f"oracle_get_transport_{self.real}")(C.byref(self._t), n, n, T.ctypes.data, Y.ctypes.data,
                                                                mu.ctypes.data, ka.ctypes.data, D.ctypes.data)
        return mu, ka, D
