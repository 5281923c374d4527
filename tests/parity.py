"""Tolerances of BASELINE.json `north_star`, used by every parity test.

    |omega_i - omega_i^oracle| <= 1e-11 * sum_k |nu_ik| (|r_f,k| + |r_r,k|)   per point and species
    |T - T^oracle| / T^oracle  <= 1e-12
"""
import numpy as np

OMEGA_TOL = 1e-11
T_TOL = 1e-12
EOS_TOL = 1e-13   # |d rho|/rho, |d p|/p: a sum of N_s positive terms in a different order


def omega_residual(omega, omega_ref, bound):
    """max over entries of |d omega| / bound (entries whose bound is 0 must match exactly)."""
    omega = np.asarray(omega, dtype=np.float64)
    omega_ref = np.asarray(omega_ref, dtype=np.float64)
    bound = np.asarray(bound, dtype=np.float64)
    err = np.abs(omega - omega_ref)
    zero = bound == 0
    assert np.all(err[zero] == 0), "species outside every reaction must have omega = 0 exactly"
    if zero.all():
        return 0.0
    return float(np.max(err[~zero] / bound[~zero]))


def assert_omega_parity(omega, omega_ref, bound):
    assert np.isfinite(omega).all()
    r = omega_residual(omega, omega_ref, bound)
    assert r <= OMEGA_TOL, f"max |d omega|/bound = {r:.3e} > {OMEGA_TOL}"
    return r


def assert_T_parity(T, T_ref):
    T = np.asarray(T, dtype=np.float64)
    T_ref = np.asarray(T_ref, dtype=np.float64)
    assert np.isfinite(T).all()
    r = float(np.max(np.abs(T - T_ref) / np.abs(T_ref))) if T.size else 0.0
    assert r <= T_TOL, f"max |dT|/T = {r:.3e} > {T_TOL}"
    return r


JAC_TOL = 1e-11   # chemical Jacobian and dS/dT: relative to the sum of the absolute terms of the entry


def assert_jacobian_parity(J, J_ref, bound):
    """|J_ik - J_ik^oracle| <= JAC_TOL * (sum of the absolute values of the entry's terms, as the oracle returns it);
    entries with no term at all must be exactly zero."""
    assert np.isfinite(J).all()
    r = omega_residual(J, J_ref, bound)
    assert r <= JAC_TOL, f"max |dJ|/bound = {r:.3e} > {JAC_TOL}"
    return r
