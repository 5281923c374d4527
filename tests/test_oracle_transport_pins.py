"""Pins of the oracle's mixture-averaged transport (no GPU): SURVEY.md 8(f) NEXT-3, (A.18)-(A.24) PAPER.md:968-996.
  X1  a single species returns its own mu_k and kappa_k (Phi_kk = 1)
  X2  identical species mix to the species value at any composition
  X3  W7: 50-digit evaluation of a hand-written three-species mixture (tests/golden/make_w7.py)
  X4  binary mixture: D_1,m = W_2 D_12 / W   (from (A.18) with X_1 + X_2 = 1)
  X5  permuting the species permutes D_k,m and leaves mu, kappa unchanged
  X6  Wilke limits: equal weights and equal viscosities give Phi = 1, so mu = sum X_k mu_k / sum X_j = mu_k
"""
import importlib.util
import os

import mpmath as mp
import numpy as np
import pytest

from conftest import read_golden
from oracle import oracle
from paper_2503_24286_b200 import inputs
from paper_2503_24286_b200.inputs import Transport


def _poly(c, x):
    return sum(cm * x ** m for m, cm in enumerate(c))


def _w7(golden_dir):
    spec = importlib.util.spec_from_file_location("make_w7", os.path.join(golden_dir, "make_w7.py"))
    mk = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mk)
    diff = np.zeros((3, 3, 5))
    for (k, j), c in mk.DIFF.items():
        diff[k, j] = diff[j, k] = [float(x) for x in c]
    diff[0, 0] = diff[1, 1] = diff[2, 2] = [1e-6, 0, 0, 0, 0]   # never read: j != k in (A.18)
    tr = Transport(mol_weight=np.array([float(w) for w in mk.WEIGHT]),
                   visc=np.array([[float(x) for x in row] for row in mk.VISC]),
                   cond=np.array([[float(x) for x in row] for row in mk.COND]), diff=diff)
    return mk, tr


def test_x3_w7_fixture_and_oracle(golden_dir):
    mk, tr = _w7(golden_dir)
    g = read_golden(os.path.join(golden_dir, "w7_transport.txt"))
    for key, val in mk.compute():   # the fixture is what the equations give
        assert abs(val / mp.mpf(g[key]) - 1) < mp.mpf("1e-18"), key
    g = {k: float(v) for k, v in g.items()}
    Y = np.array([[float(y)] for y in mk.Y])
    for real, tol in (("f64", 2e-14), ("f80", 5e-15)):   # the fits are decimal numbers rounded to double: input rounding times the conditioning of the polynomials
        mu, ka, D = oracle.TransportOracle(tr, real).get_transport([float(mk.T)], Y)
        assert abs(float(mu[0]) / g["mu_mix"] - 1) < tol
        assert abs(float(ka[0]) / g["kappa_mix"] - 1) < tol
        for k in range(3):
            assert abs(float(D[k, 0]) / g[f"D_{k}m"] - 1) < tol, k
    # the diagonal of the binary table is never read
    tr.diff[0, 0] = np.nan
    mu2, ka2, D2 = oracle.TransportOracle(tr).get_transport([float(mk.T)], Y)
    assert np.isfinite(D2).all()


def test_x1_single_species_and_x2_identical_species():
    tr9 = inputs.config_transport(0)
    for k in (0, 3, 8):
        one = Transport(mol_weight=tr9.mol_weight[k:k + 1], visc=tr9.visc[k:k + 1], cond=tr9.cond[k:k + 1],
                        diff=tr9.diff[k:k + 1, k:k + 1])
        for T in (300.0, 1234.5, 3000.0):
            mu, ka, D = oracle.TransportOracle(one).get_transport([T], [[1.0]])
            lnT = np.log(T)
            assert abs(mu[0] / (np.sqrt(T) * _poly(tr9.visc[k], lnT) ** 2) - 1) < 1e-12     # (A.22), Phi_kk = 1 (the fits cancel two digits in ln T: Horner against the power sum)
            assert abs(ka[0] / (np.sqrt(T) * _poly(tr9.cond[k], lnT)) - 1) < 1e-12          # (A.24)
        # four copies of the species: any composition gives the species' own values
        four = Transport(mol_weight=np.repeat(tr9.mol_weight[k:k + 1], 4), visc=np.repeat(tr9.visc[k:k + 1], 4, axis=0),
                         cond=np.repeat(tr9.cond[k:k + 1], 4, axis=0), diff=np.tile(tr9.diff[k, (k + 1) % 9], (4, 4, 1)))
        Y = np.random.default_rng(k).dirichlet(np.ones(4), size=5).T
        mu4, ka4, D4 = oracle.TransportOracle(four).get_transport(np.full(5, 1234.5), Y)
        mu1, ka1, _ = oracle.TransportOracle(one).get_transport([1234.5], [[1.0]])
        assert np.allclose(mu4, mu1[0], rtol=1e-13) and np.allclose(ka4, ka1[0], rtol=1e-13)
        # all binary diffusivities equal D: D_k,m = (1 - X_k) D / (1 - X_k) = D (equal weights)
        Dref = np.sqrt(1234.5) * _poly(tr9.diff[k, (k + 1) % 9], np.log(1234.5))
        assert np.allclose(D4, Dref, rtol=1e-11)


def test_x4_binary_mixture_closed_form():
    tr9 = inputs.config_transport(0)
    a, b = 2, 6
    two = Transport(mol_weight=tr9.mol_weight[[a, b]], visc=tr9.visc[[a, b]], cond=tr9.cond[[a, b]],
                    diff=tr9.diff[np.ix_([a, b], [a, b])])
    T = 1500.0
    for y in (0.1, 0.5, 0.93):
        Y = np.array([[y], [1 - y]])
        W = 1.0 / (y / two.mol_weight[0] + (1 - y) / two.mol_weight[1])
        D12 = np.sqrt(T) * _poly(two.diff[0, 1], np.log(T))
        mu, ka, D = oracle.TransportOracle(two).get_transport([T], Y)
        assert abs(D[0, 0] / (two.mol_weight[1] * D12 / W) - 1) < 1e-13
        assert abs(D[1, 0] / (two.mol_weight[0] * D12 / W) - 1) < 1e-13


@pytest.mark.parametrize("cfg", [0, 2])
def test_x5_permutation_of_species(cfg):
    tr = inputs.config_transport(cfg)
    st = inputs.config_states(cfg, n=16)
    perm = np.random.default_rng(4).permutation(tr.n_species)
    trp = Transport(mol_weight=tr.mol_weight[perm], visc=tr.visc[perm], cond=tr.cond[perm], diff=tr.diff[np.ix_(perm, perm)])
    mu, ka, D = oracle.TransportOracle(tr).get_transport(st["T"], st["Y"])
    mup, kap, Dp = oracle.TransportOracle(trp).get_transport(st["T"], st["Y"][perm])
    assert np.allclose(mup, mu, rtol=1e-13) and np.allclose(kap, ka, rtol=1e-13) and np.allclose(Dp, D[perm], rtol=1e-12)
    assert np.all(mu > 0) and np.all(ka > 0) and np.all(D > 0)
    # f64 against long double
    mu8, ka8, D8 = oracle.TransportOracle(tr, "f80").get_transport(st["T"], st["Y"])
    assert np.max(np.abs(mu / mu8.astype(np.float64) - 1)) < 1e-13 and np.max(np.abs(D / D8.astype(np.float64) - 1)) < 1e-12


def test_x6_wilke_limits():
    """Equal weights and equal viscosities: Phi_kj = (1 + 1)^2 / sqrt(16) = 1, so mu = mu_k.  Equal weights only:
    Phi_kj = (1 + sqrt(mu_k/mu_j))^2 / 4, checked on a binary mixture by hand."""
    tr9 = inputs.config_transport(0)
    T = 800.0
    two = Transport(mol_weight=np.array([20.0, 20.0]), visc=tr9.visc[[1, 4]], cond=tr9.cond[[1, 4]],
                    diff=tr9.diff[np.ix_([1, 4], [1, 4])])
    m1, m2 = (np.sqrt(T) * _poly(two.visc[i], np.log(T)) ** 2 for i in range(2))
    x1 = 0.3
    Y = np.array([[x1], [1 - x1]])   # equal weights: X = Y
    p12 = (1 + np.sqrt(m1 / m2)) ** 2 / 4
    p21 = (1 + np.sqrt(m2 / m1)) ** 2 / 4
    ref = x1 * m1 / (x1 + p12 * (1 - x1)) + (1 - x1) * m2 / (p21 * x1 + (1 - x1))
    mu, _, _ = oracle.TransportOracle(two).get_transport([T], Y)
    assert abs(mu[0] / ref - 1) < 1e-14
