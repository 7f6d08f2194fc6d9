"""Pins P5-P9 for the oracle's transport functions O4-O8 (Wilke, combination rule, mixture-averaged D).

PAPER.md names only the diffusion model ("Hirschfelder and Curtiss mixture-averaged transport
model"; "non-unity Lewis number"); BASELINE.json north_star names the viscosity and
conductivity rules.  The pins are hand-evaluated special cases, reductions and invariants.
"""
import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

from oracle import oracle
from paper_2312_05800_b200 import synth
from tests.helpers import read_textbook, tiny_mech


def _rand_Y(rng, K, n=1):
    y = rng.dirichlet(np.full(K, 0.7), size=n).T
    return np.ascontiguousarray(y)


def test_o5_fits_against_numpy_polyval(cfg1, omech1):
    """O5: sqrt(mu_k) = T^{1/4} P_b(ln T), lambda_k = T^{1/2} P_c(ln T), p D_jk = T^{3/2} P_d(ln T)."""
    mech = cfg1[0]
    pv = np.polynomial.polynomial.polyval
    for T, p in ((300.0, 101325.0), (1777.0, 5e5)):
        mu, lam, D = omech1.species_transport(T, p)
        L = np.log(T)
        for k in range(mech.K):
            assert mu[k] == pytest.approx((T ** 0.25 * pv(L, mech.visc_fit[k])) ** 2, rel=1e-13)
            assert lam[k] == pytest.approx(T ** 0.5 * pv(L, mech.cond_fit[k]), rel=1e-13)
            for j in range(mech.K):
                assert D[j, k] == pytest.approx(T ** 1.5 * pv(L, mech.bdiff_fit[j, k]) / p, rel=1e-13)
        assert np.allclose(D, D.T, rtol=0, atol=0)


def test_p9_generator_textbook_magnitudes():
    tb = read_textbook()
    v, tol = tb["n2_viscosity_300K"]
    assert abs(synth.kinetic_theory_viscosity(28.0134, 3.798, 71.4, 300.0) - v) <= tol * v
    v, tol = tb["n2_o2_diffusivity_300K_1atm"]
    d = synth.kinetic_theory_pD(28.0134, 31.998, 3.798, 3.467, 71.4, 106.7, 300.0) / 101325.0
    assert abs(d - v) <= tol * v


def test_generator_fits_reproduce_kinetic_theory(cfg1, omech1):
    """The fitted tables evaluated by the oracle track the kinetic-theory curves to < 1 % (units check)."""
    mech = cfg1[0]
    for T in (300.0, 900.0, 2500.0):
        mu, lam, D = omech1.species_transport(T, 101325.0)
        for k in range(mech.K):
            ref = synth.kinetic_theory_viscosity(mech.W[k], mech.sigma[k], mech.eps_over_k[k], T)
            assert abs(mu[k] / ref - 1) < 1e-2
        ref = synth.kinetic_theory_pD(mech.W[0], mech.W[1], mech.sigma[0], mech.sigma[1],
                                      mech.eps_over_k[0], mech.eps_over_k[1], T) / 101325.0
        assert abs(D[0, 1] / ref - 1) < 1e-2


def test_p5_one_hot_reduces_to_pure_species(cfg1, omech1):
    """P5 / A7: Y = e_k => mu = mu_k, lambda = lambda_k, D_jm = D_jk (j != k), D_km = D_kk."""
    mech = cfg1[0]
    K = mech.K
    T, p = 1450.0, 2.0e5
    mu_k, lam_k, D = omech1.species_transport(T, p)
    for k in range(K):
        Y = np.zeros((K, 1)); Y[k] = 1.0
        r = omech1.properties(np.array([T]), np.array([p]), Y)
        assert r["mu"][0] == pytest.approx(mu_k[k], rel=1e-13)
        assert r["lam"][0] == pytest.approx(lam_k[k], rel=1e-13)
        for j in range(K):
            assert r["D"][j, 0] == pytest.approx(D[j, k], rel=1e-13)   # includes j == k -> D_kk


def test_p6_identical_species():
    """P6: all species identical => Phi = 1, mu = mu_k, lambda = lambda_k, D_km = D for every Y."""
    K = 5
    visc = np.zeros((K, 5)); visc[:, 0] = 2e-3; visc[:, 1] = 1e-4
    cond = np.zeros((K, 5)); cond[:, 0] = 3e-3
    bd = np.zeros((K, K, 5)); bd[:, :, 0] = 2e-5
    m = oracle.Mech(tiny_mech(K, W=np.full(K, 17.0), visc=visc, cond=cond, bdiff=bd))
    rng = np.random.default_rng(3)
    Y = _rand_Y(rng, K, 7)
    T = np.linspace(400, 2400, 7); p = np.full(7, 101325.0)
    r = m.properties(T, p, Y)
    for i in range(7):
        mu_k, lam_k, D = m.species_transport(T[i], p[i])
        assert r["mu"][i] == pytest.approx(mu_k[0], rel=1e-13)
        assert r["lam"][i] == pytest.approx(lam_k[0], rel=1e-13)
        assert np.allclose(r["D"][:, i], D[0, 0], rtol=1e-13)


def test_p7_wilke_hand_values_K2():
    """P7: hand-evaluated Wilke for K = 2, X = (1/2, 1/2).

    (a) mu_1 = mu_2, W_2/W_1 = 16: Phi_12 = (1+2)^2/sqrt(8(1+1/16)) = 9/sqrt(8.5),
        Phi_21 = (1+1/2)^2/sqrt(8*17) = 2.25/sqrt(136); mu/mu_1 = 1/(1+Phi_12) + 1/(1+Phi_21).
    (b) mu_1 = 4 mu_2, W_1 = W_2: Phi_12 = (1+2)^2/4 = 9/4, Phi_21 = (3/2)^2/4 = 9/16;
        mu = 4 mu_1/13 + 16 mu_2/25 = (608/325) mu_2.
    """
    T, p = 900.0, 101325.0
    # (a)
    visc = np.zeros((2, 5)); visc[:, 0] = 1.5e-3
    W = np.array([1.0, 16.0])
    m = oracle.Mech(tiny_mech(2, W=W, visc=visc))
    X = np.array([0.5, 0.5]); Y = (X * W / np.sum(X * W)).reshape(2, 1)
    mu1 = np.sqrt(T) * 1.5e-3 ** 2
    expect = mu1 * (1 / (1 + 9 / np.sqrt(8.5)) + 1 / (1 + 2.25 / np.sqrt(136.0)))
    assert m.properties(np.array([T]), np.array([p]), Y)["mu"][0] == pytest.approx(expect, rel=1e-13)
    # (b)
    visc = np.zeros((2, 5)); visc[0, 0] = 2e-3; visc[1, 0] = 1e-3
    m = oracle.Mech(tiny_mech(2, W=[30.0, 30.0], visc=visc))
    mu2 = np.sqrt(T) * 1e-3 ** 2
    Y = np.array([[0.5], [0.5]])
    assert m.properties(np.array([T]), np.array([p]), Y)["mu"][0] == pytest.approx(608.0 / 325.0 * mu2, rel=1e-13)


def test_p7_binary_diffusion_closed_form():
    """P7: binary mixture D_1m = D_12 Y_2/X_2 = D_12 W_2/Wbar, D_2m = D_12 W_1/Wbar."""
    W = np.array([2.0, 32.0])
    m = oracle.Mech(tiny_mech(2, W=W))
    T, p = 1100.0, 3e5
    _, _, D = m.species_transport(T, p)
    Y = np.array([[0.2], [0.8]])
    Wbar = 1.0 / np.sum(Y[:, 0] / W)
    r = m.properties(np.array([T]), np.array([p]), Y)
    assert r["D"][0, 0] == pytest.approx(D[0, 1] * W[1] / Wbar, rel=1e-13)
    assert r["D"][1, 0] == pytest.approx(D[0, 1] * W[0] / Wbar, rel=1e-13)


def test_p7_combination_rule_hand_value():
    """O7 / A6: K = 2, X = (1/2, 1/2), lambda = (1, 3): 1/2 [2 + 1/(1/2 + 1/6)] = 1/2 [2 + 3/2] = 7/4."""
    cond = np.zeros((2, 5)); cond[0, 0] = 1.0; cond[1, 0] = 3.0
    m = oracle.Mech(tiny_mech(2, W=[10.0, 10.0], cond=cond))
    r = m.properties(np.array([1.0]), np.array([1e5]), np.array([[0.5], [0.5]]))   # sqrt(T) = 1
    assert r["lam"][0] == pytest.approx(1.75, rel=1e-14)


@settings(max_examples=25, deadline=None)
@given(st.integers(0, 10_000))
def test_p8_invariants(seed):
    """P8: harmonic <= lambda <= arithmetic; D > 0; D ~ 1/p; cp, mu, lambda independent of p;
    permutation equivariance; splitting a species into two identical copies changes nothing."""
    rng = np.random.default_rng(seed)
    K = int(rng.integers(2, 6))
    mech = synth.make_mechanism(K, 1000 + seed)
    m = oracle.Mech(mech)
    Y = _rand_Y(rng, K)
    T = np.array([rng.uniform(300, 3000)]); p = np.array([rng.uniform(5e4, 5e5)])
    r = m.properties(T, p, Y)
    mu_k, lam_k, _ = m.species_transport(T[0], p[0])
    X = (Y[:, 0] / mech.W) / np.sum(Y[:, 0] / mech.W)
    assert 1.0 / np.sum(X / lam_k) * (1 - 1e-12) <= r["lam"][0] <= np.sum(X * lam_k) * (1 + 1e-12)
    assert np.all(r["D"][:, 0] > 0)
    r2 = m.properties(T, 2 * p, Y)
    assert np.allclose(r2["D"][:, 0], 0.5 * r["D"][:, 0], rtol=1e-13)
    for key in ("cp", "h", "mu", "lam"):
        assert r2[key][0] == pytest.approx(r[key][0], rel=1e-14)
    # permutation
    perm = rng.permutation(K)
    import copy
    mp = copy.copy(mech)
    mp.W = mech.W[perm]; mp.nasa_lo = mech.nasa_lo[perm]; mp.nasa_hi = mech.nasa_hi[perm]
    mp.visc_fit = mech.visc_fit[perm]; mp.cond_fit = mech.cond_fit[perm]
    mp.bdiff_fit = mech.bdiff_fit[np.ix_(perm, perm)]
    rp = oracle.Mech(mp).properties(T, p, np.ascontiguousarray(Y[perm]))
    for key in ("cp", "h", "mu", "lam"):
        assert rp[key][0] == pytest.approx(r[key][0], rel=1e-12)
    assert np.allclose(rp["D"][:, 0], r["D"][perm, 0], rtol=1e-12)
    # split species 0 into two identical copies carrying fractions (a, 1-a) of Y_0
    idx = np.r_[0, np.arange(K)]
    ms = copy.copy(mech)
    ms.K = K + 1
    ms.W = mech.W[idx]; ms.nasa_lo = mech.nasa_lo[idx]; ms.nasa_hi = mech.nasa_hi[idx]
    ms.visc_fit = mech.visc_fit[idx]; ms.cond_fit = mech.cond_fit[idx]
    ms.bdiff_fit = mech.bdiff_fit[np.ix_(idx, idx)]
    a = rng.uniform(0.1, 0.9)
    Ys = np.ascontiguousarray(Y[idx]); Ys[0] *= a; Ys[1] *= (1 - a)
    rs = oracle.Mech(ms).properties(T, p, Ys)
    for key in ("cp", "h", "mu", "lam"):
        assert rs[key][0] == pytest.approx(r[key][0], rel=1e-12)


def test_mole_fraction_weighting_in_wilke():
    """O4/O6: a heavy trace species by MASS is a tiny MOLE fraction -- mu must follow X, not Y.
    K = 2, equal mu_k would hide it, so use Phi = 1 (equal W impossible) -> instead check the
    combination rule, which depends on X only: X from Y = (0.5, 0.5), W = (2, 32) is (16/17, 1/17)."""
    cond = np.zeros((2, 5)); cond[0, 0] = 1.0; cond[1, 0] = 2.0
    m = oracle.Mech(tiny_mech(2, W=[2.0, 32.0], cond=cond))
    r = m.properties(np.array([1.0]), np.array([1e5]), np.array([[0.5], [0.5]]))
    X = np.array([16.0 / 17.0, 1.0 / 17.0])
    expect = 0.5 * (X[0] * 1 + X[1] * 2 + 1.0 / (X[0] / 1 + X[1] / 2))
    assert r["lam"][0] == pytest.approx(expect, rel=1e-14)
