"""Pins of the oracle's NEXT-3 / NEXT-4 functions (readings A22, A23 in DESIGN.md) against what the
definitions and the already pinned functions fix: identities, closed forms, limits, brute force."""
import numpy as np
import pytest

from tests import helpers

R = helpers.R
P0 = 101325.0


@pytest.fixture(scope="module")
def case():
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech = synth.make_mechanism(9, 4242)
    cells = synth.cells_dirichlet(9, 257, 4242)
    return mech, oracle.Mech(mech), cells


# ------------------------------------------------------------------------------------------------------------------
# NEXT-4: rho, psi, alpha, rho D_k, h_k(T), s
# ------------------------------------------------------------------------------------------------------------------
def test_density_of_air_textbook():
    """rho = p Wbar / (R T): dry air (W = 28.96 kg/kmol) at 300 K, 1 atm is 1.177 kg/m^3 (textbook value, golden file)."""
    from oracle import oracle
    val, tol = helpers.read_textbook()["air_density_300K_1atm"]
    om = oracle.Mech(helpers.tiny_mech(1, W=[28.96]))
    out = om.extras(np.array([300.0]), np.array([P0]), np.ones((1, 1)))
    assert abs(out["rho"][0] / val - 1.0) <= tol


def test_identities(case):
    mech, om, cells = case
    T, p, Y = cells.T.astype(float), cells.p.astype(float) * np.linspace(0.5, 2.0, cells.n), cells.Y.astype(float)
    props = om.properties(T, p, Y)
    out = om.extras(T, p, Y, cp=props["cp"], lam=props["lam"], D=props["D"])
    Wbar = 1.0 / (Y / mech.W[:, None]).sum(axis=0)
    assert np.allclose(out["rho"] * R * T / Wbar, p, rtol=1e-13)            # ideal gas
    assert np.allclose(out["psi"] * p, out["rho"], rtol=1e-13)               # psi = d rho / d p at constant T
    assert np.allclose(out["alpha"] * props["cp"], props["lam"], rtol=1e-13)
    assert np.allclose(out["rhoD"], out["rho"][None, :] * props["D"], rtol=1e-13)
    # sum_k Y_k h_k(T) is the mixture enthalpy of the (separately pinned) O2
    _, h = om.mixture_cp_h(T, Y)
    assert np.allclose((Y * out["hk"]).sum(axis=0), h, rtol=1e-12, atol=1e-6)
    # h_k depends on T only: one-hot cells give h = h_k
    for k in range(mech.K):
        assert np.isclose(out["hk"][k, 0], om.species_thermo(k, T[0])[1] / mech.W[k], rtol=1e-14)


def test_entropy_pure_species_and_pressure_term(case):
    mech, om, _ = case
    K = mech.K
    T = np.array([400.0, 1500.0])
    for k in (0, K - 1):
        Y = np.zeros((K, 2)); Y[k] = 1.0
        for p in (P0, 3.0 * P0):
            s = om.extras(T, np.full(2, p), Y)["s"]
            ref = [om.species_thermo(k, t)[2] / mech.W[k] - R / mech.W[k] * np.log(p / P0) for t in T]
            assert np.allclose(s, ref, rtol=1e-13)


def test_entropy_of_mixing_closed_form():
    """Two identical species, equimolar: s exceeds the pure value by (R / W) ln 2; X_k = 0 terms drop out."""
    from oracle import oracle
    om = oracle.Mech(helpers.tiny_mech(3, W=[20.0, 20.0, 20.0]))
    T, p = np.array([800.0]), np.array([P0])
    pure = om.extras(T, p, np.array([[1.0], [0.0], [0.0]]))["s"][0]
    mixed = om.extras(T, p, np.array([[0.5], [0.5], [0.0]]))["s"][0]
    assert np.isclose(mixed - pure, R / 20.0 * np.log(2.0), rtol=1e-12)


def test_entropy_temperature_derivative_is_cp_over_T(case):
    """(ds/dT) at constant p, Y = cp / T: ties the mixture entropy to the pinned cp (central difference)."""
    mech, om, cells = case
    T, p, Y = cells.T.astype(float), cells.p.astype(float), cells.Y.astype(float)
    keep = np.abs(T - mech.T_mid) > 1.0          # the difference must not straddle the range break
    dT = 1e-2
    s1 = om.extras(T + dT, p, Y)["s"]
    s0 = om.extras(T - dT, p, Y)["s"]
    cp, _ = om.mixture_cp_h(T, Y)
    assert np.allclose(((s1 - s0) / (2 * dT))[keep], (cp / T)[keep], rtol=1e-7)


# ------------------------------------------------------------------------------------------------------------------
# NEXT-3: PaSR scaling and temperature gate
# ------------------------------------------------------------------------------------------------------------------
def test_pasr_hand_case():
    """One reacting species: tau_c = rho Y / |omega|; k/eps = 4 s, nu/eps = 1 s^2 -> tau_mix = sqrt(4 * 1) = 2 s."""
    from oracle import oracle
    om = oracle.Mech(helpers.tiny_mech(2, W=[28.96, 28.96]))
    T, p = np.array([600.0]), np.array([P0])
    Y = np.array([[0.25], [0.75]])
    rho = P0 * 28.96 / (R * 600.0)
    eps = 0.5
    mu = np.array([rho * 1.0 * eps])             # nu / eps = 1
    ksgs = np.array([4.0 * eps])                 # k / eps = 4
    omega = np.array([[-rho * 0.25 / 6.0], [0.0]])   # tau_c = 6 s (the non-reacting species does not count)
    out, kappa = om.pasr(T, p, Y, mu, ksgs, np.array([eps]), 500.0, omega)
    assert np.isclose(kappa[0], 6.0 / (6.0 + 2.0), rtol=1e-13)
    assert np.allclose(out, 0.75 * omega, rtol=1e-13)


def test_pasr_gate_zero_source_limits_and_brute_force(case):
    mech, om, cells = case
    rng = np.random.default_rng(7)
    n, K = cells.n, mech.K
    T, p, Y = cells.T.astype(float), cells.p.astype(float), cells.Y.astype(float)
    mu = rng.uniform(1e-5, 8e-5, n)
    ksgs, eps = rng.uniform(0.01, 10.0, n), rng.uniform(0.1, 1e4, n)
    omega = rng.normal(0.0, 50.0, (K, n))
    omega[:, :5] = 0.0                                   # nothing reacts: kappa = 0
    out, kappa = om.pasr(T, p, Y, mu, ksgs, eps, 500.0, omega)
    # slowest species time scale, brute force in numpy
    rho = p / ((Y / mech.W[:, None]).sum(axis=0) * R * T)
    with np.errstate(divide="ignore", invalid="ignore"):
        tau_k = np.where(np.abs(omega) > 0, rho[None, :] * Y / np.abs(omega), 0.0)
    tau_c = tau_k.max(axis=0)
    tau_mix = np.sqrt((ksgs / eps) * np.sqrt(mu / rho / eps))
    ref = np.where((tau_c > 0) & (T >= 500.0), tau_c / (tau_c + tau_mix), 0.0)
    assert np.allclose(kappa, ref, rtol=1e-12, atol=0)
    assert np.allclose(out, ref[None, :] * omega, rtol=1e-12, atol=0)
    assert (kappa[T < 500.0] == 0).all() and (T < 500.0).any()         # the gate
    assert (kappa[:5] == 0).all()
    assert ((kappa >= 0) & (kappa < 1)).all()
    # fast mixing: tau_mix -> 0 leaves the source untouched; slow mixing kills it
    _, k_fast = om.pasr(T, p, Y, mu, ksgs * 1e-30, eps, 0.0, omega)
    assert np.allclose(k_fast[5:], 1.0, atol=1e-6)
    _, k_slow = om.pasr(T, p, Y, mu, ksgs * 1e30, eps, 0.0, omega)
    assert np.all(k_slow < 1e-6)
    # doubling every source halves tau_c: kappa = tau_c/(tau_c + tau_mix) follows
    _, k2 = om.pasr(T, p, Y, mu, ksgs, eps, 0.0, 2.0 * omega)
    t = tau_c[5:]
    assert np.allclose(k2[5:], (t / 2) / (t / 2 + tau_mix[5:]), rtol=1e-12)
