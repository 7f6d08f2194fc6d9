"""Pins P1-P4 (+ textbook magnitudes) for the oracle's NASA-7 / Newton functions O1-O3.

The paper prints no formula or worked example for this step (PAPER.md:34-36 only says the
properties are computed on the GPU), so the oracle is pinned by closed forms, calculus
identities and invariants, chosen so a dropped term, a wrong divisor (1/2..1/5), a swapped
range or a wrong R or W fails at least one of them.
"""
import numpy as np
import pytest

from oracle import oracle
from tests.helpers import R, read_textbook, tiny_mech


def test_p2_cp_is_dh_dT_and_ds_dT(cfg1, omech1):
    """P2: cp = dh/dT and cp/T = ds/dT by central differences, both ranges, every species."""
    mech = cfg1[0]
    for k in range(mech.K):
        for T in (350.0, 640.0, 999.0, 1001.0, 1700.0, 3300.0):
            dT = 1e-2
            cp, h, s = omech1.species_thermo(k, T)
            _, hp, sp = omech1.species_thermo(k, T + dT)
            _, hm, sm = omech1.species_thermo(k, T - dT)
            assert abs((hp - hm) / (2 * dT) - cp) <= 1e-7 * cp
            assert abs((sp - sm) / (2 * dT) - cp / T) <= 1e-6 * cp / T


def test_p3_continuity_at_T_mid(cfg1, omech1):
    """P3 / A2: cp, dcp/dT, h, s continuous across 1000 K (the generator matches them)."""
    mech = cfg1[0]
    e = 1e-7
    for k in range(mech.K):
        lo = omech1.species_thermo(k, 1000.0 - e)
        hi = omech1.species_thermo(k, 1000.0 + e)
        at = omech1.species_thermo(k, 1000.0)
        for a, b in zip(lo, hi):
            assert abs(a - b) <= 1e-8 * max(abs(a), 1.0)
        # T == T_mid takes the `hi` set (A2): compare with the hi-side polynomial evaluated by numpy
        a_hi = mech.nasa_hi[k]
        cp_hi = R * np.polynomial.polynomial.polyval(1000.0, a_hi[:5])
        assert abs(at[0] - cp_hi) <= 1e-12 * cp_hi
        # slope continuity
        d = 1e-3
        s_lo = (omech1.species_thermo(k, 1000.0 - e)[0] - omech1.species_thermo(k, 1000.0 - e - d)[0]) / d
        s_hi = (omech1.species_thermo(k, 1000.0 + e + d)[0] - omech1.species_thermo(k, 1000.0 + e)[0]) / d
        assert abs(s_lo - s_hi) <= 1e-4 * max(abs(s_lo), 1.0)


def test_range_selection_uses_lo_below_and_hi_above():
    """A2: distinct constant cp in the two ranges -> which set is used is observable."""
    lo = np.zeros((1, 7)); lo[0, 0] = 3.0
    hi = np.zeros((1, 7)); hi[0, 0] = 4.0
    m = oracle.Mech(tiny_mech(1, W=[10.0], a_lo=lo, a_hi=hi))
    assert m.species_thermo(0, 999.999)[0] == pytest.approx(3.0 * R, rel=1e-15)
    assert m.species_thermo(0, 1000.0)[0] == pytest.approx(4.0 * R, rel=1e-15)
    assert m.species_thermo(0, 250.0)[0] == pytest.approx(3.0 * R, rel=1e-15)   # A3: extrapolate, no clamp
    assert m.species_thermo(0, 4000.0)[0] == pytest.approx(4.0 * R, rel=1e-15)


def test_textbook_helium_cp():
    val, tol = read_textbook()["helium_cp_mass"]
    lo = np.zeros((1, 7)); lo[0, 0] = 2.5
    m = oracle.Mech(tiny_mech(1, W=[4.002602], a_lo=lo))
    Y = np.ones((1, 1))
    cp, h = m.mixture_cp_h(np.array([300.0]), Y)
    assert abs(cp[0] - val) <= tol * val
    # and h = cp T for a6 = 0
    assert h[0] == pytest.approx(cp[0] * 300.0, rel=1e-14)


def test_p4_monatomic_closed_form_one_step():
    """P4: a1 = 2.5, a2..a5 = 0  =>  T = (h W/R - a6)/2.5 exactly, Newton converges in one step."""
    lo = np.zeros((2, 7)); lo[:, 0] = 2.5; lo[0, 5] = -1234.5; lo[1, 5] = 987.0
    W = np.array([4.0, 40.0])
    m = oracle.Mech(tiny_mech(2, W=W, a_lo=lo))
    # pure species 0
    Y = np.array([[1.0], [0.0]])
    h_in = np.array([3.1e6])
    T, it = m.T_from_h(h_in, Y, np.array([700.0]), return_iters=True)
    assert T[0] == pytest.approx((h_in[0] * W[0] / R - lo[0, 5]) / 2.5, rel=1e-14)
    assert it[0] <= 2          # one step + the step that sees |delta| < 1e-9
    # mixture: h = sum Y_k R/W_k (2.5 T + a6_k)  (linear in T)
    Y = np.array([[0.3], [0.7]])
    c1 = np.sum(Y[:, 0] * R / W * 2.5)
    c0 = np.sum(Y[:, 0] * R / W * lo[:, 5])
    T = m.T_from_h(h_in, Y, np.array([2000.0]))
    assert T[0] == pytest.approx((h_in[0] - c0) / c1, rel=1e-13)


def test_p4_linear_cp_quadratic_root():
    """P4: cp/R = a1 + a2 T  =>  h W/R = a1 T + a2 T^2/2 + a6, root by the quadratic formula."""
    lo = np.zeros((1, 7)); lo[0, 0] = 3.0; lo[0, 1] = 1e-3; lo[0, 5] = -500.0
    W = 20.0
    m = oracle.Mech(tiny_mech(1, W=[W], a_lo=lo))
    h_in = 1.4e6
    c = lo[0, 5] - h_in * W / R
    T_exact = (-3.0 + np.sqrt(9.0 - 4 * 0.5e-3 * c)) / (2 * 0.5e-3)
    for guess in (300.0, 1000.0, 3000.0):
        T = m.T_from_h(np.array([h_in]), np.ones((1, 1)), np.array([guess]))
        assert T[0] == pytest.approx(T_exact, abs=1e-8)


def test_p1_round_trip(cfg1, omech1):
    """P1: T_from_h(h(T0,Y),Y) = T0 from warm, cold and far guesses; h(T_from_h(h0,Y),Y) = h0."""
    mech, _, cells = cfg1
    n = 512
    T0 = cells.T[:n].astype(np.float64)
    Y = cells.Y[:, :n]
    cp, h = omech1.mixture_cp_h(T0, Y)
    for guess in (cells.T_guess[:n], np.full(n, 1000.0), np.full(n, 250.0), np.full(n, 3500.0),
                  np.full(n, np.nan), np.full(n, -5.0)):
        T = omech1.T_from_h(h, Y, guess)
        assert np.max(np.abs(T - T0)) <= 1e-8
        _, h2 = omech1.mixture_cp_h(T, Y)
        assert np.max(np.abs(h2 - h) / (cp * T0)) <= 1e-10


def test_one_hot_reduces_to_species(cfg1, omech1):
    """P5 (thermo part): Y = e_k  =>  cp = cp_k/W_k, h = h_k/W_k."""
    mech = cfg1[0]
    for k in range(mech.K):
        Y = np.zeros((mech.K, 1)); Y[k] = 1.0
        for T in (400.0, 1500.0):
            cp, h = omech1.mixture_cp_h(np.array([T]), Y)
            ck, hk, _ = omech1.species_thermo(k, T)
            assert cp[0] == pytest.approx(ck / mech.W[k], rel=1e-14)
            assert h[0] == pytest.approx(hk / mech.W[k], rel=1e-14)


def test_mixture_is_mass_weighted_sum(cfg1, omech1):
    """O2: linear in Y -- cp(aY1 + bY2) = a cp(Y1) + b cp(Y2) (catches mole/mass mix-ups)."""
    mech, _, cells = cfg1
    T = np.array([1234.0])
    Y1 = cells.Y[:, 0:1].astype(np.float64)
    Y2 = cells.Y[:, 1:2].astype(np.float64)
    c1, h1 = omech1.mixture_cp_h(T, Y1)
    c2, h2 = omech1.mixture_cp_h(T, Y2)
    c3, h3 = omech1.mixture_cp_h(T, 0.3 * Y1 + 0.7 * Y2)
    assert c3[0] == pytest.approx(0.3 * c1[0] + 0.7 * c2[0], rel=1e-13)
    assert h3[0] == pytest.approx(0.3 * h1[0] + 0.7 * h2[0], rel=1e-12, abs=1e-6)


def test_generator_cp_bounds(cfg1, omech1):
    """Generator property A3 relies on: cp_k/R in [2.5, 8] on [300, 3500] K and >= 2 on [200, 4000] K."""
    mech = cfg1[0]
    for k in range(mech.K):
        for T in np.linspace(200.0, 4000.0, 77):
            cpR = omech1.species_thermo(k, T)[0] / R
            assert cpR >= 2.0
            if 300.0 <= T <= 3500.0:
                assert 2.5 - 1e-9 <= cpR <= 8.0 + 1e-9
