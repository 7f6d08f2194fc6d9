"""Pins P10-P15 for the oracle's ANN functions O9-O12.

P:79 gives the inputs {T, p, F(Y)}, the output "change in species mass fraction over a given
time step", Z-score normalisation, the 1600/800/400 GELU body; P:62 the 1 us step; P:86 the
mass-fraction-unity principle.  The Box-Cox formula/lambda and the output reading are A8-A11.
"""
import numpy as np
import pytest
import torch
from scipy.stats import norm

from oracle import oracle
from tests.helpers import R, const_output_ann, read_textbook, tiny_ann, tiny_mech


def test_p10_boxcox_values_and_inverse():
    lam = 0.1
    assert oracle.boxcox(1.0, lam) == 0.0
    assert oracle.boxcox(0.0, lam) == -10.0
    assert oracle.boxcox(1e-20, lam) == pytest.approx(-9.9, rel=1e-14)
    assert oracle.boxcox(1e-10, lam) == pytest.approx(-9.0, rel=1e-14)
    for y in (1e-30, 1e-12, 3e-4, 0.2, 1.0):
        assert oracle.boxcox_inv(oracle.boxcox(y, lam), lam) == pytest.approx(y, rel=1e-11)
    # Box & Cox: the transform tends to ln(y) as lambda -> 0
    for y in (1e-3, 0.5, 2.0):
        assert oracle.boxcox(y, 1e-9) == pytest.approx(np.log(y), rel=1e-6, abs=1e-7)
    # lambda = 1 is a shift: F(y) = y - 1
    assert oracle.boxcox(0.25, 1.0) == pytest.approx(-0.75, rel=1e-15)


def test_p11_gelu_values():
    tb = read_textbook()
    assert oracle.gelu(0.0) == 0.0
    for name, x in (("gelu_1", 1.0), ("gelu_m1", -1.0), ("gelu_2", 2.0)):
        v, tol = tb[name]
        assert oracle.gelu(x) == pytest.approx(v, rel=max(tol, 1e-15))
    for x in np.linspace(-6, 6, 49):
        assert oracle.gelu(x) == pytest.approx(x * norm.cdf(x), rel=1e-12, abs=1e-300)   # x Phi(x)
        assert oracle.gelu(x) - oracle.gelu(-x) == pytest.approx(x, rel=1e-13, abs=1e-15)


def test_p12_mlp_against_numpy_and_torch():
    """P12: naive loops vs numpy `@` and vs torch.nn.functional (fp64), three hidden layers."""
    dims = [7, 13, 11, 5, 3]
    a = tiny_ann(dims, seed=4)
    o = oracle.Ann(a)
    rng = np.random.default_rng(0)
    x = rng.normal(0, 1.5, (17, dims[0]))
    got = o.mlp(x)
    cur = x.copy()
    for l in range(4):
        cur = cur @ a.W[l].astype(np.float64).T + a.b[l].astype(np.float64)
        if l < 3:
            cur = cur * norm.cdf(cur)
    assert np.allclose(got, cur, rtol=1e-12, atol=1e-14)
    t = torch.from_numpy(x)
    for l in range(4):
        t = torch.nn.functional.linear(t, torch.from_numpy(a.W[l]).double(), torch.from_numpy(a.b[l]).double())
        if l < 3:
            t = torch.nn.functional.gelu(t)           # erf form
    assert np.allclose(got, t.numpy(), rtol=1e-12, atol=1e-14)


def test_p12_mlp_zero_weights_and_identity():
    dims = [4, 4, 4]
    # zero weights -> output = last bias; hidden bias irrelevant
    a = tiny_ann(dims, W=[np.zeros((4, 4), np.float32)] * 2,
                 b=[np.ones(4, np.float32), np.array([1, -2, 3, 0.5], np.float32)])
    assert np.array_equal(oracle.Ann(a).mlp(np.ones((2, 4))), np.tile([1, -2, 3, 0.5], (2, 1)))
    # identity weights, zero bias: out_j = GELU(x_j); W[l] is [out][in]: a permutation matrix makes the
    # orientation observable: W0[o, i] = 1 iff i == (o+1) % 4  =>  hidden_o = GELU(x_{(o+1)%4})
    P = np.zeros((4, 4), np.float32)
    for o_ in range(4):
        P[o_, (o_ + 1) % 4] = 1
    a = tiny_ann(dims, W=[P, np.eye(4, dtype=np.float32)], b=[np.zeros(4, np.float32)] * 2)
    x = np.array([[0.0, 1.0, -1.0, 2.0]])
    tb = read_textbook()
    expect = [tb["gelu_1"][0], tb["gelu_m1"][0], tb["gelu_2"][0], 0.0]
    assert np.allclose(oracle.Ann(a).mlp(x)[0], expect, rtol=1e-15)


def test_o9_features_hand_values():
    """O9 / A8: T and p raw, Box-Cox on Y only, then z-score; order T, p, Y_0.."""
    K = 2
    a = tiny_ann([K + 2, 3, K], x_mean=[1000.0, 1e5, -5.0, -9.0], x_std=[500.0, 1e4, 2.0, 0.5])
    Y = np.array([[1.0], [1e-10]])
    f = oracle.Ann(a).features(np.array([1500.0]), np.array([1.2e5]), Y)
    assert np.allclose(f[0], [1.0, 2.0, (0.0 + 5.0) / 2.0, (-9.0 + 9.0) / 0.5], rtol=1e-13, atol=1e-13)


def test_p13_zero_output_gives_zero_source():
    K = 4
    mech = oracle.Mech(tiny_mech(K, W=[2.0, 18.0, 28.0, 44.0]))
    ann = oracle.Ann(const_output_ann(K, np.zeros(K)))
    rng = np.random.default_rng(1)
    Y = np.ascontiguousarray(rng.dirichlet(np.ones(K), 5).T)
    om, dY = ann.source(mech, np.full(5, 1200.0), np.full(5, 101325.0), Y)
    assert np.max(np.abs(dY)) <= 4e-16
    assert np.max(np.abs(om)) <= 4e-16 * 1.0 / 1e-6


def test_p14_unity_and_sum_omega():
    """P14 / A11: sum Y' = 1 and sum omega = rho (1 - sum Y)/dt for any weights, any (unnormalised) Y."""
    K = 6
    W = np.array([2.0, 16.0, 18.0, 28.0, 32.0, 44.0])
    mech = oracle.Mech(tiny_mech(K, W=W))
    a = tiny_ann([K + 2, 9, 8, K], seed=7, u_std=np.full(K, 0.05), x_mean=np.r_[1200, 101325, np.full(K, -4.0)],
                 x_std=np.r_[500, 1.0, np.full(K, 2.0)])
    ann = oracle.Ann(a)
    rng = np.random.default_rng(2)
    n = 33
    Y = np.ascontiguousarray(rng.dirichlet(np.full(K, 0.5), n).T) * rng.uniform(0.97, 1.03, n)
    T = rng.uniform(500, 2200, n); p = np.full(n, 101325.0)
    om, dY = ann.source(mech, T, p, Y)
    assert np.max(np.abs((Y + dY).sum(0) - 1.0)) <= 1e-14
    rho = p / (R * T * np.sum(Y / W[:, None], axis=0))
    assert np.allclose(om.sum(0), rho * (1.0 - Y.sum(0)) / 1e-6, rtol=1e-9, atol=1e-6)
    assert np.any(np.abs(dY) > 1e-6)     # the network does something


def test_p15_small_delta_linearisation_and_scales():
    """P15: only species k perturbed by a small Delta: Y*_k ~ Y_k + eps, eps = Y_k^{1-lambda} Delta;
    after Y' = Y*/sum: dY_k = eps (1 - Y_k)/(1 + eps), dY_j = -Y_j eps/(1 + eps).  Also pins
    Delta = u_std o + u_mean and omega = rho dY/dt with the textbook air density."""
    K = 3
    W = np.array([28.96, 28.96, 28.96])
    mech = oracle.Mech(tiny_mech(K, W=W))
    lam, dt = 0.1, 1e-6
    Yv = np.array([0.2, 0.5, 0.3])
    out = np.array([0.0, 2.0, 0.0])
    a = const_output_ann(K, out, lam=lam, dt=dt, u_std=[1.0, 1e-7, 1.0], u_mean=[0.0, 3e-7, 0.0])
    Delta = 1e-7 * 2.0 + 3e-7
    eps_exact = (Yv[1] ** lam + lam * Delta) ** (1 / lam) - Yv[1]
    eps_lin = Yv[1] ** (1 - lam) * Delta
    assert eps_exact == pytest.approx(eps_lin, rel=1e-5)
    om, dY = oracle.Ann(a).source(mech, np.array([300.0]), np.array([101325.0]), Yv.reshape(3, 1).copy())
    assert dY[1, 0] == pytest.approx(eps_lin * (1 - Yv[1]) / (1 + eps_lin), rel=1e-5)
    assert dY[0, 0] == pytest.approx(-Yv[0] * eps_lin / (1 + eps_lin), rel=1e-5)
    assert dY[2, 0] == pytest.approx(-Yv[2] * eps_lin / (1 + eps_lin), rel=1e-5)
    rho_tb, tol = read_textbook()["air_density_300K_1atm"]
    assert np.allclose(om[:, 0] * dt / dY[:, 0], rho_tb, rtol=tol)


def test_a10_clamp_and_zero_mass_fraction():
    """A10: base clamped at 0 (trace species, Delta < 0) and Y_k = 0 with Delta > 0 gives (lambda Delta)^{1/lambda}."""
    K = 3
    mech = oracle.Mech(tiny_mech(K))
    lam = 0.1
    a = const_output_ann(K, [-1.0, 0.5, 0.0], lam=lam)
    Y = np.array([[1e-20], [0.0], [1.0]])
    om, dY = oracle.Ann(a).source(mech, np.array([1000.0]), np.array([101325.0]), Y)
    ystar = np.array([0.0, (lam * 0.5) ** (1 / lam), 1.0])
    yprime = ystar / ystar.sum()
    assert np.allclose(dY[:, 0], yprime - Y[:, 0], rtol=1e-12, atol=1e-30)
    assert np.all(np.isfinite(om))


def test_source_brute_force_against_definition():
    """P16: the whole O9-O12 chain against an independent numpy/scipy evaluation on a tiny case."""
    K = 3
    W = np.array([2.0, 28.0, 44.0])
    mech_t = tiny_mech(K, W=W)
    a = tiny_ann([K + 2, 6, 5, K], seed=11, x_mean=[1000, 101325, -3, -4, -5], x_std=[400, 1, 1.5, 2, 2.5],
                 u_mean=[0.001, -0.002, 0.0], u_std=[0.03, 0.05, 0.07])
    rng = np.random.default_rng(5)
    n = 9
    Y = np.ascontiguousarray(rng.dirichlet(np.ones(K), n).T)
    T = rng.uniform(400, 2400, n); p = np.full(n, 101325.0)
    om, dY = oracle.Ann(a).source(oracle.Mech(mech_t), T, p, Y)
    lam = a.boxcox_lambda
    F = (Y ** lam - 1) / lam
    f = np.vstack([T, p, F]).T
    f = (f - a.x_mean) / a.x_std
    cur = f
    for l in range(3):
        cur = cur @ a.W[l].astype(np.float64).T + a.b[l]
        if l < 2:
            cur = cur * norm.cdf(cur)
    Delta = cur * a.u_std + a.u_mean                   # [n, K]
    Ystar = np.maximum(Y.T ** lam + lam * Delta, 0) ** (1 / lam)
    Yp = Ystar / Ystar.sum(1, keepdims=True)
    dY_ref = (Yp - Y.T).T
    rho = p / (R * T * np.sum(Y / W[:, None], axis=0))
    assert np.allclose(dY, dY_ref, rtol=1e-10, atol=1e-16)
    assert np.allclose(om, rho * dY_ref / a.dt, rtol=1e-10, atol=1e-9)
