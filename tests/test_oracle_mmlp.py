"""Pins of the oracle's per-species-MLP source (NEXT-1): it must be nothing more than K calls of the
already pinned mlp_forward on one-output networks, followed by the already pinned epilogue of cell_source."""
import numpy as np
import pytest

from tests import helpers


def split_into_single_output_nets(ann):
    """The K-output network `ann` as K one-output networks with the same hidden layers: mathematically the same map."""
    from types import SimpleNamespace
    K = ann.dims[-1]
    nets = []
    for k in range(K):
        W = [w.copy() for w in ann.W[:-1]] + [ann.W[-1][k:k + 1].copy()]
        b = [x.copy() for x in ann.b[:-1]] + [ann.b[-1][k:k + 1].copy()]
        nets.append(SimpleNamespace(dims=list(ann.dims[:-1]) + [1], W=W, b=b, precision=ann.precision, x_mean=ann.x_mean,
                                    x_std=ann.x_std, u_mean=np.asarray(ann.u_mean)[k:k + 1], u_std=np.asarray(ann.u_std)[k:k + 1],
                                    boxcox_lambda=ann.boxcox_lambda, dt=ann.dt))
    return nets


def test_mmlp_of_a_split_network_equals_the_single_network(cfg1, omech1):
    """Strongest pin: slicing a K-output net's last layer into K one-output nets must reproduce cell_source exactly
    (same arithmetic, operation for operation)."""
    from oracle import oracle
    mech, ann, cells = cfg1
    idx = slice(0, 300)
    om1, dY1 = oracle.Ann(ann).source(omech1, cells.T[idx], cells.p[idx], np.ascontiguousarray(cells.Y[:, idx]))
    om2, dY2 = oracle.Mmlp(split_into_single_output_nets(ann)).source(omech1, cells.T[idx], cells.p[idx],
                                                                      np.ascontiguousarray(cells.Y[:, idx]))
    assert np.array_equal(om1, om2) and np.array_equal(dY1, dY2)


def test_mmlp_two_species_constant_nets_hand_case():
    """K = 2, zero weights, last biases (0.3, -0.2): Delta_k = u_std_k o_k + u_mean_k, Y*_k = (Y_k^lam + lam Delta_k)^(1/lam),
    renormalised; the numbers below are that closed form written out."""
    from oracle import oracle
    lam, dt = 0.1, 1e-6
    mech = helpers.tiny_mech(2, W=[2.0, 32.0])
    nets = []
    for k, (o, um, us) in enumerate(((0.3, 0.01, 0.05), (-0.2, -0.02, 0.1))):
        dims = [4, 3, 1]
        nets.append(helpers.tiny_ann(dims, W=[np.zeros((3, 4), np.float32), np.zeros((1, 3), np.float32)],
                                     b=[np.zeros(3, np.float32), np.array([o], np.float32)], u_mean=[um], u_std=[us], lam=lam, dt=dt))
    Y = np.array([[0.3], [0.7]])
    T, p = np.array([1200.0]), np.array([101325.0])
    om, dY = oracle.Mmlp(nets).source(oracle.Mech(mech), T, p, Y)
    d = np.array([0.05 * float(np.float32(0.3)) + 0.01, 0.1 * float(np.float32(-0.2)) - 0.02])   # biases are fp32 values
    Ys = (Y[:, 0] ** lam + lam * d) ** (1 / lam)
    ref = Ys / Ys.sum() - Y[:, 0]
    rho = 101325.0 / ((0.3 / 2.0 + 0.7 / 32.0) * helpers.R * 1200.0)
    assert np.allclose(dY[:, 0], ref, rtol=1e-12, atol=0)
    assert np.allclose(om[:, 0], rho * ref / dt, rtol=1e-12, atol=0)
    assert abs((Y[:, 0] + dY[:, 0]).sum() - 1.0) < 1e-14


def test_mmlp_against_numpy_matmul_per_net():
    """Random small nets: every net's output recomputed with numpy `@` and scipy's erf, then the plain epilogue."""
    from scipy.special import erf
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    K, n = 5, 40
    mech = synth.make_mechanism(K, 9)
    nets = synth.make_mmlp(K, [12, 7], 0, 9)
    cells = synth.cells_dirichlet(K, n, 9)
    om, dY = oracle.Mmlp(nets).source(oracle.Mech(mech), cells.T, cells.p, cells.Y)
    lam = 0.1
    Y = cells.Y.astype(np.float64).T
    x = np.empty((n, K + 2))
    x[:, 0] = (cells.T - nets[0].x_mean[0]) / nets[0].x_std[0]
    x[:, 1] = (cells.p - nets[0].x_mean[1]) / nets[0].x_std[1]
    x[:, 2:] = ((Y ** lam - 1) / lam - nets[0].x_mean[2:]) / nets[0].x_std[2:]
    delta = np.empty((n, K))
    for k, a in enumerate(nets):
        h = x
        for l in range(2):
            z = h @ a.W[l].astype(np.float64).T + a.b[l]
            h = 0.5 * z * (1 + erf(z / np.sqrt(2)))
        delta[:, k] = a.u_std[0] * (h @ a.W[2].astype(np.float64).T + a.b[2])[:, 0] + a.u_mean[0]
    Ys = np.maximum(Y ** lam + lam * delta, 0) ** (1 / lam)
    ref = Ys / Ys.sum(1, keepdims=True) - Y
    assert np.allclose(dY.T, ref, rtol=1e-10, atol=1e-16)
    assert np.abs((Y + dY.T).sum(1) - 1).max() < 1e-14
