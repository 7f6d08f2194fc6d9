"""The error floor of a 16-bit-operand MLP chain (test infrastructure; A12).

north_star gives 2e-2 for the ANN dY on the "bf16 path".  Whether a given species can meet the element-wise form of
that bound (|d| <= 2e-2 (|ref| + RMS_cells(ref_k))) is decided by arithmetic the kernel cannot
influence: every 16-bit-operand chain rounds the features and the three hidden activations to 16 bits, and for a
species whose net change dY_k = dY*_k - Y_k (S - 1) is a small difference of two larger terms that rounding noise
alone can exceed 2e-2 of the species' scale.  `ideal_chain_source` evaluates the chain the way an *ideal*
implementation of the stated precision would: everything in fp64 exactly as the oracle does (exact erf GELU, A13),
except that the features and each hidden activation are rounded once, to nearest-even, to the 16-bit format, and
each pre-activation once to fp32 (the accumulator).  Its error against the oracle is the floor; the GPU parity
tests bound the kernel by max(2e-2, 1.25 x floor) per species (helpers.tol_16bit) and by 2e-2 normwise, flat.

With fmt=None nothing is rounded and the function must reproduce oracle.Ann.source to rounding level: that is its
pin (tests/test_tolerance_floor.py), so a slip in this restatement of O9-O12 cannot hide behind "floor".
"""
import numpy as np
from scipy.special import erf

R = 8314.46261815324


def round_bf16(x):
    """fp64 -> nearest-even bf16 value (as fp64)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).astype(np.float64).reshape(np.shape(x))


def _rounder(fmt):
    if fmt is None:
        return lambda a: a
    if fmt == "fp16":
        return lambda a: a.astype(np.float16).astype(np.float64)
    if fmt == "bf16":
        return round_bf16
    raise ValueError(fmt)


def ideal_chain_source_mmlp(mech, nets, T, p, Y, fmt="fp16"):
    """The same floor for K one-output networks (NEXT-1): net k supplies o_k; shared features and epilogue."""
    from types import SimpleNamespace
    K = len(nets)
    outs = []
    for a in nets:
        one = SimpleNamespace(W=a.W, b=a.b, x_mean=a.x_mean, x_std=a.x_std, u_mean=np.zeros(1), u_std=np.ones(1),
                              boxcox_lambda=a.boxcox_lambda, dt=a.dt)
        outs.append(_chain_outputs(one, T, p, Y, fmt, K)[:, 0])
    o = np.stack(outs, axis=1)
    u_mean = np.array([float(np.asarray(a.u_mean).ravel()[0]) for a in nets])
    u_std = np.array([float(np.asarray(a.u_std).ravel()[0]) for a in nets])
    return _epilogue(mech, nets[0].boxcox_lambda, nets[0].dt, u_mean, u_std, o, T, p, Y)


def _chain_outputs(ann, T, p, Y, fmt, K):
    rnd = _rounder(fmt)
    acc = (lambda z: z) if fmt is None else (lambda z: z.astype(np.float32).astype(np.float64))
    lam = float(ann.boxcox_lambda)
    Y = np.asarray(Y, np.float64)
    T = np.asarray(T, np.float64)
    p = np.asarray(p, np.float64)
    n = T.shape[0]
    Yt = Y[:K, :n].T
    x = np.empty((n, K + 2))
    x[:, 0] = (T - ann.x_mean[0]) / ann.x_std[0]
    x[:, 1] = (p - ann.x_mean[1]) / ann.x_std[1]
    x[:, 2:] = ((Yt ** lam - 1.0) / lam - np.asarray(ann.x_mean)[2:]) / np.asarray(ann.x_std)[2:]
    a = rnd(x)
    for l in range(len(ann.W) - 1):
        z = acc(a @ np.asarray(ann.W[l], np.float64).T + np.asarray(ann.b[l], np.float64))
        a = rnd(0.5 * z * (1.0 + erf(z / np.sqrt(2.0))))
    return a @ np.asarray(ann.W[-1], np.float64).T + np.asarray(ann.b[-1], np.float64)


def _epilogue(mech, lam, dt, u_mean, u_std, o, T, p, Y):
    lam = float(lam)
    T = np.asarray(T, np.float64)
    p = np.asarray(p, np.float64)
    n = T.shape[0]
    Yt = np.asarray(Y, np.float64)[:, :n].T
    delta = u_std * o + u_mean
    Ys = np.maximum(Yt ** lam + lam * delta, 0.0) ** (1.0 / lam)
    dY = Ys / Ys.sum(axis=1, keepdims=True) - Yt
    rho = p / ((Yt / np.asarray(mech.W)).sum(axis=1) * R * T)
    return (rho[:, None] * dY / float(dt)).T.copy(), dY.T.copy()


def ideal_chain_source(mech, ann, T, p, Y, fmt="fp16"):
    """(omega[K, n], dY[K, n]) of O9-O12 with 16-bit rounding of features/activations only (fmt: fp16|bf16|None)."""
    rnd = _rounder(fmt)
    acc = (lambda z: z) if fmt is None else (lambda z: z.astype(np.float32).astype(np.float64))
    lam = float(ann.boxcox_lambda)
    Y = np.asarray(Y, np.float64)
    T = np.asarray(T, np.float64)
    p = np.asarray(p, np.float64)
    n = T.shape[0]
    Yt = Y[:, :n].T                                             # [n, K]
    K = Yt.shape[1]
    x = np.empty((n, K + 2))
    x[:, 0] = (T - ann.x_mean[0]) / ann.x_std[0]                # x = {T, p, F(Y)}, z-scored (A8)
    x[:, 1] = (p - ann.x_mean[1]) / ann.x_std[1]
    x[:, 2:] = ((Yt ** lam - 1.0) / lam - np.asarray(ann.x_mean)[2:]) / np.asarray(ann.x_std)[2:]
    a = rnd(x)
    nl = len(ann.W)
    for l in range(nl - 1):
        z = acc(a @ np.asarray(ann.W[l], np.float64).T + np.asarray(ann.b[l], np.float64))
        a = rnd(0.5 * z * (1.0 + erf(z / np.sqrt(2.0))))       # exact GELU (A13), one rounding
    o = a @ np.asarray(ann.W[-1], np.float64).T + np.asarray(ann.b[-1], np.float64)
    delta = np.asarray(ann.u_std) * o + np.asarray(ann.u_mean)  # A9
    Ys = np.maximum(Yt ** lam + lam * delta, 0.0) ** (1.0 / lam)   # A10
    dY = Ys / Ys.sum(axis=1, keepdims=True) - Yt                # A11
    rho = p / ((Yt / np.asarray(mech.W)).sum(axis=1) * R * T)   # A17
    omega = rho[:, None] * dY / float(ann.dt)
    return omega.T.copy(), dY.T.copy()
