"""Seeded synthetic inputs for the per-cell thermochemistry update.

This module serves BOTH the CUDA path and the oracle and therefore holds none of the
method's arithmetic: it builds *tables* (NASA-7 coefficients, transport fit coefficients,
MLP weights, normalisation statistics) and *cell fields* (T, p, Y, guesses) from a seed.
Anything the method derives from them (h(T,Y), Box-Cox features, properties) is computed
by whoever consumes the inputs -- the oracle in tests, the kernels in bench.py.

The DRM19 mechanism, the trained ANN weights and the SWB5 LES fields of the paper
 are not available; these stand-ins follow BASELINE.json `configs`
and SURVEY.md section 8(d): 2.5 M-cell-scale fields, ~20 species
(PAPER.md:44), ambient pressure and three-stream stratification,
flame structure parameterised by a progress variable, dt = 1 us
(PAPER.md:62), hidden layers 1600-800-400.

Everything is numpy, fp64 for tables, fields rounded once to fp32.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np

R_UNIVERSAL = 8314.46261815324      # J/(kmol K), CODATA-2018 exact
N_AVOGADRO = 6.02214076e26          # 1/kmol
K_BOLTZMANN = 1.380649e-23          # J/K
BASE_SEED = 231205800               # + config number

T_LOW, T_MID, T_HIGH = 300.0, 1000.0, 3500.0


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64([int(seed), int(stream)]))


# --------------------------------------------------------------------------------------
# tables
# --------------------------------------------------------------------------------------
@dataclass
class Mechanism:
    """Species tables in the layout include/df_thermo.h::df_mech_create takes (all fp64)."""
    K: int
    W: np.ndarray            # [K] kg/kmol
    nasa_lo: np.ndarray      # [K,7]
    nasa_hi: np.ndarray      # [K,7]
    T_low: float
    T_mid: float
    T_high: float
    visc_fit: np.ndarray     # [K,5]   sqrt(mu_k) = T^(1/4) sum_m b_m (ln T)^m
    cond_fit: np.ndarray     # [K,5]   lambda_k  = T^(1/2) sum_m c_m (ln T)^m
    bdiff_fit: np.ndarray    # [K,K,5] p D_jk    = T^(3/2) sum_m d_m (ln T)^m
    sigma: np.ndarray = field(default=None)     # [K] Angstrom (generator bookkeeping)
    eps_over_k: np.ndarray = field(default=None)  # [K] K


def _cp_quartics(rng: np.random.Generator) -> Tuple[np.ndarray, np.ndarray]:
    """One species' cp/R as two quartics in theta = T/1000 (low, high), C0/C1 matched at theta=1."""
    nodes_lo = np.array([0.2, 0.4, 0.6, 0.8, 1.0])
    theta_chk_lo = np.linspace(0.3, 1.0, 141)
    theta_chk_hi = np.linspace(1.0, 3.5, 251)
    theta_ext_lo = np.linspace(0.2, 0.3, 21)
    theta_ext_hi = np.linspace(3.5, 4.0, 51)
    while True:
        v = np.empty(5)
        v[0] = rng.uniform(2.5, 4.5)
        v[1:] = v[0] + np.cumsum(rng.uniform(0.0, 0.6, 4))
        c = np.linalg.solve(np.vander(nodes_lo, 5, increasing=True), v)
        p1 = v[4]
        dp1 = float(np.sum(np.arange(1, 5) * c[1:]))
        hi_nodes = np.array([1.8, 2.6, 3.5])
        hv = p1 + np.cumsum(rng.uniform(0.0, 0.8, 3))
        A = np.zeros((5, 5))
        rhs = np.zeros(5)
        A[0] = 1.0                                  # q(1) = p(1)
        rhs[0] = p1
        A[1] = np.arange(5)                         # q'(1) = p'(1)
        rhs[1] = dp1
        A[2:] = np.vander(hi_nodes, 5, increasing=True)
        rhs[2:] = hv
        d = np.linalg.solve(A, rhs)
        plo = np.polynomial.polynomial.polyval
        lo_nom = plo(theta_chk_lo, c)
        hi_nom = plo(theta_chk_hi, d)
        if (lo_nom.min() < 2.5 or lo_nom.max() > 8.0 or hi_nom.min() < 2.5 or hi_nom.max() > 8.0):
            continue
        if plo(theta_ext_lo, c).min() < 2.0 or plo(theta_ext_hi, d).min() < 2.0:
            continue
        return c, d


def _nasa_integrals(a: np.ndarray, T: float) -> Tuple[float, float]:
    """(int cp/R dT, int cp/(R T) dT) of a1..a5 at T, without the a6/a7 constants."""
    i_h = a[0] * T + a[1] * T**2 / 2 + a[2] * T**3 / 3 + a[3] * T**4 / 4 + a[4] * T**5 / 5
    i_s = a[0] * np.log(T) + a[1] * T + a[2] * T**2 / 2 + a[3] * T**3 / 3 + a[4] * T**4 / 4
    return float(i_h), float(i_s)


def _omega22(t):
    return 1.16145 * t ** -0.14874 + 0.52487 * np.exp(-0.77320 * t) + 2.16178 * np.exp(-2.43787 * t)


def _omega11(t):
    return (1.06036 * t ** -0.15610 + 0.19300 * np.exp(-0.47635 * t)
            + 1.03587 * np.exp(-1.52996 * t) + 1.76474 * np.exp(-3.89411 * t))


def _fit_lnT(lnT: np.ndarray, y: np.ndarray) -> np.ndarray:
    """Degree-4 least squares in ln T, returned as power-basis coefficients in raw ln T."""
    p = np.polynomial.polynomial.Polynomial.fit(lnT, y, 4)
    return p.convert().coef.astype(np.float64)


def kinetic_theory_viscosity(W, sigma_A, eps_k, T):
    """Chapman-Enskog mu(T) [Pa s] for a Lennard-Jones species (generator physics)."""
    m = W / N_AVOGADRO
    sig = sigma_A * 1e-10
    return (5.0 / 16.0) * np.sqrt(np.pi * m * K_BOLTZMANN * T) / (np.pi * sig**2 * _omega22(T / eps_k))


def kinetic_theory_pD(Wj, Wk, sj_A, sk_A, ej, ek, T):
    """Chapman-Enskog p*D_jk(T) [Pa m^2/s]."""
    mj, mk = Wj / N_AVOGADRO, Wk / N_AVOGADRO
    mjk = mj * mk / (mj + mk)
    sig = 0.5 * (sj_A + sk_A) * 1e-10
    eps = np.sqrt(ej * ek)
    return (3.0 / 16.0) * np.sqrt(2.0 * np.pi * (K_BOLTZMANN * T) ** 3 / mjk) / (np.pi * sig**2 * _omega11(T / eps))


def make_mechanism(K: int, seed: int) -> Mechanism:
    rng = _rng(seed, 1)
    nasa_lo = np.zeros((K, 7))
    nasa_hi = np.zeros((K, 7))
    scale = 1000.0 ** -np.arange(5)
    for k in range(K):
        c, d = _cp_quartics(rng)
        nasa_lo[k, :5] = c * scale
        nasa_hi[k, :5] = d * scale
        h_f = rng.uniform(-3e8, 3e8)          # J/kmol at 298.15 K
        s_0 = rng.uniform(1.3e5, 3e5)         # J/(kmol K) at 298.15 K
        ih, is_ = _nasa_integrals(nasa_lo[k], 298.15)
        nasa_lo[k, 5] = h_f / R_UNIVERSAL - ih
        nasa_lo[k, 6] = s_0 / R_UNIVERSAL - is_
        ih_lo, is_lo = _nasa_integrals(nasa_lo[k], T_MID)
        ih_hi, is_hi = _nasa_integrals(nasa_hi[k], T_MID)
        nasa_hi[k, 5] = nasa_lo[k, 5] + ih_lo - ih_hi
        nasa_hi[k, 6] = nasa_lo[k, 6] + is_lo - is_hi
    W = rng.uniform(2.0, 44.0, K)
    sigma = rng.uniform(2.5, 4.5, K)
    eps = rng.uniform(50.0, 600.0, K)

    Tfit = np.exp(np.linspace(np.log(250.0), np.log(3600.0), 60))
    lnT = np.log(Tfit)
    visc_fit = np.zeros((K, 5))
    cond_fit = np.zeros((K, 5))
    bdiff_fit = np.zeros((K, K, 5))
    for k in range(K):
        mu = kinetic_theory_viscosity(W[k], sigma[k], eps[k], Tfit)
        a = np.where(Tfit[:, None] < T_MID, nasa_lo[k, :5][None, :], nasa_hi[k, :5][None, :])
        cp_molar = R_UNIVERSAL * np.sum(a * Tfit[:, None] ** np.arange(5)[None, :], axis=1)
        lam = mu * (cp_molar + 1.25 * R_UNIVERSAL) / W[k]     # Eucken
        visc_fit[k] = _fit_lnT(lnT, np.sqrt(mu) / Tfit**0.25)
        cond_fit[k] = _fit_lnT(lnT, lam / np.sqrt(Tfit))
        for j in range(k, K):
            pD = kinetic_theory_pD(W[j], W[k], sigma[j], sigma[k], eps[j], eps[k], Tfit)
            cf = _fit_lnT(lnT, pD / Tfit**1.5)
            bdiff_fit[j, k] = cf
            bdiff_fit[k, j] = cf
    return Mechanism(K, W, nasa_lo, nasa_hi, T_LOW, T_MID, T_HIGH, visc_fit, cond_fit, bdiff_fit,
                     sigma, eps)


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round fp32 values to the nearest bf16-representable fp32 (ties to even)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(np.shape(x))


@dataclass
class AnnModel:
    """MLP + normalisation tables in the layout df_ann_create takes."""
    dims: List[int]               # [K+2, ..., K]
    W: List[np.ndarray]           # W[l]: [dims[l+1], dims[l]] fp32 (y = x W^T + b)
    b: List[np.ndarray]           # b[l]: [dims[l+1]] fp32
    precision: int                # 0 = fp32, 1 = bf16 operands / fp32 accumulate
    x_mean: np.ndarray            # [K+2] order T, p, F(Y_0..K-1)
    x_std: np.ndarray
    u_mean: np.ndarray            # [K]
    u_std: np.ndarray
    boxcox_lambda: float
    dt: float


def make_ann(K: int, hidden: List[int], precision: int, seed: int,
             boxcox_lambda: float = 0.1, dt: float = 1e-6) -> AnnModel:
    """Xavier-uniform weights, U(+-1/sqrt(fan_in)) biases, drawn layer by layer."""
    rng = _rng(seed, 2)
    dims = [K + 2] + list(hidden) + [K]
    Ws, bs = [], []
    for l in range(len(dims) - 1):
        fan_in, fan_out = dims[l], dims[l + 1]
        lim = np.sqrt(6.0 / (fan_in + fan_out))
        Wl = rng.uniform(-lim, lim, (fan_out, fan_in)).astype(np.float32)
        bl = rng.uniform(-1.0 / np.sqrt(fan_in), 1.0 / np.sqrt(fan_in), fan_out).astype(np.float32)
        if precision == 1:
            Wl = round_to_bf16(Wl)
        Ws.append(np.ascontiguousarray(Wl))
        bs.append(np.ascontiguousarray(bl))
    # "training-set" statistics: synthetic constants (the real ones come with the trained net).
    x_mean = np.empty(K + 2)
    x_std = np.empty(K + 2)
    x_mean[0], x_std[0] = 1250.0, 550.0
    x_mean[1], x_std[1] = 101325.0, 1.0          # constant feature -> std = 1
    x_mean[2:] = rng.uniform(-5.0, -2.0, K)
    x_std[2:] = rng.uniform(1.0, 2.0, K)
    u_mean = rng.uniform(-0.005, 0.005, K)
    u_std = rng.uniform(0.02, 0.08, K)
    return AnnModel(dims, Ws, bs, precision, x_mean, x_std, u_mean, u_std, boxcox_lambda, dt)


def make_mmlp(K: int, hidden: List[int], precision: int, seed: int, boxcox_lambda: float = 0.1, dt: float = 1e-6) -> List[AnnModel]:
    """One network per species ("individual training and prediction ... for each species mass fraction"):
    K independent (K+2) -> hidden -> 1 networks, Xavier-uniform from one seeded generator (net after net), sharing
    the input statistics; net k carries species k's output statistics as its u_mean[0], u_std[0]."""
    proto = make_ann(K, hidden, precision, seed, boxcox_lambda, dt)      # shared x_mean/x_std, per-species u statistics
    rng = _rng(seed, 5)
    dims = [K + 2] + list(hidden) + [1]
    nets = []
    for k in range(K):
        Ws, bs = [], []
        for l in range(len(dims) - 1):
            fan_in, fan_out = dims[l], dims[l + 1]
            lim = np.sqrt(6.0 / (fan_in + fan_out))
            Wl = rng.uniform(-lim, lim, (fan_out, fan_in)).astype(np.float32)
            bl = rng.uniform(-1.0 / np.sqrt(fan_in), 1.0 / np.sqrt(fan_in), fan_out).astype(np.float32)
            if precision == 1:
                Wl = round_to_bf16(Wl)
            Ws.append(np.ascontiguousarray(Wl))
            bs.append(np.ascontiguousarray(bl))
        nets.append(AnnModel(dims, Ws, bs, precision, proto.x_mean, proto.x_std, proto.u_mean[k:k + 1].copy(),
                             proto.u_std[k:k + 1].copy(), boxcox_lambda, dt))
    return nets


# --------------------------------------------------------------------------------------
# cell fields
# --------------------------------------------------------------------------------------
@dataclass
class Cells:
    """SoA fp32 fields: Y[k, i] with species pitch ld = Y.shape[1] >= n."""
    n: int
    T: np.ndarray          # [n] "true" temperature the state was drawn at
    p: np.ndarray          # [n]
    Y: np.ndarray          # [K, ld]
    T_guess: np.ndarray    # [n] warm Newton guess = T + N(0, 50 K)


def _finish(rng, T, Y, n, ld=None) -> Cells:
    K = Y.shape[0]
    ld = n if ld is None else ld
    Yp = np.zeros((K, ld), dtype=np.float32)
    Yp[:, :n] = Y.astype(np.float32)
    T32 = T.astype(np.float32)
    guess = (T + rng.normal(0.0, 50.0, n)).astype(np.float32)
    p = np.full(n, 101325.0, dtype=np.float32)
    return Cells(n, T32, p, Yp, guess)


def _dirichlet_T(rng, K, n, alpha):
    g = rng.standard_gamma(alpha, size=(K, n))
    g = np.maximum(g, 1e-300)
    return g / g.sum(axis=0, keepdims=True)


def cells_dirichlet(K: int, n: int, seed: int, T_range=(300.0, 2200.0), alpha=0.5, ld=None) -> Cells:
    """cfg1: T ~ U[T_range], p = 101325 Pa, Y ~ Dirichlet(alpha)."""
    rng = _rng(seed, 3)
    T = rng.uniform(T_range[0], T_range[1], n)
    Y = _dirichlet_T(rng, K, n, alpha)
    return _finish(rng, T, Y, n, ld)


def cells_stratified(K: int, n: int, seed: int, ld=None) -> Cells:
    """cfg2-4: Z ~ Beta(2,5), c ~ U[0,1], T = 300 + 1900 c, Y blended along (Z, c)."""
    rng = _rng(seed, 3)
    Yu0, Yu1 = rng.dirichlet(np.full(K, 0.2)), rng.dirichlet(np.full(K, 0.2))
    Yb0, Yb1 = rng.dirichlet(np.full(K, 0.5)), rng.dirichlet(np.full(K, 0.5))
    Z = rng.beta(2.0, 5.0, n)
    c = rng.uniform(0.0, 1.0, n)
    T = 300.0 + 1900.0 * c
    Y = np.empty((K, n), dtype=np.float32)
    for k in range(K):           # row by row keeps the fp64 temporaries at O(n)
        Y[k] = ((1 - c) * ((1 - Z) * Yu0[k] + Z * Yu1[k]) + c * ((1 - Z) * Yb0[k] + Z * Yb1[k]))
    return _finish(rng, T, Y, n, ld)


def cells_robustness(K: int, n: int, seed: int, ld=None) -> Cells:
    """cfg5: T ~ U[250,3500] with 1 % within +-0.5 K of T_mid; 5 % near-pure; 5 % with 1e-20 traces."""
    rng = _rng(seed, 3)
    T = rng.uniform(250.0, 3500.0, n)
    sel = rng.random(n) < 0.01
    T[sel] = T_MID + rng.uniform(-0.5, 0.5, int(sel.sum()))
    Y = _dirichlet_T(rng, K, n, 0.5).astype(np.float32)
    u = rng.random(n)
    pure = np.nonzero(u < 0.05)[0]
    which = rng.integers(0, K, pure.size)
    Y[:, pure] = np.float32(1e-6 / (K - 1)) if K > 1 else np.float32(1.0)
    Y[which, pure] = np.float32(1.0 - 1e-6) if K > 1 else np.float32(1.0)
    trace = np.nonzero((u >= 0.05) & (u < 0.10))[0]
    if trace.size and K > 1:
        mask = rng.random((K, trace.size)) < (1.0 / 3.0)
        mask[rng.integers(0, K, trace.size), np.arange(trace.size)] = False  # keep >= 1 species
        sub = Y[:, trace].astype(np.float64)
        sub[mask] = 0.0
        sub /= sub.sum(axis=0, keepdims=True)
        sub[mask] = 1e-20
        Y[:, trace] = sub.astype(np.float32)
    return _finish(rng, T, Y, n, ld)


# --------------------------------------------------------------------------------------
# the five BASELINE.json configs (1-based, in file order)
# --------------------------------------------------------------------------------------
CONFIGS: Dict[int, dict] = {
    1: dict(n=4096, K=9, hidden=[64, 64], precision=0, cells="dirichlet",
            calls=("T_from_h", "properties", "ann")),
    2: dict(n=262144, K=19, hidden=[1600, 800, 400], precision=1, cells="stratified",
            calls=("ann",)),
    3: dict(n=2097152, K=19, hidden=[1600, 800, 400], precision=1, cells="stratified",
            calls=("T_from_h", "properties", "ann")),
    4: dict(n=2097152, K=53, hidden=None, precision=None, cells="stratified",
            calls=("properties",)),
    5: dict(n=16777216, K=19, hidden=None, precision=None, cells="robustness",
            calls=("T_from_h", "thermo")),
}


def config_seed(cfg: int) -> int:
    return BASE_SEED + cfg


def make_config(cfg: int, n: Optional[int] = None, ld: Optional[int] = None):
    """(Mechanism, AnnModel | None, Cells) for BASELINE.json configs[cfg-1]; `n` overrides the cell count."""
    c = CONFIGS[cfg]
    seed = config_seed(cfg)
    n = c["n"] if n is None else n
    mech = make_mechanism(c["K"], seed)
    ann = None
    if c["hidden"] is not None:
        ann = make_ann(c["K"], c["hidden"], c["precision"], seed)
    kind = c["cells"]
    if kind == "dirichlet":
        cells = cells_dirichlet(c["K"], n, seed, ld=ld)
    elif kind == "stratified":
        cells = cells_stratified(c["K"], n, seed, ld=ld)
    else:
        cells = cells_robustness(c["K"], n, seed, ld=ld)
    return mech, ann, cells
