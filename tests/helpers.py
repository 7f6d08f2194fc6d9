"""Shared test helpers: tiny hand-built mechanisms / networks and the A12 tolerance forms."""
from types import SimpleNamespace

import numpy as np

R = 8314.46261815324


def read_textbook():
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "textbook_values.txt")) as f:
        for line in f:
            if line.startswith("#") or "|" not in line:
                continue
            name, val, unit, tol, _src = [s.strip() for s in line.split("|")]
            out[name] = (float(val), float(tol))
    return out


def tiny_mech(K, W=None, a_lo=None, a_hi=None, visc=None, cond=None, bdiff=None, T_mid=1000.0):
    """Hand-built mechanism: defaults are constant cp/R = 3.5, constant-coefficient fits."""
    W = np.full(K, 28.0) if W is None else np.asarray(W, float)
    if a_lo is None:
        a_lo = np.zeros((K, 7))
        a_lo[:, 0] = 3.5
    a_lo = np.asarray(a_lo, float)
    a_hi = a_lo.copy() if a_hi is None else np.asarray(a_hi, float)
    if visc is None:
        visc = np.zeros((K, 5)); visc[:, 0] = 1e-3 * (1 + 0.1 * np.arange(K))
    if cond is None:
        cond = np.zeros((K, 5)); cond[:, 0] = 2e-3 * (1 + 0.2 * np.arange(K))
    if bdiff is None:
        bdiff = np.zeros((K, K, 5))
        for j in range(K):
            for k in range(K):
                bdiff[j, k, 0] = 1e-5 * (1 + 0.1 * (j + k))
    return SimpleNamespace(K=K, W=W, nasa_lo=a_lo, nasa_hi=a_hi, T_low=300.0, T_mid=T_mid, T_high=3500.0,
                           visc_fit=np.asarray(visc, float), cond_fit=np.asarray(cond, float),
                           bdiff_fit=np.asarray(bdiff, float))


def tiny_ann(dims, W=None, b=None, x_mean=None, x_std=None, u_mean=None, u_std=None, lam=0.1, dt=1e-6,
             precision=0, seed=0):
    rng = np.random.default_rng(seed)
    nl = len(dims) - 1
    if W is None:
        W = [rng.normal(0, 0.5, (dims[l + 1], dims[l])).astype(np.float32) for l in range(nl)]
    if b is None:
        b = [rng.normal(0, 0.2, dims[l + 1]).astype(np.float32) for l in range(nl)]
    K = dims[-1]
    return SimpleNamespace(dims=list(dims), W=W, b=b, precision=precision,
                           x_mean=np.zeros(dims[0]) if x_mean is None else np.asarray(x_mean, float),
                           x_std=np.ones(dims[0]) if x_std is None else np.asarray(x_std, float),
                           u_mean=np.zeros(K) if u_mean is None else np.asarray(u_mean, float),
                           u_std=np.ones(K) if u_std is None else np.asarray(u_std, float),
                           boxcox_lambda=lam, dt=dt)


def const_output_ann(K, out, lam=0.1, dt=1e-6, **kw):
    """Network whose output is the constant vector `out` (zero weights, last bias = out)."""
    dims = [K + 2, 4, K]
    W = [np.zeros((4, K + 2), np.float32), np.zeros((K, 4), np.float32)]
    b = [np.zeros(4, np.float32), np.asarray(out, np.float32)]
    return tiny_ann(dims, W, b, lam=lam, dt=dt, **kw)


# ---- SURVEY 8(c) A12 tolerance forms (shared by the GPU parity tests) -------------------------
def rel_err(got, ref):
    ref = np.asarray(ref, np.float64)
    return np.abs(np.asarray(got, np.float64) - ref) / np.abs(ref)


def mixed_err(got, ref, axis=-1):
    """max over elements of |d| / (|ref| + RMS_cells(ref_k)), and the per-species normwise error."""
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    d = got - ref
    rms = np.sqrt(np.mean(ref * ref, axis=axis, keepdims=True))
    mixed = np.abs(d) / (np.abs(ref) + rms + 1e-300)
    norm = np.sqrt(np.sum(d * d, axis=axis)) / (np.sqrt(np.sum(ref * ref, axis=axis)) + 1e-300)
    return float(mixed.max()), float(norm.max())


def mixed_err_table(got, ref):
    """Per-species A12 figures of a [K, n] result: element-wise mixed maximum (with the cell it occurs at) and the
    normwise error."""
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    d = got - ref
    rms = np.sqrt(np.mean(ref * ref, axis=1, keepdims=True))
    mixed = np.abs(d) / (np.abs(ref) + rms + 1e-300)
    norm = np.sqrt(np.sum(d * d, axis=1)) / (np.sqrt(np.sum(ref * ref, axis=1)) + 1e-300)
    worst = mixed.argmax(axis=1)
    return [dict(k=int(k), mixed=float(mixed[k, worst[k]]), cell=int(worst[k]), normwise=float(norm[k]),
                 p999=float(np.quantile(mixed[k], 0.999)), rms_ref=float(rms[k, 0]))
            for k in range(got.shape[0])]


def record(tag, payload):
    """Append one JSON line of measured errors to gpurun_out/parity_measured.jsonl (the folder a GPU run brings
    back); the summaries under profiles/ are copied from there.  Silent when the folder cannot be written."""
    import json
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    try:
        os.makedirs(os.path.join(root, "gpurun_out"), exist_ok=True)
        with open(os.path.join(root, "gpurun_out", "parity_measured.jsonl"), "a") as f:
            f.write(json.dumps(dict(tag=tag, **payload)) + "\n")
    except OSError:
        pass


FLOOR_FACTOR = 1.25


def bounds_16bit(ref, ideal, tol=2e-2):
    """Per-species element-wise (mixed-form) bound on the 16-bit tensor path: north_star's 2e-2, or, for a species
    whose exactly rounded fp16 chain (tests/ideal16.py) already exceeds 0.8 x that, 1.25 x that floor (A12).
    Returns (bounds[K], floor_table)."""
    floor = mixed_err_table(ideal, ref)
    return np.array([max(tol, FLOOR_FACTOR * t["mixed"]) for t in floor]), floor
