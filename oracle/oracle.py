"""ctypes wrapper over oracle/oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` leg may
import this.  It takes the table objects of `paper_2312_05800_b200.synth` by duck typing
(attributes only) and never imports the package.  All field arrays are promoted to fp64
exactly from whatever fp32 bits the caller holds ("same fp32 input bits").
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_LIB_NATIVE = os.path.join(_HERE, "liboracle_native.so")
_lib = None
_native = False
_FLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp"]
_FLAGS_NATIVE = ["-std=c++17", "-O3", "-march=native", "-ffp-contract=off", "-fopenmp"]


def build(force: bool = False) -> str:
    """g++ -O2 (generic x86-64: the .so travels to another host), OpenMP over cells."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", *_FLAGS, "-fPIC", "-shared", _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


def use_native_build() -> None:
    """bench.py's timed legs only: the same source compiled on, and for, the host it is timed
    on (-O3 -march=native; still -ffp-contract=off, so the arithmetic is the tests').  Always rebuilt: a library
    carried over from another host could hold instructions this CPU lacks.  Must be called before the first use."""
    global _native
    assert _lib is None, "use_native_build() must come before the library is loaded"
    subprocess.run(["g++", *_FLAGS_NATIVE, "-fPIC", "-shared", _SRC, "-o", _LIB_NATIVE], check=True)
    _native = True


def build_flags() -> str:
    return "g++ " + " ".join(_FLAGS_NATIVE if _native else _FLAGS)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_LIB_NATIVE if _native else build())
        d, i, ll, vp = C.c_double, C.c_int, C.c_longlong, C.c_void_p
        P = C.c_void_p
        _lib.oracle_mech_create.restype = vp
        _lib.oracle_mech_create.argtypes = [i, P, P, P, d, d, d, P, P, P]
        _lib.oracle_mech_destroy.argtypes = [vp]
        _lib.oracle_ann_create.restype = vp
        _lib.oracle_ann_create.argtypes = [i, P, P, P, P, P, P, P, d, d]
        _lib.oracle_ann_destroy.argtypes = [vp]
        _lib.oracle_set_threads.argtypes = [i]
        _lib.oracle_get_threads.restype = i
        _lib.oracle_species_thermo.argtypes = [vp, i, d, P, P, P]
        _lib.oracle_species_transport.argtypes = [vp, d, d, P, P, P]
        _lib.oracle_mixture_cp_h.argtypes = [vp, ll, ll, P, P, P, P]
        _lib.oracle_T_from_h.argtypes = [vp, ll, ll, P, P, P, P, P]
        _lib.oracle_properties.argtypes = [vp, ll, ll, P, P, P, P, P, P, P, P]
        for f in (_lib.oracle_boxcox, _lib.oracle_boxcox_inv):
            f.restype = d
            f.argtypes = [d, d]
        _lib.oracle_gelu.restype = d
        _lib.oracle_gelu.argtypes = [d]
        _lib.oracle_extras.argtypes = [vp, ll, ll] + [P] * 12
        _lib.oracle_pasr.argtypes = [vp, ll, ll, P, P, P, P, P, P, d, P, P, P]
        _lib.oracle_ann_features.argtypes = [vp, ll, ll, P, P, P, P]
        _lib.oracle_mlp_forward.argtypes = [vp, ll, P, P]
        _lib.oracle_ann_source.argtypes = [vp, vp, ll, ll, P, P, P, P, P]
        _lib.oracle_ann_source_mmlp.argtypes = [P, vp, ll, ll, P, P, P, P, P]
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def get_threads() -> int:
    return int(lib().oracle_get_threads())


class Mech:
    """fp64 species tables (attributes as synth.Mechanism)."""

    def __init__(self, m):
        self.K = int(m.K)
        t = [_f64(x) for x in (m.W, m.nasa_lo, m.nasa_hi, m.visc_fit, m.cond_fit, m.bdiff_fit)]
        assert t[1].shape == (self.K, 7) and t[5].shape == (self.K, self.K, 5)
        self.h = lib().oracle_mech_create(self.K, _p(t[0]), _p(t[1]), _p(t[2]), float(m.T_low), float(m.T_mid),
                                          float(m.T_high), _p(t[3]), _p(t[4]), _p(t[5]))

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.oracle_mech_destroy(self.h)
            self.h = None

    # --- O1
    def species_thermo(self, k: int, T: float):
        cp, h, s = C.c_double(), C.c_double(), C.c_double()
        lib().oracle_species_thermo(self.h, int(k), float(T), C.byref(cp), C.byref(h), C.byref(s))
        return cp.value, h.value, s.value

    # --- O5
    def species_transport(self, T: float, p: float):
        K = self.K
        mu, lam, D = np.empty(K), np.empty(K), np.empty((K, K))
        lib().oracle_species_transport(self.h, float(T), float(p), _p(mu), _p(lam), _p(D))
        return mu, lam, D

    @staticmethod
    def _fields(T, Y):
        Y = _f64(Y)
        T = _f64(T)
        n = T.shape[0]
        assert Y.ndim == 2 and Y.shape[1] >= n
        return T, Y, n, Y.shape[1]

    # --- O2
    def mixture_cp_h(self, T, Y):
        T, Y, n, ld = self._fields(T, Y)
        cp, h = np.empty(n), np.empty(n)
        lib().oracle_mixture_cp_h(self.h, n, ld, _p(T), _p(Y), _p(cp), _p(h))
        return cp, h

    # --- O3
    def T_from_h(self, h, Y, T_guess, return_iters=False):
        h, Y, n, ld = self._fields(h, Y)
        g = _f64(T_guess)
        T = np.empty(n)
        it = np.zeros(n, dtype=np.int32)
        lib().oracle_T_from_h(self.h, n, ld, _p(h), _p(Y), _p(g), _p(T), _p(it))
        return (T, it) if return_iters else T

    # --- O4..O8
    def properties(self, T, p, Y):
        T, Y, n, ld = self._fields(T, Y)
        p = _f64(p)
        cp, h, mu, lam = (np.empty(n) for _ in range(4))
        D = np.zeros((self.K, ld))
        lib().oracle_properties(self.h, n, ld, _p(T), _p(p), _p(Y), _p(cp), _p(h), _p(mu), _p(lam), _p(D))
        return dict(cp=cp, h=h, mu=mu, lam=lam, D=D)


    # --- NEXT-4 (A22): rho, psi, alpha, rho D_k, h_k(T), s
    def extras(self, T, p, Y, cp=None, lam=None, D=None):
        T, Y, n, ld = self._fields(T, Y)
        p = _f64(p)
        cp = None if cp is None else _f64(cp)
        lam = None if lam is None else _f64(lam)
        D = None if D is None else _f64(D)
        rho, psi, alpha, s = (np.empty(n) for _ in range(4))
        rhoD, hk = np.zeros((self.K, ld)), np.zeros((self.K, ld))
        lib().oracle_extras(self.h, n, ld, _p(T), _p(p), _p(Y), _p(cp), _p(lam), _p(D), _p(rho), _p(psi), _p(alpha),
                            _p(rhoD), _p(hk), _p(s))
        out = dict(rho=rho, psi=psi, hk=hk, s=s)
        if cp is not None and lam is not None:
            out["alpha"] = alpha
        if D is not None:
            out["rhoD"] = rhoD
        return out

    # --- NEXT-3 (A23): PaSR scaling + temperature gate
    def pasr(self, T, p, Y, mu, ksgs, eps, T_gate, omega):
        T, Y, n, ld = self._fields(T, Y)
        p, mu, ksgs, eps = (_f64(x) for x in (p, mu, ksgs, eps))
        om = _f64(omega)
        assert om.shape == Y.shape
        out = np.zeros_like(om)
        kappa = np.empty(n)
        lib().oracle_pasr(self.h, n, ld, _p(T), _p(p), _p(Y), _p(mu), _p(ksgs), _p(eps), float(T_gate), _p(om), _p(out),
                          _p(kappa))
        return out, kappa


class Ann:
    """fp64 copy of an MLP + normalisation tables (attributes as synth.AnnModel)."""

    def __init__(self, a):
        self.dims = [int(x) for x in a.dims]
        self.K = self.dims[-1]
        nl = len(self.dims) - 1
        dims = np.asarray(self.dims, dtype=np.int32)
        Wf = np.concatenate([_f64(w).ravel() for w in a.W])
        bf = np.concatenate([_f64(b).ravel() for b in a.b])
        for l in range(nl):
            assert a.W[l].shape == (self.dims[l + 1], self.dims[l])
        xs = [_f64(x) for x in (a.x_mean, a.x_std, a.u_mean, a.u_std)]
        self.h = lib().oracle_ann_create(nl, _p(dims), _p(Wf), _p(bf), _p(xs[0]), _p(xs[1]), _p(xs[2]), _p(xs[3]),
                                         float(a.boxcox_lambda), float(a.dt))

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.oracle_ann_destroy(self.h)
            self.h = None

    # --- O9
    def features(self, T, p, Y):
        T, Y, n, ld = Mech._fields(T, Y)
        p = _f64(p)
        f = np.empty((n, self.dims[0]))
        lib().oracle_ann_features(self.h, n, ld, _p(T), _p(p), _p(Y), _p(f))
        return f

    # --- O10
    def mlp(self, x):
        x = _f64(x)
        n = x.shape[0]
        assert x.shape[1] == self.dims[0]
        o = np.empty((n, self.K))
        lib().oracle_mlp_forward(self.h, n, _p(x), _p(o))
        return o

    # --- O11, O12
    def source(self, mech: Mech, T, p, Y):
        T, Y, n, ld = Mech._fields(T, Y)
        p = _f64(p)
        om = np.zeros((self.K, ld))
        dY = np.zeros((self.K, ld))
        lib().oracle_ann_source(self.h, mech.h, n, ld, _p(T), _p(p), _p(Y), _p(om), _p(dY))
        return om, dY


class Mmlp:
    """K one-output networks, one per species (NEXT-1): nets[k] has the attributes of synth.AnnModel with
    dims[0] = K + 2, dims[-1] = 1, the shared input statistics in x_mean/x_std and species k's u_mean/u_std."""

    def __init__(self, nets):
        self.K = len(nets)
        for a in nets:
            assert int(a.dims[0]) == self.K + 2 and int(a.dims[-1]) == 1
        self.nets = [Ann(a) for a in nets]
        self._arr = (C.c_void_p * self.K)(*[a.h for a in self.nets])

    def source(self, mech: Mech, T, p, Y):
        T, Y, n, ld = Mech._fields(T, Y)
        p = _f64(p)
        om = np.zeros((self.K, ld))
        dY = np.zeros((self.K, ld))
        lib().oracle_ann_source_mmlp(self._arr, mech.h, n, ld, _p(T), _p(p), _p(Y), _p(om), _p(dY))
        return om, dY


def boxcox(y: float, lam: float) -> float:
    return float(lib().oracle_boxcox(float(y), float(lam)))


def boxcox_inv(f: float, lam: float) -> float:
    return float(lib().oracle_boxcox_inv(float(f), float(lam)))


def gelu(x: float) -> float:
    return float(lib().oracle_gelu(float(x)))
