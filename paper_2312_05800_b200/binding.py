"""Thin ctypes binding over libdfthermo.so (include/df_thermo.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used for
device memory and streams.  There is no CPU fallback: importing this module raises if the
library has not been built (`python -m paper_2312_05800_b200.build`), and the create calls
raise if no CUDA device is present.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdfthermo.so")

# every symbol include/df_thermo.h declares (tests check the library exports all of them)
SYMBOLS = (
    "df_abi_version", "df_last_error",
    "df_mech_create", "df_mech_destroy", "df_mech_num_species",
    "df_ann_create", "df_ann_destroy", "df_ann_workspace_bytes",
    "df_thermo_T_from_h", "df_thermo_properties", "df_chem_ann_source",
    "df_thermo_extras", "df_chem_pasr_scale",
    "df_ann_mmlp_create", "df_ann_mmlp_destroy", "df_ann_mmlp_workspace_bytes", "df_chem_ann_source_mmlp",
    "df_step_plan_create", "df_thermochem_step", "df_step_plan_destroy",
    "df_host_ctx_create", "df_host_ctx_destroy", "df_step_host",
    "df_probe_fp32_peak",
    "df_ann_static_scratch_bytes", "df_chem_ann_source_static",
)

DF_OK, DF_ERR_INVALID_ARG, DF_ERR_UNSUPPORTED, DF_ERR_ALLOC, DF_ERR_CUDA = range(5)


class DfError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libdfthermo error {code}: {msg}")
        self.code = code


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2312_05800_b200.build` "
                      "(there is no CPU fallback)")

_lib = C.CDLL(LIB_PATH)
_vp, _ll, _i, _d, _sz = C.c_void_p, C.c_longlong, C.c_int, C.c_double, C.c_size_t
_lib.df_abi_version.restype = _i
_lib.df_last_error.restype = C.c_char_p
_lib.df_mech_create.argtypes = [C.POINTER(_vp), _i, _vp, _vp, _vp, _d, _d, _d, _vp, _vp, _vp]
_lib.df_mech_destroy.argtypes = [_vp]
_lib.df_mech_num_species.argtypes = [_vp]
_lib.df_ann_create.argtypes = [C.POINTER(_vp), _i, _vp, C.POINTER(_vp), C.POINTER(_vp), _i, _vp, _vp, _vp, _vp, _d, _d]
_lib.df_ann_destroy.argtypes = [_vp]
_lib.df_ann_workspace_bytes.restype = _sz
_lib.df_ann_workspace_bytes.argtypes = [_vp, _ll]
_lib.df_thermo_T_from_h.argtypes = [_vp, _ll, _ll, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.df_thermo_properties.argtypes = [_vp, _ll, _ll, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.df_chem_ann_source.argtypes = [_vp, _vp, _ll, _ll, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.df_ann_static_scratch_bytes.restype = _sz
_lib.df_ann_static_scratch_bytes.argtypes = []
_lib.df_chem_ann_source_static.argtypes = [_vp, _vp, _ll, _ll, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.df_thermo_extras.argtypes = [_vp, _ll, _ll] + [_vp] * 13
_lib.df_chem_pasr_scale.argtypes = [_vp, _ll, _ll, _vp, _vp, _vp, _vp, _vp, _vp, C.c_float, _vp, _vp, _vp]
_lib.df_ann_mmlp_create.argtypes = [C.POINTER(_vp), _i, _i, _vp, C.POINTER(_vp), C.POINTER(_vp), _vp, _vp, _vp, _vp, _d, _d]
_lib.df_ann_mmlp_destroy.argtypes = [_vp]
_lib.df_ann_mmlp_workspace_bytes.restype = _sz
_lib.df_ann_mmlp_workspace_bytes.argtypes = [_vp, _ll, _ll]
_lib.df_chem_ann_source_mmlp.argtypes = [_vp, _vp, _ll, _ll, _vp, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.df_step_plan_create.argtypes = [C.POINTER(_vp), _vp, _vp, _ll, _ll] + [_vp] * 11 + [_sz]
_lib.df_thermochem_step.argtypes = [_vp, _vp]
_lib.df_step_plan_destroy.argtypes = [_vp]
_lib.df_host_ctx_create.argtypes = [C.POINTER(_vp), _vp, _vp, _ll]
_lib.df_host_ctx_destroy.argtypes = [_vp]
_lib.df_step_host.argtypes = [_vp, _ll, _ll] + [_vp] * 10
_lib.df_probe_fp32_peak.argtypes = [_i, _i, _ll, _vp, C.POINTER(_d), _vp]


def _check(code: int) -> None:
    if code != DF_OK:
        raise DfError(code, (_lib.df_last_error() or b"").decode())


def abi_version() -> int:
    return int(_lib.df_abi_version())


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _np(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(_vp)


def _dp(t) -> Optional[int]:
    """Device (or pinned host) pointer of a torch tensor, None passes NULL."""
    if t is None:
        return None
    assert t.is_contiguous(), "field arrays must be contiguous"
    return t.data_ptr()


def _stream(stream) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


class Mech:
    """df_mech handle from a table object with the attributes of synth.Mechanism."""

    def __init__(self, m):
        self.K = int(m.K)
        t = [_f64(x) for x in (m.W, m.nasa_lo, m.nasa_hi, m.visc_fit, m.cond_fit, m.bdiff_fit)]
        if t[1].shape != (self.K, 7) or t[2].shape != (self.K, 7) or t[5].shape != (self.K, self.K, 5):
            raise ValueError("table shapes do not match K")
        h = _vp()
        _check(_lib.df_mech_create(C.byref(h), self.K, _np(t[0]), _np(t[1]), _np(t[2]), float(m.T_low), float(m.T_mid),
                                   float(m.T_high), _np(t[3]), _np(t[4]), _np(t[5])))
        self.handle = h

    def close(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.df_mech_destroy(self.handle)
            self.handle = None

    __del__ = close


class Ann:
    """df_ann handle from an object with the attributes of synth.AnnModel."""

    def __init__(self, a):
        self.dims = [int(x) for x in a.dims]
        self.K = self.dims[-1]
        self.precision = int(a.precision)
        nl = len(self.dims) - 1
        dims = np.asarray(self.dims, dtype=np.int32)
        Ws = [np.ascontiguousarray(w, dtype=np.float32) for w in a.W]
        bs = [np.ascontiguousarray(b, dtype=np.float32) for b in a.b]
        for l in range(nl):
            if Ws[l].shape != (self.dims[l + 1], self.dims[l]) or bs[l].shape != (self.dims[l + 1],):
                raise ValueError(f"layer {l}: weight/bias shape does not match dims")
        Wp = (_vp * nl)(*[w.ctypes.data for w in Ws])
        bp = (_vp * nl)(*[b.ctypes.data for b in bs])
        xs = [_f64(x) for x in (a.x_mean, a.x_std, a.u_mean, a.u_std)]
        h = _vp()
        _check(_lib.df_ann_create(C.byref(h), nl, _np(dims), Wp, bp, self.precision, _np(xs[0]), _np(xs[1]),
                                  _np(xs[2]), _np(xs[3]), float(a.boxcox_lambda), float(a.dt)))
        self.handle = h

    def workspace_bytes(self, n_cells: int) -> int:
        return int(_lib.df_ann_workspace_bytes(self.handle, int(n_cells)))

    def close(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.df_ann_destroy(self.handle)
            self.handle = None

    __del__ = close


class AnnMmlp:
    """df_ann_mmlp handle from a list of K one-output networks (attributes of synth.AnnModel; see synth.make_mmlp)."""

    def __init__(self, nets):
        self.K = len(nets)
        dims = np.asarray([int(x) for x in nets[0].dims], dtype=np.int32)
        nl = len(dims) - 1
        Ws = [np.ascontiguousarray(w, dtype=np.float32) for a in nets for w in a.W]
        bs = [np.ascontiguousarray(x, dtype=np.float32) for a in nets for x in a.b]
        for a in nets:
            if [int(x) for x in a.dims] != list(dims):
                raise ValueError("all networks must have the same dims")
        Wp = (_vp * len(Ws))(*[w.ctypes.data for w in Ws])
        bp = (_vp * len(bs))(*[x.ctypes.data for x in bs])
        xm, xs = _f64(nets[0].x_mean), _f64(nets[0].x_std)
        um = _f64([float(np.asarray(a.u_mean).ravel()[0]) for a in nets])
        us = _f64([float(np.asarray(a.u_std).ravel()[0]) for a in nets])
        h = _vp()
        _check(_lib.df_ann_mmlp_create(C.byref(h), self.K, nl, _np(dims), Wp, bp, _np(xm), _np(xs), _np(um), _np(us),
                                       float(nets[0].boxcox_lambda), float(nets[0].dt)))
        self.handle = h

    def workspace_bytes(self, n_cells: int, ld: int) -> int:
        return int(_lib.df_ann_mmlp_workspace_bytes(self.handle, int(n_cells), int(ld)))

    def close(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.df_ann_mmlp_destroy(self.handle)
            self.handle = None

    __del__ = close


def df_chem_ann_source_mmlp(m: AnnMmlp, mech: Mech, T, p, Y, omega=None, dY=None, workspace=None, n_cells=None,
                            stream=None) -> None:
    n = int(T.shape[0]) if n_cells is None else int(n_cells)
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(_lib.df_chem_ann_source_mmlp(m.handle, mech.handle, n, int(Y.shape[1]), _dp(T), _dp(p), _dp(Y), _dp(omega),
                                        _dp(dY), _dp(workspace), ws_bytes, _stream(stream)))


def alloc_workspace_mmlp(m: AnnMmlp, n_cells: int, ld: int, device="cuda"):
    import torch
    nbytes = m.workspace_bytes(n_cells, ld)
    ws = torch.empty(nbytes + 1024, dtype=torch.uint8, device=device)
    off = (-ws.data_ptr()) % 1024
    return ws[off:off + nbytes]


def df_thermo_T_from_h(mech: Mech, h, Y, T, cp=None, n_unconverged=None, n_cells=None, stream=None) -> None:
    """T (in: guess, out: root) from h and Y[K, ld]; torch CUDA float32 tensors."""
    n = int(T.shape[0]) if n_cells is None else int(n_cells)
    _check(_lib.df_thermo_T_from_h(mech.handle, n, int(Y.shape[1]), _dp(h), _dp(Y), _dp(T), _dp(cp),
                                   _dp(n_unconverged), _stream(stream)))


def df_thermo_properties(mech: Mech, T, p, Y, cp=None, h=None, mu=None, lam=None, D=None, n_cells=None,
                         stream=None) -> None:
    n = int(T.shape[0]) if n_cells is None else int(n_cells)
    _check(_lib.df_thermo_properties(mech.handle, n, int(Y.shape[1]), _dp(T), _dp(p), _dp(Y), _dp(cp), _dp(h),
                                     _dp(mu), _dp(lam), _dp(D), _stream(stream)))


def df_chem_ann_source(ann: Ann, mech: Mech, T, p, Y, omega=None, dY=None, workspace=None, n_cells=None,
                       stream=None) -> None:
    n = int(T.shape[0]) if n_cells is None else int(n_cells)
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(_lib.df_chem_ann_source(ann.handle, mech.handle, n, int(Y.shape[1]), _dp(T), _dp(p), _dp(Y), _dp(omega),
                                   _dp(dY), _dp(workspace), ws_bytes, _stream(stream)))


def df_ann_static_scratch_bytes() -> int:
    return int(_lib.df_ann_static_scratch_bytes())


def df_chem_ann_source_static(ann: Ann, mech: Mech, T, p, Y, omega=None, dY=None, n_cells=None, stream=None) -> None:
    """df_chem_ann_source on the library's static device scratch: no workspace argument, no allocation."""
    n = int(T.shape[0]) if n_cells is None else int(n_cells)
    _check(_lib.df_chem_ann_source_static(ann.handle, mech.handle, n, int(Y.shape[1]), _dp(T), _dp(p), _dp(Y), _dp(omega),
                                          _dp(dY), _stream(stream)))


def df_thermo_extras(mech: Mech, T, p, Y, cp=None, lam=None, D=None, rho=None, psi=None, alpha=None, rhoD=None, hk=None,
                     s=None, n_cells=None, stream=None) -> None:
    n = int(T.shape[0]) if n_cells is None else int(n_cells)
    _check(_lib.df_thermo_extras(mech.handle, n, int(Y.shape[1]), _dp(T), _dp(p), _dp(Y), _dp(cp), _dp(lam), _dp(D),
                                 _dp(rho), _dp(psi), _dp(alpha), _dp(rhoD), _dp(hk), _dp(s), _stream(stream)))


def df_chem_pasr_scale(mech: Mech, T, p, Y, mu, k_sgs, eps, T_gate, omega, kappa=None, n_cells=None, stream=None) -> None:
    n = int(T.shape[0]) if n_cells is None else int(n_cells)
    _check(_lib.df_chem_pasr_scale(mech.handle, n, int(Y.shape[1]), _dp(T), _dp(p), _dp(Y), _dp(mu), _dp(k_sgs), _dp(eps),
                                   float(T_gate), _dp(omega), _dp(kappa), _stream(stream)))


def alloc_workspace(ann: Ann, n_cells: int, device="cuda"):
    """torch-owned scratch for df_chem_ann_source (None when the path needs none)."""
    import torch
    nbytes = ann.workspace_bytes(n_cells)
    if nbytes == 0:
        return None
    ws = torch.empty(nbytes + 1024, dtype=torch.uint8, device=device)
    off = (-ws.data_ptr()) % 1024
    return ws[off:off + nbytes]


class StepPlan:
    """df_step_plan: the whole step on fixed device arrays as one CUDA graph; launch() replays it with one launch."""

    def __init__(self, mech: Mech, ann: Optional[Ann], h, p, Y, T, T_guess=None, cp=None, mu=None, lam=None, D=None,
                 omega=None, workspace=None, n_cells=None):
        n = int(T.shape[0]) if n_cells is None else int(n_cells)
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        hdl = _vp()
        _check(_lib.df_step_plan_create(C.byref(hdl), mech.handle, ann.handle if ann is not None else None, n, int(Y.shape[1]),
                                        _dp(h), _dp(p), _dp(T_guess), _dp(Y), _dp(T), _dp(cp), _dp(mu), _dp(lam), _dp(D),
                                        _dp(omega), _dp(workspace), ws_bytes))
        self.handle = hdl
        self._keep = (mech, ann, h, p, Y, T, T_guess, cp, mu, lam, D, omega, workspace)

    def launch(self, stream=None) -> None:
        _check(_lib.df_thermochem_step(self.handle, _stream(stream)))

    def close(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.df_step_plan_destroy(self.handle)
            self.handle = None

    __del__ = close


class HostCtx:
    """df_host_ctx: device staging for df_step_host (host arrays in, host arrays out)."""

    def __init__(self, mech: Mech, ann: Optional[Ann], max_cells: int):
        h = _vp()
        _check(_lib.df_host_ctx_create(C.byref(h), mech.handle, ann.handle if ann is not None else None, int(max_cells)))
        self.handle = h
        self._keep = (mech, ann)

    def step(self, n_cells, ld, h, p, T_guess, Y, T=None, cp=None, mu=None, lam=None, D=None, omega=None) -> None:
        """Arguments are torch CPU (pinned) float32 tensors or None."""
        _check(_lib.df_step_host(self.handle, int(n_cells), int(ld), _dp(h), _dp(p), _dp(T_guess), _dp(Y), _dp(T),
                                 _dp(cp), _dp(mu), _dp(lam), _dp(D), _dp(omega)))

    def close(self):
        if getattr(self, "handle", None) and _lib is not None:
            _lib.df_host_ctx_destroy(self.handle)
            self.handle = None

    __del__ = close


def df_probe_fp32_peak(variant: int, blocks: int, iters: int, out=None, stream=None) -> float:
    """Launch the FMA-chain probe; returns the flops of the launch (time it with CUDA events)."""
    fl = _d(0.0)
    _check(_lib.df_probe_fp32_peak(int(variant), int(blocks), int(iters), _dp(out), C.byref(fl), _stream(stream)))
    return float(fl.value)
