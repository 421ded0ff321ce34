"""paper_2008_08483_b200 -- B200-native batched chemical source terms (arXiv 2008.08483).

Thin Python binding of the C ABI in include/ck.h (libck.so, hand-written CUDA for
sm_100a).  Argument marshalling only: every step of the path runs in the CUDA kernels.
There is no CPU fallback; importing this package fails loudly if the library is missing
and cannot be built.  PyTorch (optional here) is only used by callers for device memory
and streams; this module accepts anything exposing `data_ptr()` or raw integer addresses.

    mech = Mechanism(ckgen_mechanism)                  # ck_mech_create
    mech.source_terms(T, P, Y, wdot, dTdt, stream=0)   # ck_source_terms (device pointers)
    mech.source_terms_host(T, P, Y)                    # ck_source_terms_host (numpy, host)
    mech.close()                                       # ck_mech_destroy
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import _build

__all__ = ["Mechanism", "CkError", "ck_mech_create", "ck_source_terms", "ck_source_terms_static", "ck_source_terms_host",
           "ck_rk4_integrate", "ck_jacobian",
           "ck_mech_destroy", "ck_last_error", "ck_mech_info", "ck_mech_note", "ck_measure_fp64_peak", "ck_measure_peaks",
           "ck_mech_jit_source",
           "library_path", "RU", "INFO", "PREC_F64", "PREC_MIXED", "PREC_F32_RATES"]

RU = 8314.46261815324  # J/(kmol K), the constant compiled into the kernels
INFO = {"S": 0, "R": 1, "nnz_reac": 2, "nnz_prod": 3, "nnz_net": 4, "n_three_body": 5,
        "n_lindemann": 6, "n_troe": 7, "n_ranges": 8, "threads": 9, "blocks_per_sm": 10,
        "smem_bytes": 11, "launches_per_call": 12, "nnz_eff": 13, "jit": 14, "s_reg": 15, "jac_cells": 16, "pair": 17, "ablation": 18, "precision": 19, "all_dmma": 20, "small_batch_max": 21, "jac_kernel": 22}
PREC_F64, PREC_MIXED, PREC_F32_RATES = 0, 1, 2

_dp = C.POINTER(C.c_double)
_bp = C.POINTER(C.c_uint8)


class _Ann(C.Structure):
    _fields_ = [("n_in", C.c_int32), ("n_layers", C.c_int32), ("n_hidden", C.c_int32),
                ("activation", C.c_int32), ("in_mean", _dp), ("in_std", _dp), ("W_in", _dp),
                ("B", _dp), ("W_hid", _dp), ("W_out", _dp), ("B_out", _dp), ("out_mean", _dp),
                ("out_std", _dp)]


class _Desc(C.Structure):
    _fields_ = [
        ("n_species", C.c_int32), ("n_reactions", C.c_int32),
        ("mol_weight", _dp), ("nu_reac", _dp), ("nu_prod", _dp),
        ("ln_A", _dp), ("b", _dp), ("Ea_over_R", _dp), ("reversible", _bp),
        ("nasa_lo", _dp), ("nasa_hi", _dp), ("T_mid", _dp), ("rxn_type", _bp),
        ("eff", _dp), ("ln_A0", _dp), ("b0", _dp), ("Ea0_over_R", _dp), ("troe", _dp),
        ("p_ref", C.c_double), ("kc_ann", C.POINTER(_Ann)), ("precision", C.c_int32),
    ]


class CkError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("ck status %d: %s" % (status, message))
        self.status = status


def library_path() -> str:
    return _build.LIB


def _load():
    path = _build.LIB
    if not os.path.exists(path) or os.path.getmtime(path) < _build._newest_source():
        path = _build.build()          # raises if nvcc is missing or compilation fails
    lib = C.CDLL(path)
    lib.ck_mech_create.restype = C.c_int
    lib.ck_mech_create.argtypes = [C.POINTER(_Desc), C.POINTER(C.c_void_p)]
    lib.ck_source_terms.restype = C.c_int
    lib.ck_source_terms.argtypes = [C.c_void_p] * 4 + [C.c_int64] + [C.c_void_p] * 3
    lib.ck_source_terms_static.restype = C.c_int
    lib.ck_source_terms_static.argtypes = [C.c_void_p] * 4 + [C.c_int64] + [C.c_void_p] * 3
    lib.ck_source_terms_host.restype = C.c_int
    lib.ck_source_terms_host.argtypes = [C.c_void_p] * 4 + [C.c_int64] + [C.c_void_p] * 3
    lib.ck_rk4_integrate.restype = C.c_int
    lib.ck_rk4_integrate.argtypes = [C.c_void_p] * 4 + [C.c_int64, C.c_double, C.c_int64, C.c_int, C.c_void_p]
    lib.ck_mech_destroy.restype = None
    lib.ck_mech_destroy.argtypes = [C.c_void_p]
    lib.ck_last_error.restype = C.c_char_p
    lib.ck_last_error.argtypes = []
    lib.ck_mech_info.restype = C.c_int64
    lib.ck_mech_info.argtypes = [C.c_void_p, C.c_int]
    lib.ck_jacobian.restype = C.c_int
    lib.ck_jacobian.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    lib.ck_mech_note.restype = C.c_char_p
    lib.ck_mech_note.argtypes = [C.c_void_p]
    lib.ck_mech_jit_source.restype = C.c_int64
    lib.ck_mech_jit_source.argtypes = [C.POINTER(_Desc), C.c_char_p, C.c_int64]
    lib.ck_measure_fp64_peak.restype = C.c_int
    lib.ck_measure_fp64_peak.argtypes = [_dp, C.c_void_p]
    lib.ck_measure_peaks.restype = C.c_int
    lib.ck_measure_peaks.argtypes = [_dp, C.c_void_p]
    return lib


_lib = _load()


def _addr(x):
    """Raw address of a device/host buffer: int, None, torch tensor or numpy array."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    raise TypeError("expected an address, a tensor or a numpy array, got %r" % type(x))


def _check(status):
    if status != 0:
        raise CkError(status, _lib.ck_last_error().decode())


# ---- the C entry points, same names, status codes raised as CkError -------------------

def ck_last_error() -> str:
    return _lib.ck_last_error().decode()


def ck_mech_create(desc: "_Desc") -> int:
    handle = C.c_void_p()
    _check(_lib.ck_mech_create(C.byref(desc), C.byref(handle)))
    return handle.value


def ck_source_terms(handle, T, P, Y, N, wdot, dTdt, stream=0) -> None:
    _check(_lib.ck_source_terms(handle, _addr(T), _addr(P), _addr(Y), int(N), _addr(wdot),
                                _addr(dTdt), stream or None))


def ck_source_terms_static(handle, T, P, Y, N, wdot, dTdt, stream=0) -> None:
    """ck_source_terms for callers that must not allocate device memory (a solver whose memory pool owns
    the device, or one that cannot afford cudaMalloc's device-wide synchronisation in its time loop): the
    kernel's scratch is a fixed 32 MiB array inside libck.so.  Not re-entrant; see include/ck.h."""
    _check(_lib.ck_source_terms_static(handle, _addr(T), _addr(P), _addr(Y), int(N), _addr(wdot),
                                       _addr(dTdt), stream or None))


def ck_source_terms_host(handle, T, P, Y, N, wdot, dTdt, stream=0) -> None:
    _check(_lib.ck_source_terms_host(handle, _addr(T), _addr(P), _addr(Y), int(N), _addr(wdot),
                                     _addr(dTdt), stream or None))


def ck_jacobian(handle, T, P, Y, N, J, stream=0) -> None:
    _check(_lib.ck_jacobian(handle, _addr(T), _addr(P), _addr(Y), int(N), _addr(J), stream or None))


def ck_rk4_integrate(handle, T, P, Y, N, dt, n_steps, use_graph=True, stream=0) -> None:
    _check(_lib.ck_rk4_integrate(handle, _addr(T), _addr(P), _addr(Y), int(N), float(dt), int(n_steps),
                                 1 if use_graph else 0, stream or None))


def ck_mech_destroy(handle) -> None:
    _lib.ck_mech_destroy(handle)


def ck_mech_info(handle, what) -> int:
    return int(_lib.ck_mech_info(handle, INFO[what] if isinstance(what, str) else int(what)))


def ck_mech_note(handle) -> str:
    return _lib.ck_mech_note(handle).decode()


def ck_mech_jit_source(mech, kc_ann=None) -> str:
    """Generated CUDA source of the specialised kernel for `mech` (needs no GPU)."""
    desc, keep = make_desc(mech, kc_ann)
    n = _lib.ck_mech_jit_source(C.byref(desc), None, 0)
    if n < 0:
        raise CkError(4, _lib.ck_last_error().decode())
    buf = C.create_string_buffer(n)
    _lib.ck_mech_jit_source(C.byref(desc), buf, n)
    del keep
    return buf.value.decode()


def ck_measure_fp64_peak(stream=0) -> float:
    out = C.c_double()
    _check(_lib.ck_measure_fp64_peak(C.byref(out), stream or None))
    return out.value


def ck_measure_peaks(stream=0) -> dict:
    """The FP64 microbenchmarks of include/ck.h, by name."""
    out = (C.c_double * 10)()
    _check(_lib.ck_measure_peaks(out, stream or None))
    return {"dfma_per_s": out[0], "dmma_per_s": out[1], "dmma_per_s_interleaved": out[2],
            "dfma_per_s_interleaved": out[3], "libm_exp_per_s": out[4], "libm_log_per_s": out[5],
            "sms": int(out[6]), "imma_s8_m16n8k32_per_s": out[7], "hmma_f16_m16n8k16_per_s": out[8]}


# ---- convenience wrapper -----------------------------------------------------------------

def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _u8(a):
    return np.ascontiguousarray(a, dtype=np.uint8)


def make_desc(mech, kc_ann=None, precision=PREC_F64):
    """ck_mech_desc from any object with ckgen.Mechanism's array attributes (and, optionally,
    a ck_kc_ann from one with ckgen.KcAnn's).  Returns (desc, keepalive) -- keepalive owns the
    host arrays the desc points to."""
    S, R = int(mech.nu_reac.shape[0]), int(mech.nu_reac.shape[1])
    keep = dict(
        mol_weight=_f64(mech.mol_weight), nu_reac=_f64(mech.nu_reac), nu_prod=_f64(mech.nu_prod),
        ln_A=_f64(mech.ln_A), b=_f64(mech.b), Ea_over_R=_f64(mech.Ea_over_R),
        reversible=_u8(mech.reversible), nasa_lo=_f64(mech.nasa_lo), nasa_hi=_f64(mech.nasa_hi),
        T_mid=_f64(mech.T_mid), rxn_type=_u8(mech.rxn_type), eff=_f64(mech.eff),
        ln_A0=_f64(mech.ln_A0), b0=_f64(mech.b0), Ea0_over_R=_f64(mech.Ea0_over_R),
        troe=_f64(mech.troe))
    shapes = dict(mol_weight=(S,), nu_reac=(S, R), nu_prod=(S, R), ln_A=(R,), b=(R,),
                  Ea_over_R=(R,), reversible=(R,), nasa_lo=(S, 7), nasa_hi=(S, 7), T_mid=(S,),
                  rxn_type=(R,), eff=(S, R), ln_A0=(R,), b0=(R,), Ea0_over_R=(R,), troe=(R, 4))
    for name, shp in shapes.items():
        if keep[name].shape != shp:
            raise ValueError("%s has shape %s, expected %s" % (name, keep[name].shape, shp))
    d = _Desc()
    d.n_species, d.n_reactions, d.p_ref = S, R, float(mech.p_ref)
    d.precision = int(precision)
    for name, arr in keep.items():
        setattr(d, name, arr.ctypes.data_as(_bp if arr.dtype == np.uint8 else _dp))
    if kc_ann is not None:
        NL, NH, NI = int(kc_ann.n_layers), int(kc_ann.n_hidden), int(kc_ann.n_in)
        ka = dict(in_mean=_f64(kc_ann.in_mean), in_std=_f64(kc_ann.in_std), W_in=_f64(kc_ann.W_in),
                  B=_f64(kc_ann.B), W_hid=_f64(kc_ann.W_hid), W_out=_f64(kc_ann.W_out),
                  B_out=_f64(kc_ann.B_out), out_mean=_f64(kc_ann.out_mean), out_std=_f64(kc_ann.out_std))
        ann_shapes = dict(in_mean=(NI,), in_std=(NI,), W_in=(NI, NH), B=(NL, NH), W_hid=(NL - 1, NH, NH),
                          W_out=(NH, R), B_out=(R,), out_mean=(R,), out_std=(R,))
        for name, shp in ann_shapes.items():
            if ka[name].shape != shp:
                raise ValueError("kc_ann.%s has shape %s, expected %s" % (name, ka[name].shape, shp))
        a = _Ann()
        a.n_in, a.n_layers, a.n_hidden, a.activation = NI, NL, NH, int(kc_ann.activation)
        for name, arr in ka.items():
            setattr(a, name, arr.ctypes.data_as(_dp))
        keep["_ann_arrays"], keep["_ann"] = ka, a
        d.kc_ann = C.pointer(a)
    return d, keep


class Mechanism:
    """Owns a ck_mech handle created from a mechanism's arrays."""

    def __init__(self, mech, kc_ann=None, precision=PREC_F64):
        desc, keep = make_desc(mech, kc_ann, precision)
        self.handle = ck_mech_create(desc)
        del keep                      # the library copied everything it needs
        self.S = ck_mech_info(self.handle, "S")
        self.R = ck_mech_info(self.handle, "R")

    def info(self, what) -> int:
        return ck_mech_info(self.handle, what)

    def note(self) -> str:
        """Why the specialised kernel is not in use ("" if it is)."""
        return ck_mech_note(self.handle)

    def source_terms(self, T, P, Y, wdot, dTdt, N=None, stream=0) -> None:
        """Device buffers (torch CUDA tensors or addresses); asynchronous on `stream`."""
        if N is None:
            N = T.shape[0]
        ck_source_terms(self.handle, T, P, Y, N, wdot, dTdt, stream)

    def source_terms_static(self, T, P, Y, wdot, dTdt, N=None, stream=0) -> None:
        """source_terms without any device allocation behind it (ck_source_terms_static): device buffers,
        asynchronous on `stream`; calls must not overlap on the GPU."""
        if N is None:
            N = T.shape[0]
        ck_source_terms_static(self.handle, T, P, Y, N, wdot, dTdt, stream)

    def jacobian(self, T, P, Y, J, N=None, stream=0) -> None:
        """J[N, S+1, S+1] = d(wdot, dT/dt)/d(Y, T) at constant P; device buffers; asynchronous."""
        if N is None:
            N = T.shape[0]
        ck_jacobian(self.handle, T, P, Y, N, J, stream)

    def source_terms_host(self, T, P, Y, wdot=None, dTdt=None, stream=0):
        """Host buffers (numpy or pinned torch CPU tensors); synchronous. Returns (wdot, dTdt)."""
        N = int(T.shape[0])
        if wdot is None:
            wdot = np.empty((self.S, N))
        if dTdt is None:
            dTdt = np.empty(N)
        ck_source_terms_host(self.handle, T, P, Y, N, wdot, dTdt, stream)
        return wdot, dTdt

    def rk4_integrate(self, T, P, Y, dt, n_steps, N=None, use_graph=True, stream=0) -> None:
        """n_steps explicit RK4 steps of the constant-pressure reactor, in place on the device
        buffers T[N], Y[S][N]; asynchronous on `stream`."""
        if N is None:
            N = T.shape[0]
        ck_rk4_integrate(self.handle, T, P, Y, N, dt, n_steps, use_graph, stream)

    def close(self) -> None:
        if getattr(self, "handle", None):
            ck_mech_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
