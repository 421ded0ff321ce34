"""CPU oracle for the batched chemical source term -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  The product (paper_2008_08483_b200) never does.  The arithmetic
lives in ck_oracle.c (plain C, fp64, one cell and one reaction at a time; citations in
ck_oracle.h); this file only marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import build as _build

_dp = C.POINTER(C.c_double)
_bp = C.POINTER(C.c_uint8)


class _Ann(C.Structure):
    _fields_ = [("n_in", C.c_int32), ("n_layers", C.c_int32), ("n_hidden", C.c_int32),
                ("activation", C.c_int32), ("in_mean", _dp), ("in_std", _dp), ("W_in", _dp),
                ("B", _dp), ("W_hid", _dp), ("W_out", _dp), ("B_out", _dp), ("out_mean", _dp),
                ("out_std", _dp)]


class _Mech(C.Structure):
    _fields_ = [
        ("S", C.c_int32), ("R", C.c_int32),
        ("W", _dp), ("nu_reac", _dp), ("nu_prod", _dp),
        ("ln_A", _dp), ("b", _dp), ("Ea_over_R", _dp), ("reversible", _bp),
        ("nasa_lo", _dp), ("nasa_hi", _dp), ("T_mid", _dp), ("rxn_type", _bp),
        ("eff", _dp), ("ln_A0", _dp), ("b0", _dp), ("Ea0_over_R", _dp), ("troe", _dp),
        ("p_ref", C.c_double), ("kc_ann", C.POINTER(_Ann)),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        # (CK_ORACLE_LIB: another build of the same sources, e.g. the sanitizer build of oracle/build.py)
        lib = C.CDLL(os.environ.get("CK_ORACLE_LIB") or _build())
        lib.ck_oracle_source_terms.restype = C.c_int
        lib.ck_oracle_source_terms.argtypes = [C.POINTER(_Mech), _dp, _dp, _dp, C.c_int64,
                                               _dp, _dp, C.c_int]
        lib.ck_oracle_cell_detail.restype = None
        lib.ck_oracle_cell_detail.argtypes = ([C.POINTER(_Mech), C.c_double, C.c_double, _dp,
                                               C.c_int64] + [_dp] * 16)
        lib.ck_oracle_jacobian.restype = C.c_int
        lib.ck_oracle_jacobian.argtypes = [C.POINTER(_Mech), _dp, _dp, _dp, C.c_int64, _dp, C.c_int]
        _lib = lib
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _u8(a):
    return np.ascontiguousarray(a, dtype=np.uint8)


class OracleMechanism:
    """Holds C-contiguous copies of a ckgen.Mechanism's arrays and the C struct."""

    def __init__(self, mech, kc_ann=None):
        """kc_ann: None (exact Kc) or an object with ckgen.KcAnn's attributes (approximate ANN
        for log Kc)."""
        self.S, self.R = mech.n_species, mech.n_reactions
        self._keep = dict(
            W=_f64(mech.mol_weight), nu_reac=_f64(mech.nu_reac), nu_prod=_f64(mech.nu_prod),
            ln_A=_f64(mech.ln_A), b=_f64(mech.b), Ea_over_R=_f64(mech.Ea_over_R),
            reversible=_u8(mech.reversible), nasa_lo=_f64(mech.nasa_lo),
            nasa_hi=_f64(mech.nasa_hi), T_mid=_f64(mech.T_mid), rxn_type=_u8(mech.rxn_type),
            eff=_f64(mech.eff), ln_A0=_f64(mech.ln_A0), b0=_f64(mech.b0),
            Ea0_over_R=_f64(mech.Ea0_over_R), troe=_f64(mech.troe),
        )
        k = self._keep
        assert k["nu_reac"].shape == (self.S, self.R) and k["eff"].shape == (self.S, self.R)
        assert k["nasa_lo"].shape == (self.S, 7) and k["troe"].shape == (self.R, 4)
        s = _Mech()
        s.S, s.R, s.p_ref = self.S, self.R, float(mech.p_ref)
        for name, arr in k.items():
            ptr_t = _bp if arr.dtype == np.uint8 else _dp
            setattr(s, name, arr.ctypes.data_as(ptr_t))
        if kc_ann is not None:
            NL, NH, NI = int(kc_ann.n_layers), int(kc_ann.n_hidden), int(kc_ann.n_in)
            ka = dict(in_mean=_f64(kc_ann.in_mean), in_std=_f64(kc_ann.in_std), W_in=_f64(kc_ann.W_in),
                      B=_f64(kc_ann.B), W_hid=_f64(kc_ann.W_hid), W_out=_f64(kc_ann.W_out),
                      B_out=_f64(kc_ann.B_out), out_mean=_f64(kc_ann.out_mean), out_std=_f64(kc_ann.out_std))
            assert ka["W_in"].shape == (NI, NH) and ka["B"].shape == (NL, NH)
            assert ka["W_hid"].shape == (NL - 1, NH, NH) and ka["W_out"].shape == (NH, self.R)
            assert ka["in_mean"].shape == (NI,) and ka["out_std"].shape == (self.R,)
            a = _Ann()
            a.n_in, a.n_layers, a.n_hidden, a.activation = NI, NL, NH, int(kc_ann.activation)
            for name, arr in ka.items():
                setattr(a, name, arr.ctypes.data_as(_dp))
            self._keep_ann, self._ann = ka, a
            s.kc_ann = C.pointer(a)
        self.c = s


def source_terms(omech: OracleMechanism, T, P, Y, nthreads: int = 0):
    """(wdot[S,N], dTdt[N], threads_used) for T[N], P[N], Y[S,N]."""
    T, P, Y = _f64(T), _f64(P), _f64(Y)
    N = T.shape[0]
    assert P.shape == (N,) and Y.shape == (omech.S, N)
    wdot = np.empty((omech.S, N))
    dTdt = np.empty(N)
    used = _load().ck_oracle_source_terms(
        C.byref(omech.c), T.ctypes.data_as(_dp), P.ctypes.data_as(_dp), Y.ctypes.data_as(_dp),
        N, wdot.ctypes.data_as(_dp), dTdt.ctypes.data_as(_dp), int(nthreads))
    return wdot, dTdt, used


def cell_detail(omech: OracleMechanism, T: float, P: float, Y):
    """Every intermediate of one cell as a dict of numpy arrays / floats."""
    Y = _f64(Y)
    assert Y.shape == (omech.S,)
    S, R = omech.S, omech.R
    sc = {n: C.c_double() for n in ("rho", "cp_mass", "dTdt")}
    per_s = {n: np.empty(S) for n in ("C", "cp_R", "h_RT", "s_R", "g_RT", "wdot")}
    per_r = {n: np.empty(R) for n in ("kf", "Kc", "kr", "M", "qf", "qr", "Q")}
    p = lambda a: a.ctypes.data_as(_dp)
    _load().ck_oracle_cell_detail(
        C.byref(omech.c), float(T), float(P), p(Y), 1,
        C.cast(C.byref(sc["rho"]), _dp), C.cast(C.byref(sc["cp_mass"]), _dp),
        p(per_s["C"]), p(per_s["cp_R"]), p(per_s["h_RT"]), p(per_s["s_R"]), p(per_s["g_RT"]),
        p(per_r["kf"]), p(per_r["Kc"]), p(per_r["kr"]), p(per_r["M"]), p(per_r["qf"]),
        p(per_r["qr"]), p(per_r["Q"]), p(per_s["wdot"]), C.cast(C.byref(sc["dTdt"]), _dp))
    out = {k: v.value for k, v in sc.items()}
    out.update(per_s)
    out.update(per_r)
    return out


def jacobian(omech: OracleMechanism, T, P, Y, nthreads: int = 0):
    """J[N, S+1, S+1] = d(wdot_0..wdot_{S-1}, dT/dt) / d(Y_0..Y_{S-1}, T) at constant P
    (ck_oracle_jac.c), for T[N], P[N], Y[S,N]."""
    T, P, Y = _f64(T), _f64(P), _f64(Y)
    N = T.shape[0]
    assert P.shape == (N,) and Y.shape == (omech.S, N)
    J = np.empty((N, omech.S + 1, omech.S + 1))
    used = _load().ck_oracle_jacobian(
        C.byref(omech.c), T.ctypes.data_as(_dp), P.ctypes.data_as(_dp), Y.ctypes.data_as(_dp),
        N, J.ctypes.data_as(_dp), int(nthreads))
    if used < 0:
        raise ValueError("the oracle Jacobian does not support the approximate-ANN Kc")
    return J
