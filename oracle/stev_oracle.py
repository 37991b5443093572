"""ctypes wrapper around oracle/stev_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It builds libstev_oracle.so with gcc on first use (build() of __graft_entry__ does the
same) and marshals numpy arrays; it contains no arithmetic of its own.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "stev_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "stev_oracle_f32.c")]
_DEPS = _SRCS + [os.path.join(_HERE, "stev_oracle_types.h")]
_LIB = os.path.join(_HERE, "libstev_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (no implicit FMA contraction: DESIGN.md section 5.1)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(d) for d in _DEPS):
        cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB, *_SRCS, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_variants = {}


def load_variant(define: str):
    """A second build of the same source with -D<define> (libstev_oracle_<define>.so), e.g. ORA_SENSITIVITY_ULP: the
    exp routine perturbed by one unit in the last place, for the self-sensitivity measurement of DESIGN.md section 5."""
    if define not in _variants:
        lib = os.path.join(_HERE, f"libstev_oracle_{define.lower()}.so")
        if not os.path.exists(lib) or os.path.getmtime(lib) < max(os.path.getmtime(d) for d in _DEPS):
            cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                   f"-D{define}", "-o", lib, *_SRCS, "-lm"]
            subprocess.run(cmd, check=True)
        _variants[define] = C.CDLL(lib)
    return _variants[define]


class _Mech(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_reactions", C.c_int32),
                ("mol_weight", C.c_void_p), ("nasa_lo", C.c_void_p), ("nasa_hi", C.c_void_p), ("t_mid", C.c_void_p),
                ("A", C.c_void_p), ("b", C.c_void_p), ("Ea", C.c_void_p), ("reversible", C.c_void_p),
                ("reac_ptr", C.c_void_p), ("reac_species", C.c_void_p), ("reac_nu", C.c_void_p),
                ("prod_ptr", C.c_void_p), ("prod_species", C.c_void_p), ("prod_nu", C.c_void_p),
                ("reac_coef", C.c_void_p), ("prod_coef", C.c_void_p), ("reac_order", C.c_void_p), ("prod_order", C.c_void_p)]


class _Est(C.Structure):
    _fields_ = [("n_in", C.c_int32), ("n_hidden", C.c_int32), ("n_out", C.c_int32), ("activation", C.c_int32),
                ("input_map", C.c_int32),
                ("in_shift", C.c_void_p), ("in_scale", C.c_void_p), ("W1", C.c_void_p), ("b1", C.c_void_p),
                ("W2", C.c_void_p), ("b2", C.c_void_p), ("h_ref_temperature", C.c_float)]


class _Params(C.Structure):
    _fields_ = [("y_step_max", C.c_double), ("delta_max", C.c_double), ("alpha", C.c_double),
                ("tol_ring", C.c_double), ("tol_freq", C.c_double), ("r_fac", C.c_double), ("rof_min", C.c_double),
                ("dft_first_high_bin", C.c_int32), ("dft_enable", C.c_int32), ("max_steps", C.c_int32),
                ("energy_mode", C.c_int32)]


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.ora_exp.restype = C.c_double
        _lib.ora_exp.argtypes = [C.c_double]
        _lib.ora_log.restype = C.c_double
        _lib.ora_log.argtypes = [C.c_double]
        for f in (_lib.ora_expf, _lib.ora_logf):
            f.restype = C.c_float
            f.argtypes = [C.c_float]
        _lib.ora_dft_bin_f32.restype = C.c_float
        _lib.ora_dft_bin_f32.argtypes = [C.c_void_p, C.c_int]
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class _Holder:
    """Keeps the numpy arrays alive next to the ctypes struct that borrows them."""

    def __init__(self, struct, arrays):
        self.struct = struct
        self.arrays = arrays


def _mech(m) -> _Holder:
    arrs = dict(
        mol_weight=np.ascontiguousarray(m.mol_weight, np.float64),
        nasa_lo=np.ascontiguousarray(m.nasa_lo, np.float64), nasa_hi=np.ascontiguousarray(m.nasa_hi, np.float64),
        t_mid=np.ascontiguousarray(m.t_mid, np.float64),
        A=np.ascontiguousarray(m.A, np.float64), b=np.ascontiguousarray(m.b, np.float64),
        Ea=np.ascontiguousarray(m.Ea, np.float64), reversible=np.ascontiguousarray(m.reversible, np.uint8),
        reac_ptr=np.ascontiguousarray(m.reac_ptr, np.int32), reac_species=np.ascontiguousarray(m.reac_species, np.int32),
        reac_nu=np.ascontiguousarray(m.reac_nu, np.int32),
        prod_ptr=np.ascontiguousarray(m.prod_ptr, np.int32), prod_species=np.ascontiguousarray(m.prod_species, np.int32),
        prod_nu=np.ascontiguousarray(m.prod_nu, np.int32))
    for k in ("reac_coef", "prod_coef", "reac_order", "prod_order"):
        v = getattr(m, k, None)
        if v is not None:
            arrs[k] = np.ascontiguousarray(v, np.float64)
    s = _Mech(n_species=m.n_species, n_reactions=m.n_reactions, **{k: _ptr(v) for k, v in arrs.items()})
    return _Holder(s, arrs)


def _est(e) -> _Holder | None:
    if e is None:
        return None
    assert e.n_in <= 64 and e.n_hidden <= 256 and e.n_out <= 512
    arrs = dict(in_shift=np.ascontiguousarray(e.in_shift, np.float32), in_scale=np.ascontiguousarray(e.in_scale, np.float32),
                W1=np.ascontiguousarray(e.W1, np.float32), b1=np.ascontiguousarray(e.b1, np.float32),
                W2=np.ascontiguousarray(e.W2, np.float32), b2=np.ascontiguousarray(e.b2, np.float32))
    s = _Est(n_in=e.n_in, n_hidden=e.n_hidden, n_out=e.n_out, activation=e.activation, input_map=e.input_map,
             h_ref_temperature=e.h_ref_temperature, **{k: _ptr(v) for k, v in arrs.items()})
    return _Holder(s, arrs)


def _params(p: dict) -> _Params:
    return _Params(**p)


def exp(x: float) -> float:
    return _load().ora_exp(float(x))


def log(x: float) -> float:
    return _load().ora_log(float(x))


def expf(x: float) -> float:
    return _load().ora_expf(float(x))


def logf(x: float) -> float:
    return _load().ora_logf(float(x))


def dft_mag_f32(ring) -> np.ndarray:
    lib = _load()
    r = np.ascontiguousarray(ring, np.float32)
    assert r.shape == (13,)
    return np.array([lib.ora_dft_bin_f32(_ptr(r), m) for m in range(7)], np.float32)


def thermo(mech, T: float):
    """cp/R, h/RT, s/R of every species at temperature T (NASA-7)."""
    lib = _load()
    mh = _mech(mech)
    S = mech.n_species
    cp, h, s = np.empty(S), np.empty(S), np.empty(S)
    lib.ora_thermo(C.byref(mh.struct), C.c_double(T), _ptr(cp), _ptr(h), _ptr(s))
    return cp, h, s


def dft_mag(ring) -> np.ndarray:
    lib = _load()
    r = np.ascontiguousarray(ring, np.float64)
    assert r.shape == (13,)
    D = np.empty(7)
    lib.ora_dft_mag(_ptr(r), _ptr(D))
    return D


def estimator_eval(est, X) -> np.ndarray:
    lib = _load()
    eh = _est(est)
    X = np.ascontiguousarray(X, np.float32)
    out = np.empty((X.shape[0], est.n_out), np.float32)
    lib.ora_estimator_eval(C.byref(eh.struct), C.c_int64(X.shape[0]), _ptr(X), _ptr(out))
    return out


def rates_eval(mech, est, params: dict, T, p, Y, rOF=None, precision: str = "f64"):
    """Right-hand side of n cells. Y is [S, n] species-major. Returns dYdt [S,n], dTdt [n], q [R,n]."""
    lib = _load()
    mh, eh, pr = _mech(mech), _est(est), _params(params)
    T = np.ascontiguousarray(T, np.float64)
    p = np.ascontiguousarray(p, np.float64)
    Y = np.ascontiguousarray(Y, np.float64)
    n = T.shape[0]
    S, R = mech.n_species, mech.n_reactions
    assert Y.shape == (S, n)
    dY, dT, q = np.empty((S, n)), np.empty(n), np.empty((R, n))
    rof = None if rOF is None else np.ascontiguousarray(rOF, np.float64)
    (lib.ora_rates_eval if precision == "f64" else lib.ora_rates_eval_f32)(C.byref(mh.struct), C.byref(eh.struct) if eh else None, C.byref(pr), C.c_int64(n), C.c_int64(n),
                       _ptr(T), _ptr(p), _ptr(Y), _ptr(rof) if rof is not None else None, _ptr(dY), _ptr(dT), _ptr(q))
    return dY, dT, q


def integrate(mech, est, params: dict, T, p, Y, dt_cfd: float, n_threads: int | None = None, variant: str | None = None,
              precision: str = "f64"):
    """Advance n cells over dt_cfd. Inputs are copied. Returns dict(T, Y, steps, status, rof_min, rc)."""
    lib = load_variant(variant) if variant else _load()
    mh, eh, pr = _mech(mech), _est(est), _params(params)
    T = np.array(T, np.float64, copy=True)
    p = np.ascontiguousarray(p, np.float64)
    Y = np.array(Y, np.float64, copy=True, order="C")
    n = T.shape[0]
    assert Y.shape == (mech.n_species, n)
    steps = np.zeros(n, np.int32)
    status = np.zeros(n, np.uint8)
    rof_min = np.ones(n)
    if n_threads is None:
        n_threads = os.cpu_count() or 1
    rc = (lib.ora_integrate if precision == "f64" else lib.ora_integrate_f32)(C.byref(mh.struct), C.byref(eh.struct) if eh else None, C.byref(pr), C.c_int64(n),
                           C.c_int64(n), _ptr(T), _ptr(p), _ptr(Y), C.c_double(dt_cfd), _ptr(steps), _ptr(status),
                           _ptr(rof_min), C.c_int32(n_threads))
    return dict(T=T, Y=Y, steps=steps, status=status, rof_min=rof_min, rc=rc, n_threads=n_threads)


def integrate_trace(mech, est, params: dict, T: float, p: float, Y, dt_cfd: float, trace_cap: int = 100000,
                    precision: str = "f64"):
    """One cell with a per-step trace: rows (t, h, T, Y[0..S), rOF[0..R))."""
    lib = _load()
    mh, eh, pr = _mech(mech), _est(est), _params(params)
    S, R = mech.n_species, mech.n_reactions
    Yc = np.array(Y, np.float64, copy=True)
    Tc = C.c_double(T)
    steps = C.c_int32(0)
    trace = np.zeros((trace_cap, 3 + S + R))
    st = (lib.ora_integrate_trace if precision == "f64" else lib.ora_integrate_trace_f32)(C.byref(mh.struct), C.byref(eh.struct) if eh else None, C.byref(pr), C.byref(Tc),
                                 C.c_double(p), _ptr(Yc), C.c_double(dt_cfd), C.byref(steps), _ptr(trace),
                                 C.c_int64(trace_cap))
    n = min(steps.value, trace_cap)
    tr = trace[:n]
    return dict(status=st, steps=steps.value, T=Tc.value, Y=Yc, t=tr[:, 0], h=tr[:, 1], T_trace=tr[:, 2],
                Y_trace=tr[:, 3:3 + S], rOF_trace=tr[:, 3 + S:])
