"""Thin ctypes binding over libstev_b200.so: same names as include/stev.h, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch supplies device memory and streams.
There is no CPU fallback: if the shared library cannot be loaded the import fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import _build

STEV_OK, STEV_EINVAL, STEV_EWORKSPACE, STEV_ECUDA = 0, -1, -2, -3
STEV_WMAXSTEPS, STEV_WNONFINITE = 1, 2
STEV_PREC_FP32, STEV_PREC_TF32, STEV_PREC_BF16 = 0, 1, 2
STEV_STATE_FP64, STEV_STATE_FP32 = 0, 1


class stev_mechanism_desc(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_elements", C.c_int32), ("n_reactions", C.c_int32),
                ("mol_weight", C.c_void_p), ("elem_comp", C.c_void_p), ("nasa_lo", C.c_void_p), ("nasa_hi", C.c_void_p),
                ("t_mid", C.c_void_p), ("A", C.c_void_p), ("b", C.c_void_p), ("Ea", C.c_void_p), ("reversible", C.c_void_p),
                ("reac_ptr", C.c_void_p), ("reac_species", C.c_void_p), ("reac_nu", C.c_void_p),
                ("prod_ptr", C.c_void_p), ("prod_species", C.c_void_p), ("prod_nu", C.c_void_p),
                ("reac_coef", C.c_void_p), ("prod_coef", C.c_void_p), ("reac_order", C.c_void_p), ("prod_order", C.c_void_p)]


class stev_estimator_desc(C.Structure):
    _fields_ = [("n_in", C.c_int32), ("n_hidden", C.c_int32), ("n_out", C.c_int32), ("activation", C.c_int32),
                ("input_map", C.c_int32), ("in_shift", C.c_void_p), ("in_scale", C.c_void_p), ("W1", C.c_void_p),
                ("b1", C.c_void_p), ("W2", C.c_void_p), ("b2", C.c_void_p), ("h_ref_temperature", C.c_float)]


class stev_params(C.Structure):
    _fields_ = [("y_step_max", C.c_double), ("delta_max", C.c_double), ("alpha", C.c_double), ("tol_ring", C.c_double),
                ("tol_freq", C.c_double), ("r_fac", C.c_double), ("rof_min", C.c_double),
                ("dft_window", C.c_int32), ("dft_first_high_bin", C.c_int32), ("dft_enable", C.c_int32),
                ("max_steps", C.c_int32), ("energy_mode", C.c_int32), ("estimator_precision", C.c_int32),
                ("state_precision", C.c_int32), ("chunk_steps", C.c_int32), ("lanes_per_cell", C.c_int32),
                ("nonblocking", C.c_int32), ("order_cells", C.c_int32)]


class stev_stats(C.Structure):
    _fields_ = [("passes", C.c_int32), ("kernel_launches", C.c_int32), ("lanes_per_cell", C.c_int32),
                ("threads_per_block", C.c_int32), ("cells_per_block", C.c_int32), ("blocks", C.c_int32),
                ("smem_bytes", C.c_int64), ("total_steps", C.c_int64), ("specialised", C.c_int32), ("reserved", C.c_int32)]


EXPORTS = ["stev_params_default", "stev_mechanism_create", "stev_mechanism_destroy", "stev_mechanism_sizes",
           "stev_estimator_load", "stev_estimator_destroy", "stev_workspace_bytes", "stev_integrate",
           "stev_integrate_host", "stev_integrate_finish", "stev_integrate_static", "stev_last_stats", "stev_rates_eval", "stev_estimator_eval", "stev_compact_active",
           "stev_dft_mag", "stev_contract_exp_log", "stev_microbench", "stev_last_error", "stev_version"]

_lib = None


def lib_path() -> str:
    return _build.LIB


def load(build: bool = True):
    """Loads (building first if sources are newer) the CUDA library.  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if build and os.environ.get("STEV_NO_BUILD") != "1":
        try:
            _build.build()
        except Exception:
            # a stale library must not stand in for sources that no longer compile: only a box without nvcc may go on
            # with the library that travelled with the snapshot
            import shutil
            if shutil.which("nvcc") is not None or not os.path.exists(_build.LIB):
                raise
    if not os.path.exists(_build.LIB):
        raise ImportError(f"{_build.LIB} is missing: run `python -m paper_1905_09395_b200._build` (no CPU fallback exists)")
    lib = C.CDLL(_build.LIB)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.stev_params_default.argtypes = [C.POINTER(stev_params)]
    lib.stev_params_default.restype = None
    lib.stev_mechanism_create.argtypes = [C.POINTER(stev_mechanism_desc), C.POINTER(vp)]
    lib.stev_mechanism_destroy.argtypes = [vp]
    lib.stev_mechanism_destroy.restype = None
    lib.stev_mechanism_sizes.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
    lib.stev_estimator_load.argtypes = [vp, C.POINTER(stev_estimator_desc), C.POINTER(vp)]
    lib.stev_estimator_destroy.argtypes = [vp]
    lib.stev_estimator_destroy.restype = None
    lib.stev_workspace_bytes.argtypes = [vp, vp, C.POINTER(stev_params), i64]
    lib.stev_workspace_bytes.restype = C.c_size_t
    lib.stev_integrate.argtypes = [vp, vp, C.POINTER(stev_params), i64, i64, vp, vp, vp, dbl, vp, vp, vp, C.c_size_t, vp]
    lib.stev_integrate_host.argtypes = [vp, vp, C.POINTER(stev_params), i64, i64, vp, vp, vp, dbl, vp, vp]
    lib.stev_integrate_finish.argtypes = [vp, vp]
    lib.stev_integrate_static.argtypes = [vp, vp, C.POINTER(stev_params), i64, i64, vp, vp, vp, dbl, vp, vp, vp]
    lib.stev_last_stats.argtypes = [C.POINTER(stev_stats)]
    lib.stev_last_stats.restype = None
    lib.stev_rates_eval.argtypes = [vp, vp, C.POINTER(stev_params), i64, i64, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.stev_estimator_eval.argtypes = [vp, i64, vp, vp, i32, vp]
    lib.stev_compact_active.argtypes = [vp, vp, i32, vp, vp, vp, C.c_size_t, vp]
    lib.stev_dft_mag.argtypes = [vp, i64, vp, vp]
    lib.stev_contract_exp_log.argtypes = [vp, i64, vp, vp, vp]
    lib.stev_microbench.argtypes = [i32, i32, C.POINTER(dbl), vp]
    lib.stev_last_error.restype = C.c_char_p
    lib.stev_version.restype = C.c_char_p
    _lib = lib
    return lib


class StevError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"stev error {code}: {msg}")
        self.code = code


def _check(rc: int) -> int:
    if rc < 0:
        raise StevError(rc, load().stev_last_error().decode())
    return rc


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def stev_params_default(**overrides) -> stev_params:
    p = stev_params()
    load().stev_params_default(C.byref(p))
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise AttributeError(k)
        setattr(p, k, v)
    return p


class Mechanism:
    """Owner of a `stev_mechanism*` (stev_mechanism_create / stev_mechanism_destroy)."""

    def __init__(self, mech, validate_elements: bool = True):
        lib = load()
        a = dict(mol_weight=_np(mech.mol_weight, np.float64), nasa_lo=_np(mech.nasa_lo, np.float64),
                 nasa_hi=_np(mech.nasa_hi, np.float64), t_mid=_np(mech.t_mid, np.float64), A=_np(mech.A, np.float64),
                 b=_np(mech.b, np.float64), Ea=_np(mech.Ea, np.float64), reversible=_np(mech.reversible, np.uint8),
                 reac_ptr=_np(mech.reac_ptr, np.int32), reac_species=_np(mech.reac_species, np.int32),
                 reac_nu=_np(mech.reac_nu, np.int32), prod_ptr=_np(mech.prod_ptr, np.int32),
                 prod_species=_np(mech.prod_species, np.int32), prod_nu=_np(mech.prod_nu, np.int32))
        for k in ("reac_coef", "prod_coef", "reac_order", "prod_order"):
            if getattr(mech, k, None) is not None:
                a[k] = _np(getattr(mech, k), np.float64)
        ec = _np(mech.elem_comp, np.float64) if validate_elements and mech.elem_comp is not None else None
        d = stev_mechanism_desc(n_species=mech.n_species, n_elements=0 if ec is None else ec.shape[1],
                                n_reactions=mech.n_reactions, elem_comp=_p(ec), **{k: _p(v) for k, v in a.items()})
        h = C.c_void_p()
        _check(lib.stev_mechanism_create(C.byref(d), C.byref(h)))
        self.handle = h
        self.n_species, self.n_reactions = mech.n_species, mech.n_reactions

    def sizes(self):
        s, r, rr = C.c_int32(), C.c_int32(), C.c_int32()
        _check(load().stev_mechanism_sizes(self.handle, C.byref(s), C.byref(r), C.byref(rr)))
        return s.value, r.value, rr.value

    def close(self):
        if getattr(self, "handle", None):
            load().stev_mechanism_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Estimator:
    """Owner of a `stev_estimator*` (stev_estimator_load / stev_estimator_destroy)."""

    def __init__(self, mechanism: Mechanism | None, est):
        lib = load()
        a = dict(in_shift=_np(est.in_shift, np.float32), in_scale=_np(est.in_scale, np.float32), W1=_np(est.W1, np.float32),
                 b1=_np(est.b1, np.float32), W2=_np(est.W2, np.float32), b2=_np(est.b2, np.float32))
        d = stev_estimator_desc(n_in=est.n_in, n_hidden=est.n_hidden, n_out=est.n_out, activation=est.activation,
                                input_map=est.input_map, h_ref_temperature=est.h_ref_temperature,
                                **{k: _p(v) for k, v in a.items()})
        h = C.c_void_p()
        _check(lib.stev_estimator_load(mechanism.handle if mechanism else None, C.byref(d), C.byref(h)))
        self.handle = h
        self.mechanism = mechanism
        self.n_in, self.n_out = est.n_in, est.n_out

    def close(self):
        if getattr(self, "handle", None):
            load().stev_estimator_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _stream_ptr(stream) -> C.c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def stev_workspace_bytes(mechanism: Mechanism, estimator: Estimator | None, params: stev_params, n_cells: int) -> int:
    return int(load().stev_workspace_bytes(mechanism.handle, estimator.handle if estimator else None, C.byref(params), n_cells))


def stev_last_stats() -> dict:
    s = stev_stats()
    load().stev_last_stats(C.byref(s))
    return {k: getattr(s, k) for k, _ in stev_stats._fields_}


def stev_integrate(mechanism: Mechanism, estimator: Estimator | None, params: stev_params, T, p, Y, dt_cfd: float,
                   steps_out, status_out=None, workspace=None, stream=None) -> int:
    """Device tensors: T [N] f64 (in/out), p [N] f64, Y [S, ld] f64 (in/out), steps_out [N] i32, status_out [N] u8.
    Returns the C return code (0, STEV_WMAXSTEPS or STEV_WNONFINITE); raises StevError on failure."""
    import torch
    n = int(T.shape[0])
    assert T.is_cuda and T.dtype == torch.float64 and T.is_contiguous()
    assert p.is_cuda and p.dtype == torch.float64 and p.is_contiguous() and p.shape[0] == n
    assert Y.is_cuda and Y.dtype == torch.float64 and Y.dim() == 2 and (Y.stride(1) == 1 or Y.shape[1] <= 1) and Y.shape[0] == mechanism.n_species
    assert steps_out.is_cuda and steps_out.dtype == torch.int32 and steps_out.is_contiguous()
    ld = int(Y.stride(0)) if Y.shape[0] > 1 else int(Y.shape[1])
    need = stev_workspace_bytes(mechanism, estimator, params, n)
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=T.device)
    assert workspace.is_cuda
    rc = load().stev_integrate(mechanism.handle, estimator.handle if estimator else None, C.byref(params), n, ld,
                               T.data_ptr(), p.data_ptr(), Y.data_ptr(), float(dt_cfd), steps_out.data_ptr(),
                               status_out.data_ptr() if status_out is not None else None, workspace.data_ptr(),
                               workspace.numel() * workspace.element_size(), _stream_ptr(stream))
    return _check(rc)


STEV_STATIC_MAX_CELLS = 262144


def stev_integrate_static(mechanism: Mechanism, estimator: Estimator | None, params: stev_params, T, p, Y, dt_cfd: float,
                          steps_out, status_out=None, stream=None) -> int:
    """stev_integrate without a workspace: the scratch is a fixed device array inside the library, nothing is allocated
    (include/stev.h).  At most STEV_STATIC_MAX_CELLS cells; calls that overlap on one GPU race on the scratch."""
    import torch
    n = int(T.shape[0])
    assert T.is_cuda and T.dtype == torch.float64 and T.is_contiguous()
    assert p.is_cuda and p.dtype == torch.float64 and p.is_contiguous() and p.shape[0] == n
    assert Y.is_cuda and Y.dtype == torch.float64 and Y.dim() == 2 and (Y.stride(1) == 1 or Y.shape[1] <= 1) and Y.shape[0] == mechanism.n_species
    assert steps_out.is_cuda and steps_out.dtype == torch.int32 and steps_out.is_contiguous()
    ld = int(Y.stride(0)) if Y.shape[0] > 1 else int(Y.shape[1])
    rc = load().stev_integrate_static(mechanism.handle, estimator.handle if estimator else None, C.byref(params), n, ld,
                                      T.data_ptr(), p.data_ptr(), Y.data_ptr(), float(dt_cfd), steps_out.data_ptr(),
                                      status_out.data_ptr() if status_out is not None else None, _stream_ptr(stream))
    return _check(rc)


def stev_integrate_finish(workspace, stream=None) -> int:
    """After a nonblocking stev_integrate: synchronises the stream and returns the call's final return code."""
    return _check(load().stev_integrate_finish(workspace.data_ptr(), _stream_ptr(stream)))


def stev_integrate_host(mechanism: Mechanism, estimator: Estimator | None, params: stev_params, T, p, Y, dt_cfd: float,
                        steps_out, status_out=None) -> int:
    """Host numpy arrays (or pinned CPU torch tensors), in place: T [N], p [N], Y [S, N], steps_out [N] i32, status_out [N] u8."""
    def ptr(a):
        if a is None:
            return None
        return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
    n = int(T.shape[0])
    ld = int(Y.shape[1])
    rc = load().stev_integrate_host(mechanism.handle, estimator.handle if estimator else None, C.byref(params), n, ld,
                                    ptr(T), ptr(p), ptr(Y), float(dt_cfd), ptr(steps_out), ptr(status_out))
    return _check(rc)


def stev_rates_eval(mechanism: Mechanism, estimator: Estimator | None, params: stev_params, T, p, Y, rOF=None, stream=None):
    import torch
    n = int(T.shape[0])
    S, R, _ = mechanism.sizes()
    dY = torch.empty((S, n), dtype=torch.float64, device=T.device)
    dT = torch.empty(n, dtype=torch.float64, device=T.device)
    q = torch.empty((R, n), dtype=torch.float64, device=T.device)
    assert Y.is_contiguous() and Y.shape == (S, n)
    _check(load().stev_rates_eval(mechanism.handle, estimator.handle if estimator else None, C.byref(params), n, n,
                                  T.data_ptr(), p.data_ptr(), Y.data_ptr(), rOF.data_ptr() if rOF is not None else None,
                                  dY.data_ptr(), dT.data_ptr(), q.data_ptr(), _stream_ptr(stream)))
    return dY, dT, q


def stev_estimator_eval(estimator: Estimator, X, precision: int = STEV_PREC_FP32, stream=None):
    import torch
    assert X.is_cuda and X.dtype == torch.float32 and X.is_contiguous() and X.shape[1] == estimator.n_in
    out = torch.empty((X.shape[0], estimator.n_out), dtype=torch.float32, device=X.device)
    _check(load().stev_estimator_eval(estimator.handle, int(X.shape[0]), X.data_ptr(), out.data_ptr(), precision, _stream_ptr(stream)))
    return out


def stev_compact_active(flags, list_in=None, stream=None):
    import torch
    n = int(flags.shape[0])
    assert flags.is_cuda and flags.dtype == torch.uint8
    out = torch.empty(max(n, 1), dtype=torch.int32, device=flags.device)
    count = torch.zeros(1, dtype=torch.int32, device=flags.device)
    scratch = torch.empty(n // 1024 + 2, dtype=torch.int32, device=flags.device)
    _check(load().stev_compact_active(flags.data_ptr(), list_in.data_ptr() if list_in is not None else None, n, out.data_ptr(),
                                      count.data_ptr(), scratch.data_ptr(), scratch.numel() * 4, _stream_ptr(stream)))
    c = int(count.item())
    return out[:c], c


def stev_dft_mag(ring, stream=None):
    import torch
    assert ring.is_cuda and ring.dtype == torch.float64 and ring.is_contiguous() and ring.shape[1] == 13
    D = torch.empty((ring.shape[0], 7), dtype=torch.float64, device=ring.device)
    _check(load().stev_dft_mag(ring.data_ptr(), int(ring.shape[0]), D.data_ptr(), _stream_ptr(stream)))
    return D


def stev_contract_exp_log(x, stream=None):
    import torch
    assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
    e, l = torch.empty_like(x), torch.empty_like(x)
    _check(load().stev_contract_exp_log(x.data_ptr(), x.numel(), e.data_ptr(), l.data_ptr(), _stream_ptr(stream)))
    return e, l


def stev_microbench(kind: int, iters: int = 4096, stream=None) -> float:
    v = C.c_double()
    _check(load().stev_microbench(kind, iters, C.byref(v), _stream_ptr(stream)))
    return v.value


def stev_version() -> str:
    return load().stev_version().decode()


def stev_last_error() -> str:
    return load().stev_last_error().decode()
