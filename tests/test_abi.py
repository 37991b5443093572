"""The C-ABI library loads and exports every symbol include/stev.h declares (no compute without a GPU)."""
import ctypes
import os
import re

import paper_1905_09395_b200 as stev

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "stev.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(stev_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = stev.load()
    names = _declared_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/stev.h but not exported"
    assert sorted(stev.EXPORTS) == names


def test_binding_has_the_same_names():
    for n in _declared_symbols():
        if n in ("stev_mechanism_create", "stev_mechanism_destroy", "stev_mechanism_sizes"):
            assert hasattr(stev.Mechanism, "__init__")
        elif n in ("stev_estimator_load", "stev_estimator_destroy"):
            assert hasattr(stev.Estimator, "__init__")
        else:
            assert hasattr(stev, n), n


def test_params_default_and_struct_layout():
    p = stev.stev_params_default()
    assert p.y_step_max == 1e-2 and p.delta_max == 1e-2 and p.alpha == 1e-5
    assert p.tol_ring == 0.5 and p.tol_freq == 0.1 and p.r_fac == 2.0 and p.rof_min == 2.0 ** -100
    assert p.dft_first_high_bin == 4 and p.dft_enable == 1 and p.max_steps == 200000
    assert p.chunk_steps == 0 and p.lanes_per_cell == 0 and p.order_cells == 1
    assert p.dft_window == 13 and p.estimator_precision == stev.STEV_PREC_FP32 and p.state_precision == 0 and p.nonblocking == 0
    assert ctypes.sizeof(stev.stev_params) == 7 * 8 + 12 * 4   # seven doubles, eleven int32 fields padded to a multiple of 8
    assert stev.stev_version().startswith("stev-b200")


def test_argument_validation_without_gpu():
    lib = stev.load()
    assert lib.stev_mechanism_create(None, None) == stev.STEV_EINVAL
    assert b"null" in lib.stev_last_error()
    assert lib.stev_integrate(None, None, None, 0, 0, None, None, None, 1e-4, None, None, None, 0, None) == stev.STEV_EINVAL
    assert lib.stev_integrate_static(None, None, None, 0, 0, None, None, None, 1e-4, None, None, None) == stev.STEV_EINVAL
