"""B200-native STEV (arxiv 1905.09395): stiff chemical kinetics integrated per cell by hand-written sm_100a kernels.

The package is a thin binding over the C ABI of include/stev.h (libstev_b200.so, built in-tree by `_build.py`).
"""
from .binding import (  # noqa: F401
    Mechanism, Estimator, StevError, load, lib_path, EXPORTS,
    stev_params, stev_params_default, stev_workspace_bytes, stev_integrate, stev_integrate_host, stev_integrate_finish, stev_integrate_static, STEV_STATIC_MAX_CELLS, stev_last_stats,
    stev_rates_eval, stev_estimator_eval, stev_compact_active, stev_dft_mag, stev_contract_exp_log, stev_microbench,
    stev_version, stev_last_error,
    STEV_OK, STEV_EINVAL, STEV_EWORKSPACE, STEV_ECUDA, STEV_WMAXSTEPS, STEV_WNONFINITE,
    STEV_PREC_FP32, STEV_PREC_TF32, STEV_PREC_BF16, STEV_STATE_FP64, STEV_STATE_FP32,
)
