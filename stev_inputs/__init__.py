"""Seeded synthetic inputs for the STEV hot path (mechanisms, cell fields, estimator weights).

This module serves both the CPU oracle (tests) and the CUDA library (tests, bench).  It holds no
solver arithmetic: it only draws mechanisms, thermodynamic tables, initial states and MLP weights
from `numpy.random.default_rng(seed)`.  The recipe is stated in DESIGN.md section 6 and stands in
for the paper's workloads (random fixed thermochemical states at growing cell counts,
PAPER.md:231; mechanism sizes up to GRI-Mech's 53/325), whose real inputs are not
available here.
"""
from .mechanisms import Mechanism, abc_mechanism, synthetic_mechanism  # noqa: F401
from .estimators import Estimator, fit_estimator  # noqa: F401
from .configs import Workload, make_workload, default_params, N_CONFIGS, shard_cells  # noqa: F401
