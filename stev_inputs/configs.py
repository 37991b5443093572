"""The five BASELINE.json workloads made concrete.

Fields are generated in independent blocks of BLOCK cells, block k seeded by [field_seed, k], so any
subset of blocks (a parity subsample, one rank's shard) is reproducible without generating the rest.
"""
from __future__ import annotations

import dataclasses
import os

import numpy as np

from .mechanisms import Mechanism, abc_mechanism, synthetic_mechanism, P_ATM
from .estimators import Estimator, fit_estimator, IN_T, IN_T_P_Y

N_CONFIGS = 5
BLOCK = 4096
BASE_SEED = 190509395

FULL_CELLS = [4096, 65536, 262144, 1048576, 4194304]
DT_CFD = [1e-4, 1e-4, 5e-5, 1e-4, 1e-4]
# One recorded scalar multiplying every A of configs 2-4 (DESIGN.md section 6 "tractability"):
# STEV cannot integrate the larger random mechanisms at config 1's rate-constant range in a
# bounded number of steps (the paper concedes the same for GRI-Mech).
STIFFNESS_SCALE = [1.0, 1.0, 1.0, 1.0e-5, 1.0]


def default_params() -> dict:
    """Solver constants: readings R3, R4, R7, R10, R12, R13, R20 of DESIGN.md section 3."""
    return dict(y_step_max=1.0e-2, delta_max=1.0e-2, alpha=1.0e-5, tol_ring=0.5, tol_freq=0.1, r_fac=2.0,
                rof_min=2.0 ** -100, dft_first_high_bin=4, dft_enable=1, max_steps=200000, energy_mode=0)


@dataclasses.dataclass
class Workload:
    config: int
    name: str
    mech: Mechanism
    estimator: Estimator | None
    params: dict
    dt_cfd: float
    T: np.ndarray  # [N]
    p: np.ndarray  # [N]
    Y: np.ndarray  # [S, N] species-major
    blocks: np.ndarray  # the global block indices held

    @property
    def n_cells(self) -> int:
        return int(self.T.shape[0])


_MECH_CACHE: dict = {}


def make_mechanism(config: int) -> Mechanism:
    if config in _MECH_CACHE:
        return _MECH_CACHE[config]
    seed = BASE_SEED + 10 * config
    if config == 0:
        m = abc_mechanism(seed)
    elif config == 1:
        m = synthetic_mechanism(9, 19, 2, seed, STIFFNESS_SCALE[1], inert_last=False)
    elif config in (2, 4):
        m = synthetic_mechanism(20, 60, 3, BASE_SEED + 20, STIFFNESS_SCALE[2], inert_last=True)
    elif config == 3:
        m = synthetic_mechanism(53, 325, 4, seed, STIFFNESS_SCALE[3], inert_last=True)
    else:
        raise ValueError("config must be 0..4")
    _MECH_CACHE[config] = m
    return m


def make_estimator(config: int, mech: Mechanism) -> Estimator | None:
    seed = BASE_SEED + 10 * config + 2
    if config == 3:
        return fit_estimator(mech, 32, seed, IN_T)
    if config == 4:
        return fit_estimator(mech, 64, seed, IN_T_P_Y)
    return None


def _relaxed_pool() -> np.ndarray:
    """Near-equilibrium states for config 2 ([512, 20] mass fractions), written once by
    oracle/make_relaxed_pool.py (the CPU oracle relaxes random states at 1000 K for 20 dt_cfd)."""
    path = os.path.join(os.path.dirname(__file__), "data", "relaxed_pool_cfg2.npy")
    return np.load(path)


def _field_block(config: int, S: int, k: int, n: int):
    rng = np.random.default_rng([BASE_SEED + 10 * config + 1, k])
    if config == 0:
        T = rng.uniform(900.0, 1500.0, n)
        Y = rng.dirichlet(np.ones(S), n)
        p = np.full(n, P_ATM)
    elif config == 1:
        T = rng.uniform(800.0, 2200.0, n)
        Y = rng.dirichlet(np.ones(S), n)
        p = np.full(n, P_ATM)
    elif config == 2:
        pool = _relaxed_pool()
        hot = rng.random(n) >= 0.6  # cell order is already interleaved hot / near-equilibrium
        T = np.where(hot, rng.uniform(1500.0, 2500.0, n), 1000.0 + rng.uniform(-5.0, 5.0, n))
        Yhot = rng.dirichlet(np.ones(S), n)
        Yeq = pool[rng.integers(0, pool.shape[0], n)] * (1.0 + 1e-3 * rng.standard_normal((n, S)))
        Yeq = np.abs(Yeq)
        Yeq /= Yeq.sum(axis=1, keepdims=True)
        Y = np.where(hot[:, None], Yhot, Yeq)
        p = rng.uniform(1.0, 5.0, n) * P_ATM
    elif config == 3:
        T = rng.uniform(1000.0, 2500.0, n)
        Y = rng.dirichlet(np.ones(S), n)
        p = np.full(n, P_ATM)
    else:
        T = rng.uniform(1000.0, 2500.0, n)
        Y = rng.dirichlet(np.full(S, 0.5), n)
        inert = rng.random(n) < 0.25
        y_in = rng.uniform(0.9, 0.99, n)
        rest = Y[:, :-1] / np.maximum(Y[:, :-1].sum(axis=1, keepdims=True), 1e-300)
        Yi = np.concatenate([rest * (1.0 - y_in)[:, None], y_in[:, None]], axis=1)
        Y = np.where(inert[:, None], Yi, Y)
        p = rng.uniform(1.0, 5.0, n) * P_ATM
    return T, p, Y


def shard_cells(n_blocks_total: int, rank: int, world: int) -> np.ndarray:
    """Interleaved block partition: rank r holds blocks r, r+world, ... (stiff cells cluster in space,
    PAPER.md:416, so slabs balance badly; cells are independent, so no exchange)."""
    return np.arange(rank, n_blocks_total, world, dtype=np.int64)


def make_workload(config: int, n_cells: int | None = None, rank: int = 0, world: int = 1,
                  weak: bool = True) -> Workload:
    """Workload `config` (0..4).  `n_cells` (default: BASELINE's full size) is the PER-RANK cell count
    when weak (the global field then has n_cells*world cells, rank r holding the interleaved blocks
    r, r+world, ...), else the global count split over ranks."""
    mech = make_mechanism(config)
    est = make_estimator(config, mech)
    S = mech.n_species
    n = FULL_CELLS[config] if n_cells is None else int(n_cells)
    n_global = n * world if weak else n
    n_blocks = (n_global + BLOCK - 1) // BLOCK
    blocks = shard_cells(n_blocks, rank, world)
    Ts, ps, Ys = [], [], []
    for k in blocks:
        nb = min(BLOCK, n_global - int(k) * BLOCK)
        T, p, Y = _field_block(config, S, int(k), nb)
        Ts.append(T); ps.append(p); Ys.append(Y)
    T = np.concatenate(Ts) if Ts else np.zeros(0)
    p = np.concatenate(ps) if ps else np.zeros(0)
    Y = np.concatenate(Ys, axis=0) if Ys else np.zeros((0, S))
    names = ["cfg0_abc_4096", "cfg1_9sp19rx_65536", "cfg2_20sp60rx_bimodal_262144",
             "cfg3_53sp325rx_mlp_1048576", "cfg4_20sp60rx_multiphase_mlp_4194304"]
    return Workload(config=config, name=names[config], mech=mech, estimator=est, params=default_params(),
                    dt_cfd=DT_CFD[config], T=np.ascontiguousarray(T), p=np.ascontiguousarray(p),
                    Y=np.ascontiguousarray(Y.T), blocks=blocks)
