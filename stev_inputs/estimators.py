"""Shallow-MLP property estimator weights.

The paper trains its one-hidden-layer network with a Levenberg-Marquardt solver;
that trainer is offline and out of scope.  Here the hidden layer is drawn from the seed and the
linear output layer is a ridge least-squares fit to the mechanism's NASA-7 polynomials
(BASELINE.json configs 3 and 4: "weights least-squares fitted to the seeded NASA-7 polynomials on
T in [300,3000] K").  Outputs: cp_i/R (first S) and h_i/(R * h_ref_temperature) (next S).
"""
from __future__ import annotations

import dataclasses

import numpy as np

from .mechanisms import Mechanism, P_ATM

ACT_TANH, ACT_SIGMOID = 0, 1
IN_T, IN_T_P_Y = 0, 1


@dataclasses.dataclass
class Estimator:
    n_in: int
    n_hidden: int
    n_out: int
    activation: int
    input_map: int
    in_shift: np.ndarray  # float32 [n_in]
    in_scale: np.ndarray  # float32 [n_in]
    W1: np.ndarray  # float32 [H, n_in]
    b1: np.ndarray  # float32 [H]
    W2: np.ndarray  # float32 [n_out, H]
    b2: np.ndarray  # float32 [n_out]
    h_ref_temperature: float = 1000.0


def _nasa_targets(mech: Mechanism, T: np.ndarray, h_ref: float) -> np.ndarray:
    """[n, 2S] training targets from the NASA-7 tables (numpy polynomial evaluation)."""
    S = mech.n_species
    out = np.empty((T.size, 2 * S))
    for i in range(S):
        a = np.where((T < mech.t_mid[i])[:, None], mech.nasa_lo[i][None, :], mech.nasa_hi[i][None, :])
        cp = a[:, 0] + a[:, 1] * T + a[:, 2] * T**2 + a[:, 3] * T**3 + a[:, 4] * T**4
        h_rt = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T**2 / 3 + a[:, 3] * T**3 / 4 + a[:, 4] * T**4 / 5 + a[:, 5] / T
        out[:, i] = cp
        out[:, S + i] = h_rt * T / h_ref
    return out


def fit_estimator(mech: Mechanism, n_hidden: int, seed: int, input_map: int = IN_T,
                  activation: int = ACT_TANH, n_samples: int = 4096, ridge: float = 1e-6,
                  sample_inputs: np.ndarray | None = None) -> Estimator:
    """Hidden layer ~ U[-3,3] from the seed; output layer by ridge least squares.

    `sample_inputs` ([n, n_in] raw inputs) lets config 4 fit on its own input distribution; by
    default T is uniform on [300, 3000] K (and p, Y columns are drawn like config 4's field)."""
    rng = np.random.default_rng(seed)
    S = mech.n_species
    n_in = 1 if input_map == IN_T else 2 + S
    shift = np.zeros(n_in)
    scale = np.ones(n_in)
    shift[0], scale[0] = 1650.0, 1.0 / 1350.0
    if input_map == IN_T_P_Y:
        shift[1], scale[1] = 3.0 * P_ATM, 1.0 / (2.0 * P_ATM)
    W1 = rng.uniform(-3.0, 3.0, (n_hidden, n_in))
    if input_map == IN_T_P_Y:
        W1[:, 1:] = rng.uniform(-0.05, 0.05, (n_hidden, n_in - 1))  # weak p, Y dependence
    b1 = rng.uniform(-3.0, 3.0, n_hidden)
    if sample_inputs is None:
        raw = np.zeros((n_samples, n_in))
        raw[:, 0] = rng.uniform(300.0, 3000.0, n_samples)
        if input_map == IN_T_P_Y:
            raw[:, 1] = rng.uniform(1.0, 5.0, n_samples) * P_ATM
            raw[:, 2:] = rng.dirichlet(np.full(S, 0.5), n_samples)
    else:
        raw = np.asarray(sample_inputs, dtype=np.float64)
    x = (raw - shift) * scale
    z = x @ W1.T + b1
    hid = np.tanh(z) if activation == ACT_TANH else 1.0 / (1.0 + np.exp(-z))
    Phi = np.concatenate([hid, np.ones((hid.shape[0], 1))], axis=1)
    h_ref = 1000.0
    tgt = _nasa_targets(mech, raw[:, 0], h_ref)
    G = Phi.T @ Phi / Phi.shape[0]
    G += ridge * np.trace(G) / G.shape[0] * np.eye(G.shape[0])
    coef = np.linalg.solve(G, Phi.T @ tgt / Phi.shape[0])  # [H+1, 2S]
    return Estimator(n_in=n_in, n_hidden=n_hidden, n_out=2 * S, activation=activation, input_map=input_map,
                     in_shift=shift.astype(np.float32), in_scale=scale.astype(np.float32),
                     W1=W1.astype(np.float32), b1=b1.astype(np.float32),
                     W2=np.ascontiguousarray(coef[:-1].T.astype(np.float32)), b2=coef[-1].astype(np.float32),
                     h_ref_temperature=h_ref)
