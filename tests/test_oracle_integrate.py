"""Pins for the oracle's STEV loop: closed forms, convergence, conservation, limiter / timing / rOF
properties, stiff-reversible damping and brute-force comparison (P1-P3, P6, P8-P12)."""
import math

import numpy as np
import pytest

from stev_inputs.configs import default_params, make_mechanism, make_workload
from stev_inputs.mechanisms import P_ATM, R_U
from tests.helpers import build_mechanism, flat_thermo, nasa_numpy, numpy_rhs, rate_constants_numpy


def _params(**kw):
    p = default_params()
    p.update(kw)
    return p


def _ab_mechanism(kf, a6B=-1500.0, extra=None):
    lo, hi = flat_thermo(3, 3.5, a6=[0.0, a6B, -4000.0], a7=[5.0, 5.0, 5.0])
    rx = [([(0, 1)], [(1, 1)], kf, 0.0, 0.0, 1)]
    if extra:
        rx += extra
    return build_mechanism([28.0, 28.0, 28.0], lo, hi, rx)


# ---------------------------------------------------------------- P1 / P2
def test_P1_discrete_euler_closed_form(oracle):
    """A <=> B isothermal, alpha = 0, DFT off, limiter idle: every step has h = t_f delta_max, so
    A_n = A_eq + (A_0 - A_eq)(1 - (k_f + k_r) h)^n  with n = 1/delta_max (Eq 18 applied to a linear ODE)."""
    T, t_f = 1200.0, 1e-4
    mech = _ab_mechanism(kf=8000.0)
    kf, Kc = rate_constants_numpy(mech, T)
    kr = kf[0] / Kc[0]
    prm = _params(alpha=0.0, dft_enable=0, y_step_max=1.0, energy_mode=1)
    Y0 = np.array([[0.9], [0.1], [0.0]])
    r = oracle.integrate(mech, None, prm, [T], [P_ATM], Y0, t_f)
    assert r["steps"][0] == 100 and r["status"][0] == 0
    A_eq = 1.0 * kr / (kf[0] + kr)
    h = t_f * 0.01
    A_n = A_eq + (0.9 - A_eq) * (1 - (kf[0] + kr) * h) ** 100
    assert abs(r["Y"][0, 0] - A_n) < 1e-13
    assert abs(r["Y"][1, 0] - (1.0 - A_n)) < 1e-13
    assert r["T"][0] == T


def test_P2_first_order_convergence_to_continuous_solution(oracle):
    T, t_f = 1200.0, 1e-4
    mech = _ab_mechanism(kf=8000.0)
    kf, Kc = rate_constants_numpy(mech, T)
    lam = kf[0] + kf[0] / Kc[0]
    A_eq = (kf[0] / Kc[0]) / lam
    exact = A_eq + (0.9 - A_eq) * math.exp(-lam * t_f)
    errs = []
    for dmax in [0.01, 0.005, 0.0025]:
        prm = _params(alpha=0.0, dft_enable=0, y_step_max=1.0, energy_mode=1, delta_max=dmax)
        r = oracle.integrate(mech, None, prm, [T], [P_ATM], np.array([[0.9], [0.1], [0.0]]), t_f)
        assert r["steps"][0] == round(1 / dmax)
        errs.append(r["Y"][0, 0] - exact)
    assert 1.95 < errs[0] / errs[1] < 2.05 and 1.95 < errs[1] / errs[2] < 2.05


# ---------------------------------------------------------------- P3
@pytest.mark.parametrize("config,n", [(0, 256), (1, 96), (2, 48), (3, 24)])
def test_P3_mass_and_element_conservation_with_stabilisers_on(oracle, config, n):
    w = make_workload(config, n)
    r = oracle.integrate(w.mech, w.estimator, w.params, w.T, w.p, w.Y, w.dt_cfd)
    assert (r["status"] == 0).all()
    assert np.max(np.abs(r["Y"].sum(axis=0) - 1.0)) < 1e-12
    e0 = w.mech.elem_comp.T @ (w.Y / w.mech.mol_weight[:, None])
    e1 = w.mech.elem_comp.T @ (r["Y"] / w.mech.mol_weight[:, None])
    assert np.max(np.abs(e1 - e0)) < 1e-12
    assert r["Y"].min() > -1e-15 and r["Y"].max() < 1 + 1e-12      # PAPER.md:53 "between zero and unity"


# ---------------------------------------------------------------- P6 brute force / library integrator
def _reference_solution(mech, T0, p, Y0, t_f):
    from scipy.integrate import solve_ivp

    def f(t, x):
        dY, dT, _ = numpy_rhs(mech, x[0], p, x[1:])
        return np.concatenate([[dT], dY])
    sol = solve_ivp(f, (0, t_f), np.concatenate([[T0], Y0]), method="Radau", rtol=1e-8, atol=1e-12)
    assert sol.success
    return sol.y[0, -1], sol.y[1:, -1]


def test_P6_against_library_stiff_integrator_and_tiny_step_euler(oracle):
    """STEV (defaults) vs scipy Radau of the unstabilised ODE on the 3-species config-0 system, and vs forward
    Euler with a step far below the stability limit on the mildest cell (the brute-force definition)."""
    w = make_workload(0, 4096)
    idx = [0, 100, 2000]
    r = oracle.integrate(w.mech, None, w.params, w.T[idx], w.p[idx], w.Y[:, idx], w.dt_cfd)
    errY, errT = [], []
    for k, c in enumerate(idx):
        T_ref, Y_ref = _reference_solution(w.mech, w.T[c], w.p[c], w.Y[:, c], w.dt_cfd)
        errY.append(np.abs(r["Y"][:, k] - Y_ref).max())
        errT.append(abs(r["T"][k] - T_ref) / T_ref)
    assert max(errY) < 1e-2 and max(errT) < 5e-3
    # brute force: A <=> B + slow drain, non-stiff rates, 40 000 Euler steps of the plain ODE
    mech = _ab_mechanism(kf=5.0e4, extra=[([(0, 1)], [(2, 1)], 3.0e3, 0.0, 0.0, 0)])
    T, Yc, n_bf = 1100.0, np.array([0.6, 0.3, 0.1]), 40000
    hb = 1e-4 / n_bf
    for _ in range(n_bf):
        dY, dT, _ = numpy_rhs(mech, T, P_ATM, Yc)
        Yc = Yc + hb * dY
        T = T + hb * dT
    errs = []
    for dmax, ysm in [(0.01, 1e-2), (0.005, 5e-3)]:
        rr = oracle.integrate(mech, None, _params(delta_max=dmax, y_step_max=ysm), [1100.0], [P_ATM],
                              np.array([[0.6], [0.3], [0.1]]), 1e-4)
        errs.append(np.abs(rr["Y"][:, 0] - Yc).max())
        assert abs(rr["T"][0] - T) < 5e-3 * T
    assert errs[0] < 1e-2 and errs[1] < 0.7 * errs[0]        # shrinks ~first order


# ---------------------------------------------------------------- P8 / P9 / P10 from per-step traces
@pytest.mark.parametrize("config,cells", [(0, [0, 7, 99]), (1, [0, 5]), (2, [1, 2])])
def test_P8_P9_P10_limiter_timing_and_rof_properties(oracle, config, cells):
    w = make_workload(config, 128)
    for c in cells:
        tr = oracle.integrate_trace(w.mech, None, w.params, w.T[c], w.p[c], w.Y[:, c], w.dt_cfd)
        assert tr["status"] == 0
        Yt = np.vstack([w.Y[:, c][None, :], tr["Y_trace"]])
        cons = Yt[:-1] - Yt[1:]                                  # consumption per step
        cap = np.minimum(w.params["y_step_max"], np.where(Yt[:-1] < 1e-20, 1.0, 0.9 * Yt[:-1]))
        assert np.all(cons <= cap * (1 + 1e-12) + 1e-300)        # PAPER.md:53 (Eq 3)
        assert Yt.min() >= -1e-15
        assert tr["t"][-1] == w.dt_cfd                           # lands on t_f exactly
        assert np.all(np.diff(tr["t"]) > 0)
        assert np.all(tr["h"] <= w.dt_cfd * w.params["delta_max"] * (1 + 1e-15))   # Eq 4-5
        assert tr["steps"] >= round(1 / w.params["delta_max"])
        rof = tr["rOF_trace"]
        assert rof.max() <= 1.0 and rof.min() >= w.params["rof_min"]     # PAPER.md:95, R13
        m, e = np.frexp(rof)
        assert np.all(m == 0.5)                                  # r_fac = 2: rOF is always 2^-k
        irreversible = w.mech.reversible == 0
        assert np.all(rof[:, irreversible] == 1.0)


def test_P9_non_reacting_cell_takes_exactly_one_over_delta_max_steps(oracle):
    mech = _ab_mechanism(kf=1e-30)
    for dmax in [0.01, 0.002]:
        r = oracle.integrate(mech, None, _params(delta_max=dmax), [1000.0], [P_ATM], np.array([[0.5], [0.3], [0.2]]), 1e-4)
        assert r["steps"][0] == round(1 / dmax) and r["status"][0] == 0
        np.testing.assert_allclose(r["Y"][:, 0], [0.5, 0.3, 0.2], atol=1e-30)


def test_P10_rof_stays_one_on_monotone_relaxation(oracle):
    """rOF 'will not decline unless the reversible rate is both ringing and at equilibrium'."""
    for kf in [5.0e3, 2.0e4, 1.0e5]:
        mech = _ab_mechanism(kf=kf)
        tr = oracle.integrate_trace(mech, None, _params(energy_mode=1), 1200.0, P_ATM, np.array([0.9, 0.1, 0.0]), 1e-4)
        assert tr["status"] == 0 and np.all(tr["rOF_trace"][:, 0] == 1.0)
        assert np.all(np.diff(tr["Y_trace"][:, 0]) <= 0)          # A relaxes monotonically


def test_max_steps_status_and_irreversible_infinite_stiffness(oracle):
    """an arbitrarily stiff irreversible reaction is integrable; R20: max_steps gives status 1."""
    lo, hi = flat_thermo(2, 3.5)
    mech = build_mechanism([28.0, 28.0], lo, hi, [([(0, 1)], [(1, 1)], 1e18, 0.0, 0.0, 0)])
    r = oracle.integrate(mech, None, _params(energy_mode=1), [1000.0], [P_ATM], np.array([[1.0], [0.0]]), 1e-4)
    assert r["status"][0] == 0 and r["steps"][0] < 1000 and r["Y"][0, 0] < 1e-6 and r["Y"][0, 0] >= 0
    r = oracle.integrate(mech, None, _params(energy_mode=1, max_steps=50), [1000.0], [P_ATM], np.array([[1.0], [0.0]]), 1e-4)
    assert r["status"][0] == 1 and r["steps"][0] == 50 and r["rc"] == 1


# ---------------------------------------------------------------- P11 stiff reversible damping
@pytest.mark.parametrize("kf", [1e7, 1e9, 1e11, 1e13])
def test_P11_stiff_reversible_reaction_is_damped(oracle, kf):
    """A <=> B with k from 1e7 to 1e13 1/s plus a slow drain A -> C: with the DFT stabiliser the integration
    finishes in a few hundred steps at every stiffness and matches the partial-equilibrium solution; without it
    (k >= 1e9) it does not finish within 50 000 steps."""
    kd, T, t_f = 5.0e2, 1200.0, 1e-4
    mech = _ab_mechanism(kf=kf, extra=[([(0, 1)], [(2, 1)], kd, 0.0, 0.0, 0)])
    _, Kc = rate_constants_numpy(mech, T)
    Y0 = np.array([[0.5], [0.5], [0.0]])
    r = oracle.integrate(mech, None, _params(energy_mode=1, max_steps=50000), [T], [P_ATM], Y0, t_f)
    assert r["status"][0] == 0
    assert r["steps"][0] <= 2.5 * 100
    # partial equilibrium: B = K A at all times, (A + B) decays at rate kd / (1 + K)
    K = Kc[0]
    ab = math.exp(-kd / (1 + K) * t_f)
    ref = np.array([ab / (1 + K), ab * K / (1 + K), 1 - ab])
    assert np.abs(r["Y"][:, 0] - ref).max() < 1e-3
    if kf >= 1e9:
        r_off = oracle.integrate(mech, None, _params(energy_mode=1, max_steps=50000, dft_enable=0), [T], [P_ATM], Y0, t_f)
        assert r_off["status"][0] == 1
    assert r["rof_min"][0] < 1.0 or kf < 1e9


# ---------------------------------------------------------------- P12 enthalpy
def test_P12_adiabatic_enthalpy_drift_is_first_order(oracle):
    """Constant-pressure adiabatic reading (R15): mixture enthalpy sum_i Y_i h_i(T)/W_i is conserved by the ODE,
    so the Euler drift is O(h) and halves with delta_max."""
    w = make_workload(0, 64)
    c = 5

    def H(T, Y):
        _, h, _ = nasa_numpy(w.mech, T)
        return np.sum(Y * h * R_U * T / w.mech.mol_weight)
    H0 = H(w.T[c], w.Y[:, c])
    drift = []
    for dmax, ysm in [(0.01, 1e-2), (0.005, 5e-3), (0.0025, 2.5e-3)]:
        r = oracle.integrate(w.mech, None, _params(delta_max=dmax, y_step_max=ysm), [w.T[c]], [w.p[c]], w.Y[:, [c]], w.dt_cfd)
        drift.append(abs(H(r["T"][0], r["Y"][:, 0]) - H0))
    cpT = 4.5 * R_U * w.T[c] / 28.0
    assert drift[0] < 2e-2 * cpT
    assert drift[1] < 0.75 * drift[0] and drift[2] < 0.75 * drift[1]


def test_isothermal_mode_keeps_T(oracle):
    w = make_workload(1, 8)
    r = oracle.integrate(w.mech, None, _params(energy_mode=1), w.T, w.p, w.Y, w.dt_cfd)
    np.testing.assert_array_equal(r["T"], w.T)


def test_mlp_estimator_run_is_close_to_nasa_run_on_benign_config(oracle):
    """Config-0-like benign chemistry: swapping NASA cp,h for the fitted MLP moves T by well
    under 1 % (paper: ANN within 0.436 % of the polynomial)."""
    from stev_inputs.estimators import fit_estimator
    w = make_workload(0, 32)
    est = fit_estimator(w.mech, 16, seed=3)
    a = oracle.integrate(w.mech, None, w.params, w.T, w.p, w.Y, w.dt_cfd)
    b = oracle.integrate(w.mech, est, w.params, w.T, w.p, w.Y, w.dt_cfd)
    assert np.max(np.abs(a["T"] - b["T"]) / a["T"]) < 1e-2
    assert np.max(np.abs(a["Y"] - b["Y"])) < 2e-2
