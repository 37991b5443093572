"""Pins for the oracle's rate evaluation (P4, P5 and an independent matrix-form cross-check)."""
import math

import numpy as np
import pytest

from stev_inputs.configs import default_params, make_mechanism
from stev_inputs.mechanisms import P_ATM, R_CAL, R_U
from tests.helpers import build_mechanism, flat_thermo, numpy_rhs, rate_constants_numpy


def _params(**kw):
    p = default_params()
    p.update(kw)
    return p


def test_Kc_dnu_zero_reduces_to_exp_minus_dG(oracle):
    """P5 / Eq 30: dN = 0 => K = exp(-dG/RT).  A <=> B with a6, a7 set by hand:
    g/RT = cp(1 - ln T) + a6/T - a7 ; dG/RT = (a6_B - a6_A)/T - (a7_B - a7_A)."""
    lo, hi = flat_thermo(2, 3.5, a6=[0.0, -2000.0], a7=[5.0, 4.0])
    mech = build_mechanism([28.0, 28.0], lo, hi, [([(0, 1)], [(1, 1)], 1e3, 0.0, 0.0, 1)])
    T, p = 1250.0, P_ATM
    K = math.exp(-(-2000.0 / T - (4.0 - 5.0)))
    # at Y_B / Y_A = K the net rate vanishes; elsewhere q = k_f (C_A - C_B / K)
    Y = np.array([[1.0 / (1.0 + K)], [K / (1.0 + K)]])
    _, _, q = oracle.rates_eval(mech, None, _params(alpha=0.0), [T], [p], Y)
    C = p / (R_U * T)
    assert abs(q[0, 0]) <= 1e-12 * 1e3 * C * Y[0, 0]
    Y = np.array([[0.7], [0.3]])
    _, _, q = oracle.rates_eval(mech, None, _params(alpha=0.0), [T], [p], Y)
    assert abs(q[0, 0] - 1e3 * C * (0.7 - 0.3 / K)) <= 1e-13 * 1e3 * C


def test_Kc_dnu_plus_one_hand_calculation(oracle):
    """P5: A <=> 2 B has dN = +1: K_c = (p_atm / R_u T) exp(-dG/RT)."""
    lo, hi = flat_thermo(2, 3.0, a6=[-8000.0, 0.0], a7=[6.0, 5.0])
    mech = build_mechanism([40.0, 20.0], lo, hi, [([(0, 1)], [(1, 2)], 1e5, 0.0, 0.0, 1)])
    T, p = 1500.0, 2.0 * P_ATM
    gA = 3.0 * (1 - math.log(T)) - 8000.0 / T - 6.0
    gB = 3.0 * (1 - math.log(T)) - 5.0
    Kc = (P_ATM / (R_U * T)) * math.exp(-(2 * gB - gA))
    Y = np.array([[0.4], [0.6]])
    rho = p / (R_U * T) / (0.4 / 40 + 0.6 / 20)
    CA, CB = rho * 0.4 / 40, rho * 0.6 / 20
    _, _, q = oracle.rates_eval(mech, None, _params(alpha=0.0), [T], [p], Y)
    ref = 1e5 * (CA - CB * CB / Kc)
    assert abs(q[0, 0] - ref) <= 1e-12 * abs(1e5 * CA)


@pytest.mark.parametrize("config", [1, 2, 3])
def test_rates_against_matrix_form_numpy(oracle, config):
    """Eqs 28-30 evaluated with stoichiometric matrices and numpy exp/log (alpha = 0): catches a wrong sign,
    index, transposed operand or dropped term anywhere in the oracle's CSR loops."""
    mech = make_mechanism(config)
    rng = np.random.default_rng(11 + config)
    n = 16
    T = rng.uniform(800, 2500, n)
    p = rng.uniform(1, 5, n) * P_ATM
    Y = np.ascontiguousarray(rng.dirichlet(np.ones(mech.n_species), n).T)
    dY, dT, q = oracle.rates_eval(mech, None, _params(alpha=0.0), T, p, Y)
    for c in range(n):
        dY_n, dT_n, q_n = numpy_rhs(mech, T[c], p[c], Y[:, c])
        scale = np.abs(q_n).max()
        np.testing.assert_allclose(q[:, c], q_n, rtol=1e-9, atol=1e-10 * scale)
        np.testing.assert_allclose(dY[:, c], dY_n, rtol=1e-8, atol=1e-10 * np.abs(dY_n).max())
        assert abs(dT[c] - dT_n) <= 1e-8 * abs(dT_n) + 1e-6


def test_forward_reverse_ratio_is_Kc(oracle):
    """P4: k_f / k_r = K_c.  With only products present q = -k_r prod C; with only reactants q = k_f prod C."""
    lo, hi = flat_thermo(4, 3.5, a6=[-1000.0, -3000.0, -2500.0, -500.0], a7=[5.0, 6.0, 4.5, 7.0])
    mech = build_mechanism([10.0, 30.0, 25.0, 15.0], lo, hi, [([(0, 1), (1, 1)], [(2, 1), (3, 1)], 3e12, 0.5, 20000.0, 1)])
    T, p = 1800.0, P_ATM
    kf, Kc = rate_constants_numpy(mech, T)
    prm = _params(alpha=0.0)
    Yr = np.array([[0.5], [0.5], [0.0], [0.0]])
    Yp = np.array([[0.0], [0.0], [0.5], [0.5]])
    _, _, qf = oracle.rates_eval(mech, None, prm, [T], [p], Yr)
    _, _, qr = oracle.rates_eval(mech, None, prm, [T], [p], Yp)
    rho_r = p / (R_U * T) / (0.5 / 10 + 0.5 / 30)
    rho_p = p / (R_U * T) / (0.5 / 25 + 0.5 / 15)
    kf_o = qf[0, 0] / ((rho_r * 0.5 / 10) * (rho_r * 0.5 / 30))
    kr_o = -qr[0, 0] / ((rho_p * 0.5 / 25) * (rho_p * 0.5 / 15))
    assert abs(kf_o / kf[0] - 1) < 1e-12
    assert abs(kf_o / kr_o / Kc[0] - 1) < 1e-12


def test_gamma_stabilisation(oracle):
    """Eqs 6-7: y -> gamma(y) y, gamma = y/(alpha+y); unity for y >> alpha, zero for y << alpha."""
    lo, hi = flat_thermo(2, 3.5)
    mech = build_mechanism([28.0, 28.0], lo, hi, [([(0, 1)], [(1, 1)], 1e3, 0.0, 0.0, 0)])
    T, p, alpha = 1000.0, P_ATM, 1e-5
    C = p / (R_U * T)
    for yA in [0.5, 1e-5, 1e-9]:
        Y = np.array([[yA], [1 - yA]])
        _, _, q = oracle.rates_eval(mech, None, _params(alpha=alpha), [T], [p], Y)
        ref = 1e3 * C * yA * yA / (alpha + yA)
        assert abs(q[0, 0] - ref) <= 1e-13 * ref
    Y = np.array([[-1e-9], [1 + 1e-9]])            # negative mass fraction is clamped inside the rate only (R7)
    dY, _, q = oracle.rates_eval(mech, None, _params(alpha=alpha), [T], [p], Y)
    assert q[0, 0] == 0.0 and dY[0, 0] == 0.0


def test_rof_scales_reversible_rates_only(oracle):
    """Eq 14: r_eff = r_rev * rOF, irreversible reactions untouched."""
    mech = make_mechanism(1)
    rng = np.random.default_rng(5)
    Y = np.ascontiguousarray(rng.dirichlet(np.ones(9), 3).T)
    T, p = np.array([1200.0, 1600.0, 2000.0]), np.full(3, P_ATM)
    _, _, q1 = oracle.rates_eval(mech, None, _params(), T, p, Y)
    rof = np.full((mech.n_reactions, 3), 0.25)
    _, _, q2 = oracle.rates_eval(mech, None, _params(), T, p, Y, rOF=rof)
    rev = mech.reversible == 1
    np.testing.assert_array_equal(q2[rev], 0.25 * q1[rev])
    np.testing.assert_array_equal(q2[~rev], q1[~rev])


def test_source_terms_conserve_mass_and_elements(oracle):
    """P3 at the rate level: sum_i dY_i/dt = 0 and element moles sum_i a_ei (dY_i/dt)/W_i = 0."""
    for config in [1, 2, 3]:
        mech = make_mechanism(config)
        rng = np.random.default_rng(config)
        n = 8
        Y = np.ascontiguousarray(rng.dirichlet(np.ones(mech.n_species), n).T)
        dY, _, _ = oracle.rates_eval(mech, None, _params(), rng.uniform(900, 2400, n), np.full(n, P_ATM), Y)
        scale = np.abs(dY).max(axis=0)
        assert np.all(np.abs(dY.sum(axis=0)) <= 1e-12 * scale)
        elem = mech.elem_comp.T @ (dY / mech.mol_weight[:, None])
        assert np.all(np.abs(elem) <= 1e-12 * scale / mech.mol_weight.min())
