"""Pins for real stoichiometric coefficients and rate-law exponents (Eqs 26-30: the BFER-shaped
mechanism; reading R22).  The constants of Table 1 are the paper's; the thermodynamics are synthetic."""
import numpy as np
import pytest

from stev_inputs.configs import default_params, make_workload
from stev_inputs.mechanisms import P_ATM, R_CAL, R_U, bfer_shaped_field, bfer_shaped_mechanism
from tests.helpers import nasa_numpy, numpy_rhs, rate_constants_numpy


def _params(**kw):
    p = default_params()
    p.update(kw)
    return p


def test_table_1_constants_are_the_papers():
    m = bfer_shaped_mechanism()
    np.testing.assert_array_equal(m.A, [4.9e9, 2.0e8])          # PAPER.md:222-225 (Table 1)
    np.testing.assert_array_equal(m.Ea, [35500.0, 12000.0])
    np.testing.assert_array_equal(m.b, [0.0, 0.7])              # Eq 29: T^0.7
    np.testing.assert_array_equal(m.reac_order, [0.5, 0.65, 1.0, 0.5])   # Eqs 28, 29
    np.testing.assert_array_equal(m.reac_coef, [1.0, 1.5, 1.0, 0.5])     # Eqs 26, 27
    assert np.abs(m.stoich_matrix() @ m.elem_comp).max() == 0.0          # both reactions conserve H, O, C, N


def test_rates_are_the_printed_rate_laws(oracle):
    """Eq 28: r = k exp(-Ea/RT) C_CH4^0.5 C_O2^0.65;  Eq 29: r = k T^0.7 exp(-Ea/RT) (C_CO C_O2^0.5 - C_CO2/K), K of Eq 30
    with Delta N = -0.5 -- written out with numpy's power and exponential on the same concentrations."""
    m = bfer_shaped_mechanism()
    T, p, Y = bfer_shaped_field(64)
    _, _, q = oracle.rates_eval(m, None, _params(alpha=0.0), T, p, Y)
    for c in range(64):
        rho = p[c] / (R_U * T[c]) / np.sum(Y[:, c] / m.mol_weight)
        C = rho * Y[:, c] / m.mol_weight
        q0 = 4.9e9 * np.exp(-35500.0 / (R_CAL * T[c])) * C[0] ** 0.5 * C[1] ** 0.65
        _, h, s = nasa_numpy(m, T[c])
        g = h - s
        K = (P_ATM / (R_U * T[c])) ** (-0.5) * np.exp(-(g[4] - g[2] - 0.5 * g[1]))
        q1 = 2.0e8 * T[c] ** 0.7 * np.exp(-12000.0 / (R_CAL * T[c])) * (C[2] * C[1] ** 0.5 - C[4] / K)
        assert abs(q[0, c] / q0 - 1.0) < 1e-12
        assert abs(q[1, c] - q1) <= 1e-12 * max(abs(q1), 2.0e8 * T[c] ** 0.7 * np.exp(-12000.0 / (R_CAL * T[c])) * C[2] * C[1] ** 0.5)
    # the whole right-hand side against the matrix-form numpy RHS (real coefficients in the source terms, orders in the rates)
    dY, dT, _ = oracle.rates_eval(m, None, _params(alpha=0.0), T, p, Y)
    for c in range(0, 64, 7):
        dYn, dTn, _ = numpy_rhs(m, T[c], p[c], Y[:, c])
        np.testing.assert_allclose(dY[:, c], dYn, rtol=1e-11, atol=1e-11 * np.abs(dYn).max())
        assert abs(dT[c] - dTn) <= 1e-10 * abs(dTn)


def test_order_is_the_logarithmic_derivative(oracle):
    """d ln q / d ln C_i = order_i (Eq 28): scaling p scales every concentration by the same factor lam at fixed T and Y,
    so q_MEPOX scales by lam^(0.5 + 0.65)."""
    m = bfer_shaped_mechanism()
    T, p, Y = bfer_shaped_field(16)
    _, _, q1 = oracle.rates_eval(m, None, _params(alpha=0.0), T, p, Y)
    _, _, q2 = oracle.rates_eval(m, None, _params(alpha=0.0), T, 1.001 * p, Y)
    slope = np.log(q2[0] / q1[0]) / np.log(1.001)
    np.testing.assert_allclose(slope, 1.15, atol=1e-9)


@pytest.mark.parametrize("config", [1, 2])
def test_integer_orders_given_as_reals_reproduce_the_integer_path_bit_for_bit(oracle, config):
    import dataclasses
    w = make_workload(config, 48)
    m = w.mech
    as_real = dataclasses.replace(m, reac_coef=m.reac_nu.astype(float), prod_coef=m.prod_nu.astype(float),
                                  reac_order=m.reac_nu.astype(float), prod_order=m.prod_nu.astype(float))
    a = oracle.integrate(m, None, w.params, w.T, w.p, w.Y, w.dt_cfd)
    b = oracle.integrate(as_real, None, w.params, w.T, w.p, w.Y, w.dt_cfd)
    for k in ("T", "Y", "steps", "status"):
        np.testing.assert_array_equal(a[k], b[k])


def test_integration_conserves_and_matches_a_stiff_library_integrator(oracle):
    from scipy.integrate import solve_ivp
    m = bfer_shaped_mechanism()
    T, p, Y = bfer_shaped_field(24)
    t_f = 1.0e-3                                              # "an integration final time of 1 millisecond"
    r = oracle.integrate(m, None, _params(), T, p, Y, t_f)
    assert (r["status"] == 0).all() and r["steps"].max() > 150     # the limiter is at work on the hot cells
    assert np.abs(r["Y"].sum(axis=0) - 1.0).max() < 1e-12
    zW = m.elem_comp / m.mol_weight[:, None]
    assert np.abs(zW.T @ r["Y"] - zW.T @ Y).max() < 1e-12
    assert r["Y"].min() > -1e-15
    for c in (0, 5, 11, 17):
        def f(t, x):
            dY, dT, _ = numpy_rhs(m, x[0], p[c], np.maximum(x[1:], 0.0))
            return np.concatenate([[dT], dY])
        sol = solve_ivp(f, (0, t_f), np.concatenate([[T[c]], Y[:, c]]), method="Radau", rtol=1e-9, atol=1e-13)
        assert sol.success
        assert np.abs(r["Y"][:, c] - sol.y[1:, -1]).max() < 1e-2
        assert abs(r["T"][c] - sol.y[0, -1]) < 1e-2 * sol.y[0, -1]


def test_vanished_reactant_stops_the_reaction(oracle):
    """R22: C^x = 0 for C <= 0, so a cell without fuel has q_MEPOX = 0 exactly and keeps it."""
    m = bfer_shaped_mechanism()
    Y = np.array([[0.0], [0.2], [0.0], [0.0], [0.0], [0.8]])
    _, _, q = oracle.rates_eval(m, None, _params(), np.array([1800.0]), np.array([P_ATM]), Y)
    assert q[0, 0] == 0.0 and q[1, 0] == 0.0
    r = oracle.integrate(m, None, _params(), [1800.0], [P_ATM], Y, 1e-3)
    np.testing.assert_array_equal(r["Y"], Y)
    assert r["steps"][0] == 100
