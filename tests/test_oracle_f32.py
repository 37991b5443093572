"""Pins for the oracle's binary32 mode (oracle/stev_oracle_f32.c; the paper solved the thermochemical
state in 32-bit precision).  The same closed forms and invariants as the binary64 mode at float tolerances, its exp / log
against libm, and the binary64 oracle at the paper's own accuracy scale (per-cell differences of 1e-4 relative,
PAPER.md:237)."""
import math

import numpy as np
import pytest

from stev_inputs.configs import default_params, make_workload
from stev_inputs.mechanisms import P_ATM, bfer_shaped_field, bfer_shaped_mechanism
from tests.helpers import build_mechanism, flat_thermo, rate_constants_numpy
from tests.test_oracle_step_logic import _expected_rof, _slow_reversible

F32 = dict(precision="f32")


def _params(**kw):
    p = default_params()
    p.update(kw)
    return p


def _ulp32(x):
    return float(np.spacing(np.float32(abs(x))))


def test_exp_log_float_within_two_ulp_of_libm_and_saturate(oracle):
    rng = np.random.default_rng(32)
    for x in np.concatenate([rng.uniform(-87, 88, 4000), rng.uniform(-1, 1, 1000), [0.0, 88.0, -87.0, 1e-8]]).astype(np.float32):
        ref = math.exp(float(x))
        assert abs(oracle.expf(float(x)) - ref) <= 2.0 * _ulp32(ref), x
    assert oracle.expf(88.5) == math.inf and oracle.expf(-87.5) == 0.0 and math.isnan(oracle.expf(float("nan")))
    for x in np.concatenate([10.0 ** rng.uniform(-37, 38, 4000), rng.uniform(0.5, 2.0, 1000), [1.0, 2.0 ** 0.5]]).astype(np.float32):
        ref = math.log(float(x))
        assert abs(oracle.logf(float(x)) - ref) <= 2.0 * max(_ulp32(ref), 2.0 ** -24 * 0.35), x
    assert oracle.logf(1.0) == 0.0 and oracle.logf(0.0) == -math.inf and math.isnan(oracle.logf(-1.0))
    # functional equation on exactly representable shifts: exp(x + ln 2 k) = 2^k exp(x) up to the reduction's rounding
    for x in (0.1, 1.7, -3.3):
        assert abs(oracle.expf(x + 5 * math.log(2.0)) / oracle.expf(x) / 32.0 - 1.0) < 1e-6


def test_dft_float_against_numpy_fft_and_closed_forms(oracle):
    rng = np.random.default_rng(13)
    for _ in range(50):
        ring = (rng.standard_normal(13) * 10.0 ** rng.uniform(-12, 0)).astype(np.float32)
        D = oracle.dft_mag_f32(ring)
        ref = np.abs(np.fft.rfft(ring.astype(np.float64)))
        np.testing.assert_allclose(D, ref, rtol=0, atol=4e-6 * np.abs(ring).sum())
    D = oracle.dft_mag_f32(0.37 * (-1.0) ** np.arange(13))
    for m in range(7):
        assert abs(D[m] - 0.37 / abs(math.cos(math.pi * m / 13))) < 3e-6
    np.testing.assert_allclose(oracle.dft_mag_f32(np.ones(13))[1:], 0.0, atol=2e-6)


def test_P1_discrete_euler_closed_form_in_float(oracle):
    lo, hi = flat_thermo(3, 3.5, a6=[0.0, -1500.0, -4000.0], a7=[5.0, 5.0, 5.0])
    mech = build_mechanism([28.0] * 3, lo, hi, [([(0, 1)], [(1, 1)], 8000.0, 0.0, 0.0, 1)])
    T, t_f = 1200.0, 1e-4
    kf, Kc = rate_constants_numpy(mech, T)
    kr = kf[0] / Kc[0]
    r = oracle.integrate(mech, None, _params(alpha=0.0, dft_enable=0, y_step_max=1.0, energy_mode=1), [T], [P_ATM],
                         np.array([[0.9], [0.1], [0.0]]), t_f, **F32)
    assert r["steps"][0] == 100 and r["status"][0] == 0 and r["T"][0] == T
    A_eq = kr / (kf[0] + kr)
    A_n = A_eq + (0.9 - A_eq) * (1 - (kf[0] + kr) * t_f * 0.01) ** 100
    assert abs(r["Y"][0, 0] - A_n) < 2e-6 and abs(r["Y"][1, 0] - (1.0 - A_n)) < 2e-6


def test_limiter_closed_form_in_float(oracle):
    """The binary32 twin of test_limiter_picks_exactly_min_ystepmax_ninety_percent."""
    k, t_f, ysm = 1.0e8, 1.0e-4, 1.0e-2
    lo, hi = flat_thermo(2, 3.5)
    mech = build_mechanism([28.0, 28.0], lo, hi, [([(0, 1)], [(1, 1)], k, 0.0, 0.0, 0)])
    tr = oracle.integrate_trace(mech, None, _params(alpha=0.0, dft_enable=0, energy_mode=1), 1000.0, P_ATM,
                                np.array([0.505, 0.495]), t_f, **F32)
    assert tr["status"] == 0 and tr["steps"] == 168
    yA = np.concatenate([[np.float32(0.505)], tr["Y_trace"][:, 0]])
    for n in range(0, 51):
        assert abs(yA[n] - (0.505 - ysm * n)) < 5e-6
    for n in range(0, 50):
        assert abs(tr["h"][n] / (ysm / (k * yA[n])) - 1.0) < 2e-6
    for m in range(1, 17):
        assert abs(yA[51 + m] / yA[50 + m] - 0.1) < 1e-6         # ninety percent per step (Eq 2)
    assert tr["t"][-1] == np.float32(t_f)


@pytest.mark.parametrize("tol_ring,tol_freq_over_a,n_hf", [(1.5, 1e30, 4), (2.5, 1e30, 4), (1.5, 1e30, 1), (1e30, 0.5, 4),
                                                            (1e30, 1.9, 4), (0.5, 1e30, 4)])
def test_rof_sequence_in_float(oracle, tol_ring, tol_freq_over_a, n_hf):
    """Eqs 8-13 on the known window of a constant slow reaction (see test_oracle_step_logic), binary32 mode."""
    mech, T, kf, kr = _slow_reversible()
    t_f, dmax = 1.0e-4, 1.0e-2
    Y0 = np.array([0.9, 0.1, 0.0])
    a = (kf * Y0[0] - kr * Y0[1]) * t_f * dmax
    expected, margin = _expected_rof(a, 40, tol_ring, tol_freq_over_a * a, n_hf)
    assert margin > 5e-3
    for p in (P_ATM, 5.0 * P_ATM):
        tr = oracle.integrate_trace(mech, None, _params(alpha=0.0, energy_mode=1, tol_ring=min(tol_ring, 3e38),
                                                        tol_freq=min(tol_freq_over_a * a, 3e38), dft_first_high_bin=n_hf),
                                    T, p, Y0, t_f, **F32)
        np.testing.assert_array_equal(tr["rOF_trace"][:40, 0], expected)


@pytest.mark.parametrize("kf", [1e7, 1e9, 1e11])
def test_P11_stiff_reversible_reaction_is_damped_in_float(oracle, kf):
    kd, T, t_f = 5.0e2, 1200.0, 1e-4
    lo, hi = flat_thermo(3, 3.5, a6=[0.0, -1500.0, -4000.0], a7=[5.0, 5.0, 5.0])
    mech = build_mechanism([28.0] * 3, lo, hi, [([(0, 1)], [(1, 1)], kf, 0.0, 0.0, 1), ([(0, 1)], [(2, 1)], kd, 0.0, 0.0, 0)])
    _, Kc = rate_constants_numpy(mech, T)
    r = oracle.integrate(mech, None, _params(energy_mode=1, max_steps=50000), [T], [P_ATM], np.array([[0.5], [0.5], [0.0]]), t_f, **F32)
    assert r["status"][0] == 0 and r["steps"][0] <= 300
    K = Kc[0]
    ab = math.exp(-kd / (1 + K) * t_f)
    ref = np.array([ab / (1 + K), ab * K / (1 + K), 1 - ab])
    assert np.abs(r["Y"][:, 0] - ref).max() < 1e-3


@pytest.mark.parametrize("config,n", [(0, 512), (1, 64), (3, 16)])
def test_conservation_and_agreement_with_the_binary64_oracle(oracle, config, n):
    """Element mass is conserved to float rounding, and on the benign config 0 the binary32 result agrees with the binary64
    one at the paper's own accuracy scale (per-cell differences up to 0.006 %)."""
    w = make_workload(config, n)
    r32 = oracle.integrate(w.mech, w.estimator, w.params, w.T, w.p, w.Y, w.dt_cfd, **F32)
    r64 = oracle.integrate(w.mech, w.estimator, w.params, w.T, w.p, w.Y, w.dt_cfd)
    assert (r32["status"] == 0).all()
    assert np.abs(r32["Y"].sum(axis=0) - 1.0).max() < 2e-4
    zW = w.mech.elem_comp / w.mech.mol_weight[:, None]
    e0 = zW.T @ w.Y
    assert (np.abs(zW.T @ r32["Y"] - e0) / np.maximum(e0, 1e-30)).max() < 5e-4
    assert r32["Y"].min() > -1e-6
    if config == 0:
        assert np.abs(r32["Y"] - r64["Y"]).max() < 2e-3 and (np.abs(r32["T"] - r64["T"]) / r64["T"]).max() < 1e-3
        assert np.median(np.abs(r32["Y"] - r64["Y"]).max(axis=0)) < 1e-4
        assert (r32["steps"] == r64["steps"]).mean() > 0.5
    else:   # chaotic burst dynamics: same solution within the method's own scatter
        assert np.median(np.abs(r32["Y"] - r64["Y"]).max(axis=0)) < 2e-2


def test_bfer_shaped_case_in_float(oracle):
    m = bfer_shaped_mechanism()
    T, p, Y = bfer_shaped_field(48)
    r32 = oracle.integrate(m, None, _params(), T, p, Y, 1e-3, **F32)
    r64 = oracle.integrate(m, None, _params(), T, p, Y, 1e-3)
    assert (r32["status"] == 0).all()
    assert np.abs(r32["Y"] - r64["Y"]).max() < 2e-2 and (np.abs(r32["T"] - r64["T"]) / r64["T"]).max() < 2e-2
    assert np.median(np.abs(r32["Y"] - r64["Y"]).max(axis=0)) < 1e-3
