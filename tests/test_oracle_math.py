"""Pins for the oracle's contract exp/log, NASA-7 thermo, DFT and MLP forward pass (P5, P7, P12)."""
import math

import numpy as np
import pytest

from stev_inputs.configs import make_mechanism, make_workload
from stev_inputs.estimators import fit_estimator, IN_T, IN_T_P_Y, ACT_SIGMOID
from tests.helpers import nasa_numpy


def _ulps(a, b):
    return abs(a - b) / (abs(b) * 2.0**-52)


def test_exp_matches_libm_within_2_ulp(oracle):
    rng = np.random.default_rng(0)
    xs = np.concatenate([rng.uniform(-708, 709, 20000), rng.uniform(-1, 1, 5000), [0.0, -708.0, 709.0, 1e-300, -1e-17]])
    worst = max(_ulps(oracle.exp(x), math.exp(x)) for x in xs)
    assert worst <= 2.0
    assert oracle.exp(0.0) == 1.0
    assert oracle.exp(709.5) == math.inf and oracle.exp(-708.5) == 0.0   # stated saturation, DESIGN.md 5.3
    assert math.isnan(oracle.exp(math.nan))


def test_log_matches_libm_within_2_ulp(oracle):
    rng = np.random.default_rng(1)
    xs = np.concatenate([10.0 ** rng.uniform(-300, 300, 20000), rng.uniform(0.5, 2.0, 20000), [1.0, 2.0, 0.5, math.sqrt(2)]])
    worst = 0.0
    for x in xs:
        ref = math.log(x)
        if ref == 0.0:
            assert oracle.log(x) == 0.0
        else:
            worst = max(worst, _ulps(oracle.log(x), ref))
    assert worst <= 2.0
    assert oracle.log(0.0) == -math.inf and math.isnan(oracle.log(-1.0))


def test_exp_log_roundtrip_and_functional_equations(oracle):
    for x in [0.3, 7.0, 123.456, 2000.0]:
        assert abs(oracle.exp(oracle.log(x)) - x) <= 4e-16 * x * max(1.0, abs(math.log(x)))
    assert abs(oracle.exp(1.0) - math.e) <= 4.5e-16
    assert abs(oracle.log(10.0) - 2.302585092994046) <= 4.5e-16


@pytest.mark.parametrize("config", [0, 1, 3])
def test_nasa7_against_plain_power_form_and_cp_is_dh_dT(oracle, config):
    """Eqs 15-16 in Horner form vs plain powers; cp = d(h)/dT by central differences (P12)."""
    mech = make_mechanism(config)
    for T in [350.0, 999.0, 1000.0, 1001.0, 1777.0, 2900.0]:
        cp, h, s = oracle.thermo(mech, T)
        cp_n, h_n, s_n = nasa_numpy(mech, T)
        np.testing.assert_allclose(cp, cp_n, rtol=1e-14)
        np.testing.assert_allclose(h, h_n, rtol=1e-13, atol=1e-13)
        np.testing.assert_allclose(s, s_n, rtol=1e-14)
    for T in [500.0, 1500.0, 2500.0]:
        d = 0.01
        _, hp, sp = oracle.thermo(mech, T + d)
        _, hm, sm = oracle.thermo(mech, T - d)
        cp, _, _ = oracle.thermo(mech, T)
        dh_dT = (hp * (T + d) - hm * (T - d)) / (2 * d)       # d(h/R)/dT = cp/R
        np.testing.assert_allclose(dh_dT, cp, rtol=1e-6)
        ds_dT = (sp - sm) / (2 * d)                           # d(s/R)/dT = cp/(R T)
        np.testing.assert_allclose(ds_dT, cp / T, rtol=1e-6)


def test_thermo_continuous_at_split(oracle):
    mech = make_mechanism(1)
    lo = oracle.thermo(mech, 1000.0 - 1e-9)
    hi = oracle.thermo(mech, 1000.0)
    for a, b in zip(lo, hi):
        np.testing.assert_allclose(a, b, rtol=1e-9)


# ---------------------------------------------------------------- P7: DFT closed forms (Eq 9)
def test_dft_against_numpy_fft(oracle):
    rng = np.random.default_rng(3)
    for _ in range(50):
        ring = rng.standard_normal(13) * 10.0 ** rng.uniform(-12, 2)
        D = oracle.dft_mag(ring)
        ref = np.abs(np.fft.fft(ring))[:7]
        np.testing.assert_allclose(D, ref, rtol=0, atol=1e-13 * np.abs(ring).sum())


def test_dft_closed_forms(oracle):
    k = np.arange(13)
    a = 0.37
    D = oracle.dft_mag(a * (-1.0) ** k)                       # pure alternation
    assert abs(D[0] - a) < 1e-13
    assert abs(D[6] - a / math.sin(math.pi / 26)) < 1e-12     # = 8.29623 a
    assert abs(D[0] / D[4:].max() - math.sin(math.pi / 26)) < 1e-13   # f_ring = 0.120537
    D = oracle.dft_mag(np.full(13, 2.5))                      # constant: all high bins vanish
    assert abs(D[0] - 32.5) < 1e-13 and D[1:].max() < 1e-13
    D = oracle.dft_mag(k.astype(float))                       # ramp: D^j = 13 / (2 sin(pi j / 13))
    for j in range(1, 7):
        assert abs(D[j] - 13.0 / (2 * math.sin(math.pi * j / 13))) < 1e-12
    assert abs(D[0] / D[4:].max() - 78.0 / (13.0 / (2 * math.sin(math.pi * 4 / 13)))) < 1e-12   # 9.8758
    e = np.zeros(13); e[5] = 3.0                              # single sample: flat spectrum
    np.testing.assert_allclose(oracle.dft_mag(e), 3.0, rtol=1e-14)


def test_dft_shift_invariance_and_mirror(oracle):
    rng = np.random.default_rng(4)
    ring = rng.standard_normal(13)
    D = oracle.dft_mag(ring)
    for sft in [1, 5, 12]:
        np.testing.assert_allclose(oracle.dft_mag(np.roll(ring, sft)), D, atol=1e-13)
    full = np.abs(np.fft.fft(ring))
    np.testing.assert_allclose(full[7:], full[1:7][::-1], atol=1e-13)   # bins 7..12 mirror 6..1 (R10)


# ---------------------------------------------------------------- P12: MLP forward vs numpy float64 matmul
@pytest.mark.parametrize("config,input_map,hidden", [(3, IN_T, 32), (4, IN_T_P_Y, 64)])
def test_mlp_forward_against_numpy(oracle, config, input_map, hidden):
    mech = make_mechanism(config)
    est = fit_estimator(mech, hidden, seed=7, input_map=input_map)
    rng = np.random.default_rng(8)
    n = 257
    X = np.zeros((n, est.n_in), np.float32)
    X[:, 0] = rng.uniform(300, 3000, n)
    if input_map == IN_T_P_Y:
        X[:, 1] = rng.uniform(1, 5, n) * 1.01325e6
        X[:, 2:] = rng.dirichlet(np.full(mech.n_species, 0.5), n)
    out = oracle.estimator_eval(est, X)
    x = (X.astype(np.float64) - est.in_shift.astype(np.float64)) * est.in_scale.astype(np.float64)
    ref = np.tanh(x @ est.W1.astype(np.float64).T + est.b1) @ est.W2.astype(np.float64).T + est.b2
    scale = np.maximum(np.abs(ref), np.sqrt(np.mean(ref**2, axis=0, keepdims=True)))   # R24 norm
    assert np.max(np.abs(out - ref) / scale) < 1e-5
    # the fitted network reproduces the NASA-7 tables it was fitted to (max 0.436 %)
    cp_ref = np.array([nasa_numpy(mech, float(t))[0] for t in X[:, 0]])
    assert np.max(np.abs(out[:, :mech.n_species] - cp_ref) / cp_ref) < 1e-2


def test_mlp_sigmoid_option(oracle):
    mech = make_mechanism(1)
    est = fit_estimator(mech, 16, seed=9, activation=ACT_SIGMOID)
    X = np.linspace(300, 3000, 64, dtype=np.float32)[:, None]
    out = oracle.estimator_eval(est, X)
    x = (X.astype(np.float64) - est.in_shift) * est.in_scale
    ref = (1 / (1 + np.exp(-(x @ est.W1.astype(np.float64).T + est.b1)))) @ est.W2.astype(np.float64).T + est.b2
    assert np.max(np.abs(out - ref) / np.maximum(np.abs(ref), 1.0)) < 1e-5
