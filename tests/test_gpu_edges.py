"""GPU parity at the edges of what include/stev.h admits: stoichiometric coefficients of 3 and three concentration
factors on a side (only the shared-memory-history kernel takes them; the tensor-memory kernels must refuse), mechanisms
at the species counts where the lock-step kernel's lane ownership changes (31..33, 54, 63, 64), the parameters that are validated rather than
implemented (dft_window, estimator_precision), and the non-blocking return."""
import time

import numpy as np
import pytest

from stev_inputs.configs import default_params, make_workload
from stev_inputs.mechanisms import P_ATM, synthetic_mechanism
from tests.gpu_util import assert_parity
from tests.helpers import build_mechanism, flat_thermo

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def stev():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    import paper_1905_09395_b200 as stev
    stev.load()
    return stev


def _run(stev, mech, est, params, T, p, Y, dt, **over):
    import torch
    dev = torch.device("cuda:0")
    m = stev.Mechanism(mech)
    e = stev.Estimator(m, est) if est is not None else None
    Td, pd, Yd = (torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev) for a in (T, p, Y))
    n = T.shape[0]
    steps = torch.full((n,), -1, dtype=torch.int32, device=dev)
    status = torch.full((n,), 255, dtype=torch.uint8, device=dev)
    prm = stev.stev_params_default(**dict(params, **over))
    rc = stev.stev_integrate(m, e, prm, Td, pd, Yd, dt, steps, status)
    torch.cuda.synchronize()
    return dict(rc=rc, T=Td.cpu().numpy(), Y=Yd.cpu().numpy(), steps=steps.cpu().numpy(), status=status.cpu().numpy(),
                stats=stev.stev_last_stats())


def _field(S, n, seed, t_lo=1000.0, t_hi=2200.0):
    rng = np.random.default_rng(seed)
    return rng.uniform(t_lo, t_hi, n), np.full(n, P_ATM), np.ascontiguousarray(rng.dirichlet(np.ones(S), n).T)


def _multi_factor_mechanism():
    """A (1 atom), B (3), C (1), D (2), E (4):  3 A <=> B (nu = 3),  2 A + D <=> E (three factors on a side),
    A + C -> D (plain), B + C <=> 2 D (nu = 2 on the product side)."""
    atoms = np.array([1.0, 3.0, 1.0, 2.0, 4.0])
    lo, hi = flat_thermo(5, 3.5, a6=[0.0, -9000.0, -500.0, -6000.0, -14000.0], a7=[4.0, 5.0, 4.5, 6.0, 7.0])
    rx = [([(0, 3)], [(1, 1)], 1.0e16, 0.0, 8000.0, 1),
          ([(0, 2), (3, 1)], [(4, 1)], 3.0e15, 0.5, 3000.0, 1),
          ([(0, 1), (2, 1)], [(3, 1)], 1.0e12, 0.0, 10000.0, 0),
          ([(1, 1), (2, 1)], [(3, 2)], 5.0e11, 0.0, 6000.0, 1)]
    return build_mechanism(10.0 * atoms, lo, hi, rx, elem_comp=atoms[:, None])


@pytest.mark.parametrize("lanes", [0, 1, 4, 32])
def test_nu_three_and_three_factors_on_the_shared_memory_kernel(stev, oracle, lanes):
    mech = _multi_factor_mechanism()
    T, p, Y = _field(5, 700, 11, 900.0, 1800.0)
    prm = default_params()
    ref = oracle.integrate(mech, None, prm, T, p, Y, 1e-4)
    assert (ref["steps"] > 100).any()                       # the limiter is active: not a trivial run
    gpu = _run(stev, mech, None, prm, T, p, Y, 1e-4, lanes_per_cell=lanes)
    assert gpu["stats"]["lanes_per_cell"] <= 32             # the default falls back to the shared-memory-history kernel
    rep = assert_parity(gpu, ref)
    assert gpu["rc"] == ref["rc"] and rep["bit_exact"] == 1.0, rep


@pytest.mark.parametrize("kernel", [512, 513])
def test_tensor_memory_kernels_refuse_more_than_two_factors(stev, kernel):
    mech = _multi_factor_mechanism()
    T, p, Y = _field(5, 64, 12)
    with pytest.raises(stev.StevError) as err:
        _run(stev, mech, None, default_params(), T, p, Y, 1e-4, lanes_per_cell=kernel)
    assert err.value.code == stev.STEV_EINVAL and "two" in str(err.value)


@pytest.mark.parametrize("S,R,E,kernels,scale", [(32, 90, 3, (512, 513), 1.0e-3), (31, 60, 3, (512, 8), 1.0e-2),
                                                 (33, 100, 3, (512, 513), 1.0e-3), (54, 180, 4, (512,), 1.0e-5),
                                                 (63, 200, 4, (513,), 1.0e-5), (64, 220, 4, (512, 513, 16), 1.0e-5)])
def test_species_limits_of_the_tensor_memory_kernels(stev, oracle, S, R, E, kernels, scale):
    mech = synthetic_mechanism(S, R, E, seed=7000 + S, stiffness_scale=scale)
    T, p, Y = _field(S, 160, S)
    prm = dict(default_params(), max_steps=4000)
    ref = oracle.integrate(mech, None, prm, T, p, Y, 1e-4)
    for kernel in kernels:
        gpu = _run(stev, mech, None, prm, T, p, Y, 1e-4, lanes_per_cell=kernel)
        assert gpu["stats"]["lanes_per_cell"] == kernel
        rep = assert_parity(gpu, ref)
        assert gpu["rc"] == ref["rc"] and rep["bit_exact"] == 1.0, (kernel, rep)


def test_validated_parameters(stev):
    w = make_workload(3, 32)
    for over, word in [(dict(dft_window=12), "thirteen"), (dict(estimator_precision=stev.STEV_PREC_TF32), "fp32"),
                       (dict(estimator_precision=stev.STEV_PREC_BF16), "fp32"), (dict(state_precision=7), "state_precision")]:
        with pytest.raises(stev.StevError) as err:
            _run(stev, w.mech, w.estimator, w.params, w.T, w.p, w.Y, w.dt_cfd, **over)
        assert err.value.code == stev.STEV_EINVAL and word in str(err.value)


@pytest.mark.parametrize("config,lanes", [(3, 0), (1, 0), (2, 0), (1, 8)])
def test_nonblocking_return_overlaps_host_work(stev, oracle, config, lanes):
    """stev_params.nonblocking = 1 (the CFD code calls the solver and may do its own work meanwhile):
    stev_integrate returns while the kernel is still running; stev_integrate_finish delivers the return code; the
    results are those of the blocking call."""
    import torch
    w = make_workload(config, 4096 if config != 3 else 2048)
    dev = torch.device("cuda:0")
    m = stev.Mechanism(w.mech)
    e = stev.Estimator(m, w.estimator) if w.estimator is not None else None

    def run(nonblocking):
        Td, pd, Yd = (torch.tensor(a, dtype=torch.float64, device=dev) for a in (w.T, w.p, w.Y))
        steps = torch.zeros(w.n_cells, dtype=torch.int32, device=dev)
        status = torch.zeros(w.n_cells, dtype=torch.uint8, device=dev)
        prm = stev.stev_params_default(**dict(w.params, nonblocking=nonblocking, lanes_per_cell=lanes))
        ws = torch.empty(max(stev.stev_workspace_bytes(m, e, prm, w.n_cells), 256), dtype=torch.uint8, device=dev)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        rc = stev.stev_integrate(m, e, prm, Td, pd, Yd, w.dt_cfd, steps, status, workspace=ws)
        t_call = time.perf_counter() - t0
        host_work = 0
        if nonblocking:
            ev = torch.cuda.Event()
            ev.record()
            while not ev.query():          # the host is free while the kernel runs
                host_work += 1
            rc = stev.stev_integrate_finish(ws)
        torch.cuda.synchronize()
        t_all = time.perf_counter() - t0
        return rc, t_call, t_all, host_work, Td.cpu().numpy(), Yd.cpu().numpy(), steps.cpu().numpy(), status.cpu().numpy()

    run(0)                                  # warm-up (module load, table upload)
    rc_b, tc_b, ta_b, _, T_b, Y_b, s_b, st_b = run(0)
    rc_n, tc_n, ta_n, spins, T_n, Y_n, s_n, st_n = run(1)
    assert rc_b == rc_n
    np.testing.assert_array_equal(T_b, T_n)
    np.testing.assert_array_equal(Y_b, Y_n)
    np.testing.assert_array_equal(s_b, s_n)
    np.testing.assert_array_equal(st_b, st_n)
    print(f"config {config}: blocking call {tc_b * 1e3:.2f} ms; nonblocking call returned after {tc_n * 1e3:.2f} ms of "
          f"{ta_n * 1e3:.2f} ms, host spun {spins} times meanwhile")
    assert tc_n < 0.5 * ta_n and spins > 10     # the call came back well before the kernel finished


# ------------------------------------------------------------------------------------------ real coefficients / orders
@pytest.mark.parametrize("lanes,n", [(0, 3000), (1, 500), (2, 500), (8, 777), (32, 500)])
def test_bfer_shaped_mechanism_parity(stev, oracle, lanes, n):
    """Eqs 26-30 with Table 1's constants and synthetic thermodynamics: real stoichiometric coefficients (1.5, 0.5) and
    rate-law exponents (0.5, 0.65), t_f = 1 ms.  Runs on the shared-memory-history kernel, bit for bit."""
    from stev_inputs.mechanisms import bfer_shaped_field, bfer_shaped_mechanism
    mech = bfer_shaped_mechanism()
    T, p, Y = bfer_shaped_field(n)
    prm = default_params()
    ref = oracle.integrate(mech, None, prm, T, p, Y, 1e-3)
    gpu = _run(stev, mech, None, prm, T, p, Y, 1e-3, lanes_per_cell=lanes)
    assert gpu["stats"]["lanes_per_cell"] <= 32
    rep = assert_parity(gpu, ref)
    print(f"BFER-shaped, {n} cells, lanes {gpu['stats']['lanes_per_cell']}: {rep}, steps {ref['steps'].min()}..{ref['steps'].max()}")
    assert gpu["rc"] == ref["rc"] and rep["bit_exact"] == 1.0, rep


def test_real_coefficients_are_refused_by_the_tensor_memory_kernels_and_integers_as_reals_agree(stev, oracle):
    import dataclasses
    from stev_inputs.mechanisms import bfer_shaped_field, bfer_shaped_mechanism
    mech = bfer_shaped_mechanism()
    T, p, Y = bfer_shaped_field(64)
    for kernel in (512, 513):
        with pytest.raises(stev.StevError) as err:
            _run(stev, mech, None, default_params(), T, p, Y, 1e-3, lanes_per_cell=kernel)
        assert err.value.code == stev.STEV_EINVAL
    w = make_workload(1, 200)
    m = w.mech
    as_real = dataclasses.replace(m, reac_coef=m.reac_nu.astype(float), prod_coef=m.prod_nu.astype(float),
                                  reac_order=m.reac_nu.astype(float), prod_order=m.prod_nu.astype(float))
    a = _run(stev, m, None, w.params, w.T, w.p, w.Y, w.dt_cfd, lanes_per_cell=16)
    b = _run(stev, as_real, None, w.params, w.T, w.p, w.Y, w.dt_cfd)
    assert b["stats"]["lanes_per_cell"] <= 32
    for k in ("T", "Y", "steps", "status"):
        np.testing.assert_array_equal(a[k], b[k])


# ------------------------------------------------------------------------------------------ hand-rolled synchronisation
@pytest.mark.parametrize("config,kernel,n", [(3, 512, 600), (3, 513, 300), (2, 512, 2000), (1, 512, 3000), (4, 512, 1000), (0, 513, 4000)])
def test_repeated_runs_under_different_schedules_are_identical(stev, config, kernel, n):
    """compute-sanitizer is closed on this GPU pool, so the named-barrier hand-off between the scalar
    warp and the other warps, the block barriers and shared-memory atomics of the lock-step kernel and the tensor-memory allocation are checked the
    way that is left: a race shows as run-to-run differences, so the same cells are integrated twelve times -- in three
    launch orders, with the block count halved and quartered by integrating sub-ranges -- and every result must be
    bit-identical to the first."""
    import torch
    w = make_workload(config, n)
    dev = torch.device("cuda:0")
    m = stev.Mechanism(w.mech)
    e = stev.Estimator(m, w.estimator) if w.estimator is not None else None

    def run(lo, hi, order):
        Td, pd, Yd = (torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
                      for a in (w.T[lo:hi], w.p[lo:hi], w.Y[:, lo:hi]))
        steps = torch.zeros(hi - lo, dtype=torch.int32, device=dev)
        prm = stev.stev_params_default(**dict(w.params, lanes_per_cell=kernel, order_cells=order, max_steps=6000))
        stev.stev_integrate(m, e, prm, Td, pd, Yd, w.dt_cfd, steps, None)
        torch.cuda.synchronize()
        return Td.cpu().numpy(), Yd.cpu().numpy(), steps.cpu().numpy()

    T0, Y0, s0 = run(0, n, 1)
    for rep in range(3):
        for order in (0, 1, 2):
            T1, Y1, s1 = run(0, n, order)
            assert np.array_equal(T0, T1) and np.array_equal(Y0, Y1) and np.array_equal(s0, s1)
    for parts in (2, 4):
        edges = np.linspace(0, n, parts + 1).astype(int)
        for a, b in zip(edges[:-1], edges[1:]):
            T1, Y1, s1 = run(a, b, 1)
            assert np.array_equal(T0[a:b], T1) and np.array_equal(Y0[:, a:b], Y1) and np.array_equal(s0[a:b], s1)
