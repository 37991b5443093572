"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json's: final Y within 1e-6 absolute, T within 1e-3 K, identical per-cell
step counts for >= 99.9 % of cells.  Because both sides implement the arithmetic contract the
observed agreement is bit-for-bit; the tests print it."""
import numpy as np
import pytest

from stev_inputs.configs import make_workload, make_mechanism, default_params
from stev_inputs.mechanisms import P_ATM
from tests.gpu_util import GpuCase, assert_parity, to_params

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def stev():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    import paper_1905_09395_b200 as stev
    stev.load()
    return stev


def _dev(a, dtype=None):
    import torch
    return torch.tensor(a, dtype=dtype, device="cuda:0")


# ------------------------------------------------------------------------------------------------ building blocks
def test_contract_exp_log_bit_exact(stev, oracle):
    import torch
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.uniform(-720, 720, 5000), rng.uniform(-2, 2, 2000), [0.0, 709.0, 709.1, -708.0, -708.1]])
    e, _ = stev.stev_contract_exp_log(_dev(x, torch.float64))
    ref = np.array([oracle.exp(v) for v in x])
    np.testing.assert_array_equal(e.cpu().numpy(), ref)
    xl = np.concatenate([10.0 ** rng.uniform(-300, 300, 5000), rng.uniform(0.5, 2, 2000), [1.0, 2.0 ** 0.5]])
    _, l = stev.stev_contract_exp_log(_dev(xl, torch.float64))
    ref = np.array([oracle.log(v) for v in xl])
    np.testing.assert_array_equal(l.cpu().numpy(), ref)


def test_dft_magnitudes_bit_exact(stev, oracle):
    import torch
    rng = np.random.default_rng(1)
    ring = rng.standard_normal((777, 13)) * 10.0 ** rng.uniform(-200, 3, (777, 1))
    ring[5] = 0.0
    ring[6] = 1.0
    ring[7] = (-1.0) ** np.arange(13)
    D = stev.stev_dft_mag(_dev(ring, torch.float64)).cpu().numpy()
    ref = np.array([oracle.dft_mag(r) for r in ring])
    np.testing.assert_array_equal(D, ref)


@pytest.mark.parametrize("n", [0, 1, 31, 1024, 1025, 70001])
def test_compaction_against_numpy(stev, n):
    import torch
    rng = np.random.default_rng(n)
    flags = (rng.random(n) < 0.37).astype(np.uint8)
    lst = rng.permutation(n).astype(np.int32)
    out, c = stev.stev_compact_active(_dev(flags), _dev(lst))
    np.testing.assert_array_equal(out.cpu().numpy(), lst[flags != 0])
    assert c == int(flags.sum())
    out, c = stev.stev_compact_active(_dev(flags), None)
    np.testing.assert_array_equal(out.cpu().numpy(), np.nonzero(flags)[0].astype(np.int32))
    if n:
        out, c = stev.stev_compact_active(_dev(np.ones(n, np.uint8)), None)
        assert c == n
        out, c = stev.stev_compact_active(_dev(np.zeros(n, np.uint8)), None)
        assert c == 0


@pytest.mark.parametrize("config,lanes", [(0, 0), (0, 4), (1, 0), (1, 1), (1, 32), (2, 0), (2, 8), (3, 0), (3, 16), (4, 0)])
def test_rates_bit_exact(stev, oracle, config, lanes):
    """Rows a1, a2 (and a7's fp32 path for configs 3, 4): dY/dt, dT/dt and every q_j equal the oracle's bit for bit."""
    import torch
    w = make_workload(config, 300)
    case = GpuCase(stev, w)
    rng = np.random.default_rng(config)
    rof = 2.0 ** -rng.integers(0, 6, (w.mech.n_reactions, w.n_cells)).astype(np.float64)
    prm = to_params(stev, w.params, lanes_per_cell=lanes)
    for use_rof in (False, True):
        dY, dT, q = stev.stev_rates_eval(case.mech, case.est, prm, _dev(w.T), _dev(w.p), _dev(w.Y),
                                         _dev(rof) if use_rof else None)
        rY, rT, rq = oracle.rates_eval(w.mech, w.estimator, w.params, w.T, w.p, w.Y, rof if use_rof else None)
        np.testing.assert_array_equal(q.cpu().numpy(), rq)
        np.testing.assert_array_equal(dY.cpu().numpy(), rY)
        np.testing.assert_array_equal(dT.cpu().numpy(), rT)


@pytest.mark.parametrize("config", [3, 4])
def test_estimator_fp32_matches_cpu_forward_pass(stev, oracle, config):
    """North star: 'The MLP path must match a CPU forward pass of the same weights to 1e-5 relative in fp32'."""
    import torch
    w = make_workload(config, 1000)
    est = stev.Estimator(None, w.estimator)
    X = np.zeros((w.n_cells, w.estimator.n_in), np.float32)
    X[:, 0] = w.T
    if w.estimator.n_in > 1:
        X[:, 1] = w.p
        X[:, 2:] = w.Y.T
    out = stev.stev_estimator_eval(est, _dev(X), stev.STEV_PREC_FP32).cpu().numpy()
    ref = oracle.estimator_eval(w.estimator, X)
    scale = np.maximum(np.abs(ref), np.sqrt(np.mean(ref.astype(np.float64) ** 2, axis=0, keepdims=True)))
    assert np.max(np.abs(out - ref) / scale) <= 1e-5
    np.testing.assert_array_equal(out, ref)   # and in fact bit for bit (R18)


def _estimator_inputs(w):
    X = np.zeros((w.n_cells, w.estimator.n_in), np.float32)
    X[:, 0] = w.T
    if w.estimator.n_in > 1:
        X[:, 1] = w.p
        X[:, 2:] = w.Y.T
    return X


@pytest.mark.parametrize("config,n", [(3, 1000), (4, 1000), (4, 1), (4, 128), (3, 129), (4, 70001)])
@pytest.mark.parametrize("precision", ["TF32", "BF16"])
def test_estimator_tensor_core_path(stev, oracle, config, n, precision):
    """Row a7, tcgen05 path (stev_mlp_tc.cu).  North star: 'the MLP path must match a CPU forward pass of the same
    weights to ... 1e-2 relative where TF32/BF16 tensor cores are used'; relative error in the R24 norm
    (|a - b| / max(|b|, RMS of that output over the batch))."""
    w = make_workload(config, n)
    est = stev.Estimator(None, w.estimator)
    X = _estimator_inputs(w)
    prec = getattr(stev, "STEV_PREC_" + precision)
    out = stev.stev_estimator_eval(est, _dev(X), prec).cpu().numpy()
    ref = oracle.estimator_eval(w.estimator, X)
    assert out.shape == ref.shape and np.isfinite(out).all()
    scale = np.maximum(np.abs(ref), np.sqrt(np.mean(ref.astype(np.float64) ** 2, axis=0, keepdims=True)))
    err = float(np.max(np.abs(out - ref) / scale))
    print(f"config {config} n={n} {precision}: max rel err (R24) {err:.3e}")
    assert err <= 1e-2
    # the tensor path really rounds its operands: it is not the fp32 path in disguise
    if n >= 1000:
        assert err > 1e-7


def test_estimator_tensor_core_path_sigmoid_and_odd_widths(stev, oracle):
    """Sigmoid activation (the paper's choice) and widths that are not multiples of the MMA shapes."""
    import copy
    rng = np.random.default_rng(5)
    w = make_workload(4, 777)
    e = copy.deepcopy(w.estimator)
    e.activation = 1
    e.n_hidden, e.n_out = 24, 13          # 24 -> padded to 32 columns, 13 outputs -> scalar row stores
    e.W1 = rng.uniform(-1, 1, (e.n_hidden, e.n_in)).astype(np.float32)
    e.b1 = rng.uniform(-1, 1, e.n_hidden).astype(np.float32)
    e.W2 = rng.uniform(-1, 1, (e.n_out, e.n_hidden)).astype(np.float32)
    e.b2 = rng.uniform(-1, 1, e.n_out).astype(np.float32)
    est = stev.Estimator(None, e)
    X = _estimator_inputs(w)
    ref = oracle.estimator_eval(e, X)
    scale = np.maximum(np.abs(ref), np.sqrt(np.mean(ref.astype(np.float64) ** 2, axis=0, keepdims=True)))
    for prec in (stev.STEV_PREC_FP32, stev.STEV_PREC_TF32, stev.STEV_PREC_BF16):
        out = stev.stev_estimator_eval(est, _dev(X), prec).cpu().numpy()
        err = float(np.max(np.abs(out - ref) / scale))
        assert err <= (1e-5 if prec == stev.STEV_PREC_FP32 else 1e-2), (prec, err)


# ------------------------------------------------------------------------------------------------ the integrator
@pytest.mark.parametrize("config,n", [(0, 4096), (1, 1500), (2, 700), (3, 300), (4, 300)])
def test_integrate_parity(stev, oracle, config, n):
    w = make_workload(config, n)
    ref = oracle.integrate(w.mech, w.estimator, w.params, w.T, w.p, w.Y, w.dt_cfd)
    gpu = GpuCase(stev, w).integrate()
    rep = assert_parity(gpu, ref)
    print(f"config {config}: n={n} {rep} stats={gpu['stats']}")
    assert gpu["rc"] == ref["rc"]
    # conservation on the GPU result itself (P3)
    assert np.max(np.abs(gpu["Y"].sum(axis=0) - 1.0)) < 1e-12


# --------------------------------------------------------------------- full size, the launch configuration bench.py times
@pytest.mark.parametrize("config", [0, 1, 2, 3, 4])
def test_full_size_sampled_parity_and_invariants(stev, oracle, config):
    """BASELINE.json's full cell counts with the default parameters and kernel selection (what `bench.py --config C` times).
    Cells are independent, so the oracle integrates a seeded sample of them one by one; the whole field is
    checked through what holds at any size: mass fractions sum to one, element mass fractions are conserved (pins P3/P4 on
    the GPU result), Y >= 0 (Eq 3 caps consumption at 0.9 y), every cell took at least one step and reports a status."""
    w = make_workload(config)
    n = w.n_cells
    gpu = GpuCase(stev, w).integrate()
    assert gpu["rc"] in (0, stev.STEV_WMAXSTEPS)
    assert np.isfinite(gpu["T"]).all() and np.isfinite(gpu["Y"]).all()
    assert (gpu["steps"] >= 1).all() and np.isin(gpu["status"], (0, 1)).all()
    assert (gpu["status"] == 0).mean() >= 0.995
    assert gpu["Y"].min() >= 0.0
    assert np.max(np.abs(gpu["Y"].sum(axis=0) - 1.0)) < 1e-12
    zW = w.mech.elem_comp / w.mech.mol_weight[:, None]            # [S, E] moles of element per unit mass of species
    drift = np.abs(zW.T @ gpu["Y"] - zW.T @ w.Y) / np.maximum(zW.T @ w.Y, 1e-300)
    assert drift.max() < 1e-11, drift.max()
    # sampled cells, one by one through the oracle: a seeded draw plus the cells that took the most steps
    rng = np.random.default_rng(20260000 + config)
    m = {0: 4096, 1: 8192, 2: 8192, 3: 8192, 4: 2048}[config]   # >= 0.78 % of config 3's cells, one by one through the oracle
    idx = np.unique(np.concatenate([rng.choice(n, size=min(m, n), replace=False), np.argsort(gpu["steps"])[-8:],
                                    [0, n - 1]]))
    ref = oracle.integrate(w.mech, w.estimator, w.params, w.T[idx], w.p[idx], np.ascontiguousarray(w.Y[:, idx]), w.dt_cfd)
    sub = dict(T=gpu["T"][idx], Y=gpu["Y"][:, idx], steps=gpu["steps"][idx], status=gpu["status"][idx])
    rep = assert_parity(sub, ref)
    print(f"config {config} full size n={n}: sampled {idx.size} cells {rep} kernel lanes={gpu['stats']['lanes_per_cell']} "
          f"mean steps {gpu['steps'].mean():.0f} finished {(gpu['status'] == 0).mean():.5f}")
    assert rep["bit_exact"] == 1.0


@pytest.mark.parametrize("config,n,lanes", [(0, 500, 1), (0, 500, 2), (0, 500, 32), (1, 300, 1), (1, 300, 8), (1, 300, 32),
                                            (2, 200, 4), (2, 200, 32), (3, 64, 16)])
def test_result_does_not_depend_on_lanes_per_cell(stev, oracle, config, n, lanes):
    w = make_workload(config, n)
    ref = oracle.integrate(w.mech, w.estimator, w.params, w.T, w.p, w.Y, w.dt_cfd)
    gpu = GpuCase(stev, w).integrate(lanes_per_cell=lanes)
    assert gpu["stats"]["lanes_per_cell"] == lanes
    rep = assert_parity(gpu, ref)
    assert rep["bit_exact"] == 1.0


def test_default_kernel_selection(stev):
    """lanes_per_cell = 0: the lock-step kernel (test_gpu_lockstep.py) with compile-time dimensions for the five configs,
    the shared-memory-history kernel for what the lock-step kernel does not take (chunked passes here; three factors per
    side and real coefficients in test_gpu_edges.py)."""
    cells = {0: 32, 1: 32, 2: 32, 3: 8, 4: 32}
    for config in range(5):
        gpu = GpuCase(stev, make_workload(config, 64)).integrate()
        st = gpu["stats"]
        assert st["lanes_per_cell"] == 512 and st["specialised"] == 1 and st["threads_per_block"] == 512, (config, st)
        assert st["cells_per_block"] == cells[config], (config, st)
    gpu = GpuCase(stev, make_workload(2, 64)).integrate(chunk_steps=50)
    assert gpu["stats"]["lanes_per_cell"] <= 32
    with pytest.raises(stev.StevError):
        GpuCase(stev, make_workload(2, 64)).integrate(lanes_per_cell=64)   # the round-1 warp-pair kernel is gone


@pytest.mark.parametrize("config,n,over", [(2, 3000, {}), (1, 2000, {}), (3, 300, {}), (4, 500, {}), (2, 700, dict(chunk_steps=400)),
                                           (2, 900, dict(lanes_per_cell=513)), (0, 5000, {})])
def test_launch_order_is_pure_scheduling(stev, config, n, over):
    """stev_params.order_cells: the persistent kernels pull the hottest cells first (counting sort on the device);
    nothing of the result may depend on it."""
    w = make_workload(config, n)
    case = GpuCase(stev, w)
    a = case.integrate(order_cells=0, **over)
    for mode in (1, 2, 3, 4):       # by state size (cell by cell here), cell by cell, aligned groups of four / eight cells
        b = case.integrate(order_cells=mode, **over)
        for k in ("T", "Y", "steps", "status"):
            np.testing.assert_array_equal(a[k], b[k])
    b = case.integrate(T=w.T[:n - 3], p=w.p[:n - 3], Y=w.Y[:, :n - 3], order_cells=3, **over)   # ragged last group
    for k in ("T", "steps", "status"):
        np.testing.assert_array_equal(a[k][:n - 3], b[k])
    np.testing.assert_array_equal(a["Y"][:, :n - 3], b["Y"])
    # degenerate temperatures (all equal, out of the bucket range, NaN) still give a permutation
    T = w.T.copy()
    T[: n // 3] = 5000.0
    T[n // 3: n // 2] = 150.0
    d = case.integrate(T=T, order_cells=0, max_steps=50, **over)
    for mode in (1, 3, 4):
        c = case.integrate(T=T, order_cells=mode, max_steps=50, **over)
        assert (c["steps"] > 0).all()
        for k in ("T", "Y", "steps", "status"):
            np.testing.assert_array_equal(c[k], d[k])


@pytest.mark.parametrize("config,n,chunk", [(0, 3000, 64), (1, 600, 100), (1, 600, 1000), (2, 300, 333), (3, 100, 150)])
def test_chunked_passes_with_compaction_give_identical_results(stev, config, n, chunk):
    """Row a6: retiring / spilling / compacting is pure scheduling -- results cannot depend on chunk_steps."""
    w = make_workload(config, n)
    case = GpuCase(stev, w)
    a = case.integrate()
    b = case.integrate(chunk_steps=chunk)
    assert b["stats"]["passes"] == -(-int(a["steps"].max()) // chunk)
    assert b["stats"]["passes"] > 1
    for k in ("T", "Y", "steps", "status"):
        np.testing.assert_array_equal(a[k], b[k])


def test_edge_cases(stev, oracle):
    import torch
    w = make_workload(1, 100)
    case = GpuCase(stev, w)
    # empty input is a no-op
    prm = to_params(stev, w.params)
    z = torch.zeros(0, dtype=torch.float64, device="cuda:0")
    assert stev.stev_integrate(case.mech, None, prm, z, z, torch.zeros((9, 0), dtype=torch.float64, device="cuda:0"), 1e-4,
                               torch.zeros(0, dtype=torch.int32, device="cuda:0")) == 0
    # one cell; a ragged count; a leading dimension larger than n
    for n, ld in [(1, None), (37, None), (37, 64), (100, 101)]:
        ref = oracle.integrate(w.mech, None, w.params, w.T[:n], w.p[:n], w.Y[:, :n], w.dt_cfd)
        gpu = case.integrate(T=w.T[:n], p=w.p[:n], Y=w.Y[:, :n], ld=ld)
        assert assert_parity(gpu, ref)["bit_exact"] == 1.0
    # max_steps: status 1, warning return code, state at t_reached (R20)
    ref = oracle.integrate(w.mech, None, dict(w.params, max_steps=150), w.T, w.p, w.Y, w.dt_cfd)
    gpu = case.integrate(max_steps=150)
    assert gpu["rc"] == stev.STEV_WMAXSTEPS == ref["rc"] and (gpu["status"] == 1).any()
    assert assert_parity(gpu, ref)["bit_exact"] == 1.0
    # non-finite input: status 2 on that cell only
    T = w.T.copy()
    T[3] = np.nan
    gpu = case.integrate(T=T)
    assert gpu["rc"] == stev.STEV_WNONFINITE and gpu["status"][3] == 2 and (np.delete(gpu["status"], 3) == 0).all()
    # DFT off, gamma off, isothermal
    for over in [dict(dft_enable=0, max_steps=3000), dict(alpha=0.0), dict(energy_mode=1), dict(dft_first_high_bin=1),
                 dict(dft_first_high_bin=6), dict(delta_max=0.002, y_step_max=0.05)]:
        ref = oracle.integrate(w.mech, None, dict(w.params, **over), w.T[:40], w.p[:40], w.Y[:, :40], w.dt_cfd)
        gpu = case.integrate(T=w.T[:40], p=w.p[:40], Y=w.Y[:, :40], **over)
        assert assert_parity(gpu, ref)["bit_exact"] == 1.0, over
    # errors: small workspace, bad params
    Td, pd, Yd = _dev(w.T), _dev(w.p), _dev(w.Y)
    steps = torch.zeros(100, dtype=torch.int32, device="cuda:0")
    with pytest.raises(stev.StevError) as ei:
        stev.stev_integrate(case.mech, None, to_params(stev, w.params, chunk_steps=10), Td, pd, Yd, 1e-4, steps,
                            workspace=torch.empty(512, dtype=torch.uint8, device="cuda:0"))
    assert ei.value.code == stev.STEV_EWORKSPACE
    with pytest.raises(stev.StevError) as ei:
        stev.stev_integrate(case.mech, None, to_params(stev, w.params, r_fac=0.5), Td, pd, Yd, 1e-4, steps)
    assert ei.value.code == stev.STEV_EINVAL
    np.testing.assert_array_equal(Td.cpu().numpy(), w.T)   # nothing written on error


def test_mechanism_validation(stev):
    import copy
    m = copy.deepcopy(make_mechanism(1))
    m.prod_species = m.prod_species.copy()
    used = set(m.reac_species[:2]) | set(m.prod_species[:2])
    m.prod_species[0] = next(i for i in range(9) if i not in used)   # break element conservation of reaction 0
    with pytest.raises(stev.StevError):
        stev.Mechanism(m)
    stev.Mechanism(m, validate_elements=False).close()


def test_host_buffer_entry_point_matches_device_entry_point(stev):
    w = make_workload(1, 777)
    case = GpuCase(stev, w)
    a = case.integrate()
    T, Y = w.T.copy(), w.Y.copy()
    steps, status = np.zeros(w.n_cells, np.int32), np.zeros(w.n_cells, np.uint8)
    rc = stev.stev_integrate_host(case.mech, None, to_params(stev, w.params), T, w.p, Y, w.dt_cfd, steps, status)
    assert rc == a["rc"]
    np.testing.assert_array_equal(T, a["T"])
    np.testing.assert_array_equal(Y, a["Y"])
    np.testing.assert_array_equal(steps, a["steps"])
    assert stev.stev_last_stats()["total_steps"] == int(steps.sum())


def test_fp64_microbenchmarks_run(stev):
    dfma = stev.stev_microbench(0, 2048)
    cexp = stev.stev_microbench(1, 256)
    chain = stev.stev_microbench(2, 2048)   # one dependent DFMA chain in one warp per SM
    print(f"DFMA {dfma / 1e12:.2f} T/s, contract exp {cexp / 1e9:.1f} G/s, dependent DFMA chain {chain / 1e9:.1f} G/s")
    assert dfma > 1e12 and cexp > 1e10 and 1e10 < chain < dfma
