"""GPU parity of the binary32 state path (stev_params.state_precision = STEV_STATE_FP32) against the
oracle's binary32 mode: both implement the float arithmetic contract of DESIGN.md section 5b, so the comparison is bit
for bit (the asserted bar is BASELINE.json's tolerances, the observed agreement is printed)."""
import numpy as np
import pytest

from stev_inputs.configs import default_params, make_workload
from tests.gpu_util import GpuCase, assert_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def stev():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    import paper_1905_09395_b200 as stev
    stev.load()
    return stev


@pytest.mark.parametrize("config,lanes", [(0, 0), (1, 0), (1, 4), (2, 0), (2, 32), (3, 0), (4, 0)])
def test_rates_bit_exact_in_float(stev, oracle, config, lanes):
    import torch
    w = make_workload(config, 300)
    case = GpuCase(stev, w)
    rng = np.random.default_rng(config)
    rof = 2.0 ** -rng.integers(0, 6, (w.mech.n_reactions, w.n_cells)).astype(np.float64)
    prm = stev.stev_params_default(**dict(w.params, lanes_per_cell=lanes, state_precision=stev.STEV_STATE_FP32))
    dev = torch.device("cuda:0")
    t = lambda a: torch.tensor(a, dtype=torch.float64, device=dev)
    dY, dT, q = stev.stev_rates_eval(case.mech, case.est, prm, t(w.T), t(w.p), t(w.Y), t(rof))
    rdY, rdT, rq = oracle.rates_eval(w.mech, w.estimator, w.params, w.T, w.p, w.Y, rof, precision="f32")
    np.testing.assert_array_equal(q.cpu().numpy(), rq)
    np.testing.assert_array_equal(dY.cpu().numpy(), rdY)
    np.testing.assert_array_equal(dT.cpu().numpy(), rdT)


@pytest.mark.parametrize("config,n,over", [(0, 2000, {}), (1, 600, {}), (2, 300, {}), (3, 96, {}), (4, 200, {}),
                                           (0, 2000, dict(lanes_per_cell=4)), (1, 600, dict(lanes_per_cell=16)),
                                           (2, 300, dict(lanes_per_cell=8)), (3, 96, dict(lanes_per_cell=32)),
                                           (4, 200, dict(lanes_per_cell=32)), (3, 700, dict(lanes_per_cell=513)),
                                           (3, 1, {}), (3, 19, {}), (4, 1000, dict(lanes_per_cell=513)), (2, 1500, dict(lanes_per_cell=512)),
                                           (3, 64, dict(use_estimator=False)), (1, 200, dict(lanes_per_cell=1)),
                                           (1, 200, dict(lanes_per_cell=32)), (2, 200, dict(chunk_steps=300)),
                                           (1, 100, dict(max_steps=150)), (2, 100, dict(alpha=0.0, dft_first_high_bin=1)),
                                           (2, 100, dict(energy_mode=1, delta_max=0.002, y_step_max=0.05)),
                                           (1, 100, dict(dft_enable=0, max_steps=3000))])
def test_integrate_parity_in_float(stev, oracle, config, n, over):
    over = dict(over)
    w = make_workload(config, n)
    est = w.estimator if over.pop("use_estimator", True) else None
    sched = {k: over.pop(k) for k in ("lanes_per_cell", "chunk_steps") if k in over}
    prm = dict(w.params, **over)
    ref = oracle.integrate(w.mech, est, prm, w.T, w.p, w.Y, w.dt_cfd, precision="f32")
    case = GpuCase(stev, w)
    if est is None:
        case.est = None
    gpu = case.integrate(state_precision=stev.STEV_STATE_FP32, **over, **sched)
    if "lanes_per_cell" in sched:
        assert gpu["stats"]["lanes_per_cell"] == sched["lanes_per_cell"]
    elif "chunk_steps" in sched:
        assert gpu["stats"]["lanes_per_cell"] <= 32           # chunked passes: the shared-memory-history kernel
    else:
        assert gpu["stats"]["lanes_per_cell"] == 512          # default: the lock-step kernel, binary32 instantiation
    rep = assert_parity(gpu, ref)
    print(f"binary32 config {config}: n={n} {rep} lanes={gpu['stats']['lanes_per_cell']} steps {ref['steps'].min()}..{ref['steps'].max()}")
    assert gpu["rc"] == ref["rc"]
    assert rep["bit_exact"] == 1.0


def test_bfer_shaped_mechanism_in_float(stev, oracle):
    import torch
    from stev_inputs.mechanisms import bfer_shaped_field, bfer_shaped_mechanism
    mech = bfer_shaped_mechanism()
    T, p, Y = bfer_shaped_field(1500)
    prm = default_params()
    ref = oracle.integrate(mech, None, prm, T, p, Y, 1e-3, precision="f32")
    dev = torch.device("cuda:0")
    m = stev.Mechanism(mech)
    Td, pd, Yd = (torch.tensor(a, dtype=torch.float64, device=dev) for a in (T, p, Y))
    steps = torch.zeros(1500, dtype=torch.int32, device=dev)
    status = torch.zeros(1500, dtype=torch.uint8, device=dev)
    rc = stev.stev_integrate(m, None, stev.stev_params_default(state_precision=stev.STEV_STATE_FP32, **prm), Td, pd, Yd, 1e-3, steps, status)
    torch.cuda.synchronize()
    gpu = dict(T=Td.cpu().numpy(), Y=Yd.cpu().numpy(), steps=steps.cpu().numpy(), status=status.cpu().numpy())
    rep = assert_parity(gpu, ref)
    assert rc == ref["rc"] and rep["bit_exact"] == 1.0, rep


def test_unknown_kernel_id_is_refused(stev):
    w = make_workload(3, 32)
    for prec in (stev.STEV_STATE_FP32, stev.STEV_STATE_FP64):
        with pytest.raises(stev.StevError) as err:
            GpuCase(stev, w).integrate(state_precision=prec, lanes_per_cell=64)
        assert err.value.code == stev.STEV_EINVAL
