"""GPU parity tests of the lock-step integrator (stev_ls_kernel.cuh, lanes_per_cell = 512): all cells of a block step
together, work is flattened over (cell, reaction) / (cell, species) pairs, the DFT history lives in tensor memory.
Bit-exact against the oracle on every config, with and without estimator, at block-boundary sizes and edge cases."""
import dataclasses

import numpy as np
import pytest

from stev_inputs.configs import make_workload
from tests.gpu_util import GpuCase, assert_parity

pytestmark = pytest.mark.gpu
LS = 512


@pytest.fixture(scope="module")
def stev():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    import paper_1905_09395_b200 as stev
    stev.load()
    return stev


@pytest.mark.parametrize("config,n,over", [(3, 500, {}), (3, 37, {}), (3, 1, {}), (3, 200, dict(use_estimator=False)),
                                           (1, 400, {}), (1, 5000, {}), (2, 300, {}), (2, 4737, {}), (4, 300, {}), (0, 600, {}),
                                           (0, 4096, {}), (3, 1400, {}),
                                           (1, 100, dict(max_steps=150)), (2, 100, dict(alpha=0.0, dft_first_high_bin=1)),
                                           (2, 100, dict(dft_first_high_bin=6)),
                                           (2, 100, dict(energy_mode=1, delta_max=0.002, y_step_max=0.05)),
                                           (1, 100, dict(dft_enable=0, max_steps=3000)),
                                           (4, 100, dict(use_estimator=False)), (3, 100, dict(order_cells=0))])
@pytest.mark.parametrize("kernel", [512, 513])
def test_lockstep_parity(stev, oracle, kernel, config, n, over):
    """512: the instantiation with the mechanism's dimensions as compile-time constants where the shape list has one;
    513: dimensions read at run time (what any other mechanism runs)."""
    over = dict(over)
    w = make_workload(config, n)
    est = w.estimator if over.pop("use_estimator", True) else None
    prm = dict(w.params, **{k: v for k, v in over.items() if k != "order_cells"})
    ref = oracle.integrate(w.mech, est, prm, w.T, w.p, w.Y, w.dt_cfd)
    case = GpuCase(stev, w)
    if est is None:
        case.est = None
    gpu = case.integrate(lanes_per_cell=kernel, **over)
    assert gpu["stats"]["lanes_per_cell"] == kernel
    assert gpu["stats"]["specialised"] in ((0, 1) if kernel == 512 else (0,))
    rep = assert_parity(gpu, ref)
    print(f"lock-step config {config}: n={n} {rep} stats={gpu['stats']}")
    assert gpu["rc"] == ref["rc"]
    assert rep["bit_exact"] == 1.0


@pytest.mark.parametrize("config,n_rev", [(3, 1), (3, 31), (3, 32), (3, 33), (3, 64), (3, 65), (3, 128), (3, 193), (3, 224),
                                          (2, 1), (2, 31), (2, 32), (2, 33), (1, 1), (1, 7)])
def test_lockstep_number_of_reversible_reactions(stev, oracle, config, n_rev):
    """Cells per block and the flattened passes follow from the number of reversible reactions; run it at and around
    the 32-lane boundaries (the first n_rev reversible reactions stay reversible, the others become irreversible)."""
    w = make_workload(config, 96)
    rev = np.array(w.mech.reversible).copy()
    idx = np.nonzero(rev)[0]
    assert n_rev <= idx.size
    rev[idx[n_rev:]] = 0
    mech = dataclasses.replace(w.mech, reversible=rev)
    prm = dict(w.params, max_steps=4000)
    ref = oracle.integrate(mech, None, prm, w.T, w.p, w.Y, w.dt_cfd)
    w2 = dataclasses.replace(w, mech=mech, estimator=None)
    gpu = GpuCase(stev, w2).integrate(lanes_per_cell=LS, max_steps=4000)
    assert gpu["stats"]["lanes_per_cell"] == LS
    rep = assert_parity(gpu, ref)
    assert rep["bit_exact"] == 1.0, rep


def test_lockstep_padded_leading_dimension_and_nan_cell(stev, oracle):
    w = make_workload(1, 300)
    ref = oracle.integrate(w.mech, None, w.params, w.T, w.p, w.Y, w.dt_cfd)
    gpu = GpuCase(stev, w).integrate(lanes_per_cell=LS, ld=437)
    assert assert_parity(gpu, ref)["bit_exact"] == 1.0
    T = w.T.copy()
    T[[3, 77]] = np.nan
    ref = oracle.integrate(w.mech, None, w.params, T, w.p, w.Y, w.dt_cfd)
    gpu = GpuCase(stev, w).integrate(T=T, lanes_per_cell=LS)
    assert gpu["rc"] == ref["rc"] == 2
    np.testing.assert_array_equal(gpu["status"], ref["status"])
    np.testing.assert_array_equal(gpu["steps"], ref["steps"])
    ok = ref["status"] == 0
    np.testing.assert_array_equal(gpu["Y"][:, ok], ref["Y"][:, ok])
    np.testing.assert_array_equal(gpu["T"][ok], ref["T"][ok])
