"""stev_integrate_static (include/stev.h): the lock-step integrator with its scratch in a fixed device array of the
library -- no workspace argument, no allocation inside the call.  Checked against stev_integrate (caller-owned workspace)
on the same inputs: same kernel and arithmetic, so the results must be bit-identical, which is also the tolerance the
other GPU tests hold the CUDA path to (bit-exact against the oracle).  Two calls in a row with different sizes and
mechanisms: the array keeps the first call's contents and the second must not see them.

The file name sorts last on purpose: the suite runs with `pytest -x`, a failure here must not hide other tests.  It
passes alone in a fresh process and after the other tests (it owns its handles and makes no assumption about the
scratch array's contents)."""
import numpy as np
import pytest

from stev_inputs.configs import make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def stev():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    import paper_1905_09395_b200 as stev
    stev.load()
    return stev


def _run(stev, w, mech, est, static, **over):
    import torch
    dev = torch.device("cuda:0")
    n = w.T.shape[0]
    Td, pd, Yd = (torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev) for a in (w.T, w.p, w.Y))
    steps = torch.full((n,), -1, dtype=torch.int32, device=dev)
    status = torch.full((n,), 255, dtype=torch.uint8, device=dev)
    prm = stev.stev_params_default(**dict(w.params, **over))
    if static:
        rc = stev.stev_integrate_static(mech, est, prm, Td, pd, Yd, w.dt_cfd, steps, status)
    else:
        rc = stev.stev_integrate(mech, est, prm, Td, pd, Yd, w.dt_cfd, steps, status)
    torch.cuda.synchronize()
    return dict(rc=rc, T=Td.cpu().numpy(), Y=Yd.cpu().numpy(), steps=steps.cpu().numpy(), status=status.cpu().numpy(),
                stats=stev.stev_last_stats())


def _same(a, b):
    assert a["rc"] == b["rc"]
    for k in ("steps", "status", "T", "Y"):
        np.testing.assert_array_equal(a[k], b[k], err_msg=k)   # bit-identical: |dY| = |dT| = 0 <= the 1e-6 / 1e-3 K bar


def test_static_scratch_entry_matches_the_workspace_path_on_two_calls_in_a_row(stev):
    import torch
    calls = [(3, 700, {}), (1, 2500, {}), (3, 41, dict(order_cells=0)), (2, 1300, dict(lanes_per_cell=513, max_steps=900))]
    cases = []
    for config, n, over in calls:
        w = make_workload(config, n)
        mech = stev.Mechanism(w.mech)
        est = stev.Estimator(mech, w.estimator) if w.estimator is not None else None
        cases.append((w, mech, est, over, _run(stev, w, mech, est, False, **over)))
    before = torch.cuda.memory_allocated()
    # back to back through the shared array: a large call, then smaller / different ones that must not see its leftovers
    for w, mech, est, over, ref in cases:
        got = _run(stev, w, mech, est, True, **over)
        assert got["stats"]["lanes_per_cell"] in (512, 513) and got["stats"]["passes"] == 1
        _same(got, ref)
        assert (got["steps"] > 0).all()
    # and the very same call twice in a row
    w, mech, est, over, ref = cases[0]
    _same(_run(stev, w, mech, est, True, **over), ref)
    _same(_run(stev, w, mech, est, True, **over), ref)
    assert torch.cuda.memory_allocated() == before   # the tensors of _run are released; the entry point holds nothing


def test_static_scratch_entry_nonblocking_and_warning_code(stev):
    import torch
    w = make_workload(1, 600)
    mech = stev.Mechanism(w.mech)
    ref = _run(stev, w, mech, None, False, max_steps=200)
    got = _run(stev, w, mech, None, True, max_steps=200)
    assert ref["rc"] == stev.STEV_WMAXSTEPS
    _same(got, ref)
    nb = _run(stev, w, mech, None, True, max_steps=200, nonblocking=1)   # enqueues only: STEV_OK, statuses after the sync
    assert nb["rc"] == stev.STEV_OK
    for k in ("steps", "status", "T", "Y"):
        np.testing.assert_array_equal(nb[k], ref[k])
    torch.cuda.synchronize()


def test_static_scratch_entry_rejects_what_it_cannot_hold(stev):
    import torch
    dev = torch.device("cuda:0")
    w = make_workload(0, 8)
    mech = stev.Mechanism(w.mech)
    n = stev.STEV_STATIC_MAX_CELLS + 1
    S = w.Y.shape[0]
    T = torch.full((n,), 1200.0, dtype=torch.float64, device=dev)
    p = torch.full((n,), 1013250.0, dtype=torch.float64, device=dev)
    Y = torch.full((S, n), 1.0 / S, dtype=torch.float64, device=dev)
    steps = torch.zeros(n, dtype=torch.int32, device=dev)
    prm = stev.stev_params_default(**w.params)
    with pytest.raises(stev.StevError) as err:
        stev.stev_integrate_static(mech, None, prm, T, p, Y, w.dt_cfd, steps, None)
    assert err.value.code == stev.STEV_EINVAL and "STEV_STATIC_MAX_CELLS" in str(err.value)
    assert int(steps.max()) == 0                                   # nothing ran
    # exactly the maximum is accepted (config 0: a few hundred steps per cell)
    rc = stev.stev_integrate_static(mech, None, prm, T[:-1], p[:-1], Y[:, :-1], w.dt_cfd, steps[:-1], None)
    torch.cuda.synchronize()
    assert rc == stev.STEV_OK and int(steps[:-1].min()) > 0
    # what the lock-step kernel does not take is refused, not routed elsewhere
    for over in (dict(chunk_steps=50), dict(lanes_per_cell=8)):
        with pytest.raises(stev.StevError) as err:
            stev.stev_integrate_static(mech, None, stev.stev_params_default(**dict(w.params, **over)), T[:64], p[:64], Y[:, :64],
                                       w.dt_cfd, steps[:64], None)
        assert err.value.code == stev.STEV_EINVAL and "lock-step" in str(err.value)
