"""Helpers for the -m gpu parity tests: run a Workload through the C ABI (via the Python binding) on cuda:0."""
import numpy as np


def to_params(stev, params: dict, **over):
    d = dict(params)
    d.update(over)
    return stev.stev_params_default(**d)


class GpuCase:
    def __init__(self, stev, workload):
        self.stev = stev
        self.w = workload
        self.mech = stev.Mechanism(workload.mech)
        self.est = stev.Estimator(self.mech, workload.estimator) if workload.estimator is not None else None

    def integrate(self, T=None, p=None, Y=None, ld=None, **over):
        import torch
        stev, w = self.stev, self.w
        T = w.T if T is None else T
        p = w.p if p is None else p
        Y = w.Y if Y is None else Y
        n = T.shape[0]
        dev = torch.device("cuda:0")
        Td = torch.tensor(T, dtype=torch.float64, device=dev)
        pd = torch.tensor(p, dtype=torch.float64, device=dev)
        S = Y.shape[0]
        ld = n if ld is None else ld
        Ybuf = torch.full((S, ld), float("nan"), dtype=torch.float64, device=dev)
        Ybuf[:, :n] = torch.tensor(Y, dtype=torch.float64, device=dev)
        Yd = Ybuf[:, :n] if ld != n else Ybuf
        steps = torch.full((n,), -1, dtype=torch.int32, device=dev)
        status = torch.full((n,), 255, dtype=torch.uint8, device=dev)
        prm = to_params(stev, w.params, **over)
        rc = stev.stev_integrate(self.mech, self.est, prm, Td, pd, Yd, w.dt_cfd, steps, status)
        torch.cuda.synchronize()
        return dict(rc=rc, T=Td.cpu().numpy(), Y=Ybuf[:, :n].cpu().numpy(), steps=steps.cpu().numpy(),
                    status=status.cpu().numpy(), stats=stev.stev_last_stats())


def assert_parity(gpu, ref, y_tol=1e-6, t_tol=1e-3, min_same_steps=0.999):
    """BASELINE.json north_star tolerances: |dY| <= 1e-6, |dT| <= 1e-3 K, identical step counts for >= 99.9 %."""
    same = gpu["steps"] == ref["steps"]
    assert same.mean() >= min_same_steps, f"only {same.mean():.5f} of cells have identical step counts"
    np.testing.assert_array_equal(gpu["status"], ref["status"])
    dy = np.abs(gpu["Y"] - ref["Y"]).max(axis=0)
    dt = np.abs(gpu["T"] - ref["T"])
    ok = (dy <= y_tol) & (dt <= t_tol)
    assert ok.mean() >= min_same_steps, f"{(~ok).sum()} cells outside tolerance (max dY {dy.max():.3e}, max dT {dt.max():.3e})"
    return dict(same_steps=float(same.mean()), bit_exact=float(((dy == 0) & (dt == 0) & same).mean()),
                max_dY=float(dy.max()), max_dT=float(dt.max()))
