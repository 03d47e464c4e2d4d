"""jipm_solve_batch_static (include/jipm.h): the solve for callers that must not allocate, its scratch in a static
device array of JIPM_STATIC_SCRATCH_BYTES.  Collected last on purpose (the suite runs with pytest -x).  The new entry
point is compared with the existing path (jipm_create + jipm_solve_batch) on two calls in a row: same problems, same
arguments -> the two paths run the same kernel on the same data and must agree bit for bit (the tolerance the
batch-independence tests of test_gpu_parity.py use: exact)."""
import numpy as np
import pytest

from paper_2606_26341_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _outputs(torch, P, n, m, fill):
    """Caller-owned outputs, pre-filled with garbage so that a call that writes nothing cannot pass."""
    return dict(x=torch.full((P, n), fill, dtype=torch.float64, device="cuda"),
                lam=torch.full((P, m), fill, dtype=torch.float64, device="cuda"),
                zL=torch.full((P, n), fill, dtype=torch.float64, device="cuda"),
                zU=torch.full((P, n), fill, dtype=torch.float64, device="cuda"),
                status=torch.full((P,), -7, dtype=torch.int32, device="cuda"),
                iters=torch.full((P,), -7, dtype=torch.int32, device="cuda"))


@pytest.mark.parametrize("cfg,P,kw", [(0, 48, {}), (1, 6, dict(horizon_N=7))])
def test_static_entry_matches_existing_path_on_two_calls_in_a_row(cfg, P, kw):
    import torch
    from paper_2606_26341_b200 import jipm
    d = wl.config_dims(cfg, **kw)
    d, theta, x0 = wl.generate(cfg, 2 * P, d)
    xL, xU = wl.bounds(d)
    x0_d, th_d = torch.as_tensor(x0, device="cuda"), torch.as_tensor(theta, device="cuda")
    s = jipm.Solver(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt, xL, xU)
    # two different batches, so that the second call finds the first one's leftovers in the static array
    for call, sl in enumerate((slice(0, P), slice(P, 2 * P))):
        xa, ta = x0_d[sl].contiguous(), th_d[sl].contiguous()
        ref = s.solve_batch(xa, ta)
        out = _outputs(torch, P, d.n, d.m, float("nan"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        jipm.solve_batch_static(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt, xL, xU, xa, ta, out)
        torch.cuda.synchronize()
        if call == 1:   # (the first call may load the module that holds the static array)
            assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated or freed inside the call"
        st = ref["status"].cpu().numpy()
        assert np.array_equal(out["status"].cpu().numpy(), st), call
        assert np.array_equal(out["iters"].cpu().numpy(), ref["iters"].cpu().numpy()), call
        assert (st == 0).sum() >= P // 2, st          # the comparison is of real solves, not of failures
        for key in ("x", "lam", "zL", "zU"):
            a, b = out[key].cpu().numpy(), ref[key].cpu().numpy()
            assert np.all(np.isfinite(a[st == 0])), (call, key)
            assert np.array_equal(a, b, equal_nan=True), (call, key, float(np.nanmax(np.abs(a - b))))
    s.close()


def test_static_entry_rejects_what_does_not_fit():
    """C2 of BASELINE.json needs more scratch than JIPM_STATIC_SCRATCH_BYTES: a clear error, nothing launched."""
    import torch
    from paper_2606_26341_b200 import jipm
    d = wl.config_dims(2)
    d, theta, x0 = wl.generate(2, 1, d)
    xL, xU = wl.bounds(d)
    out = _outputs(torch, 1, d.n, d.m, 0.0)
    with pytest.raises(jipm.JipmError, match="static maximum"):
        jipm.solve_batch_static(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt, xL, xU,
                                torch.as_tensor(x0, device="cuda"), torch.as_tensor(theta, device="cuda"), out)
    assert int(out["status"][0]) == -7
    assert jipm.STATIC_SCRATCH_BYTES == 64 << 20
