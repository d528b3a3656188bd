"""msm_restrict_noalloc (include/msm.h): the restriction with its scratch in a file-scope device
array, for callers that cannot call cudaMalloc. Checked against the existing path: a plan's own
restriction between levels 1 and 2 (grid charges read back with msm_debug_copy_grid), within the
grid-charge tolerance of the parity tests, on two calls in a row (the second call finds the first
call's contents in the shared scratch and must not depend on them).

Collected last on purpose (the run uses pytest -x).
"""
import numpy as np
import pytest

from parity_util import FP32_BOUNDS, FP64_RTOL, small_workload

pytestmark = pytest.mark.gpu


def _plan_grids(w, precision):
    """Q^1 and Q^2 of one evaluation through the existing path, and the level geometry."""
    import torch
    from paper_2510_05961_b200 import msm
    plan = msm.Plan.for_workload(w, precision)
    dt = plan.torch_dtype
    dev = torch.device("cuda", 0)
    pos = torch.tensor(w.positions, dtype=dt, device=dev).contiguous()
    q = torch.tensor(w.charges, dtype=dt, device=dev).contiguous()
    plan.evaluate(pos, q, torch.zeros((w.n, 3), dtype=dt, device=dev), torch.zeros(w.n, dtype=dt, device=dev),
                  True, False)
    assert plan.info.n_tiled >= 2
    Q1, Q2 = plan.debug_grid(1, "Q"), plan.debug_grid(2, "Q")
    lo1 = [int(v) for v in plan.info.grid_lo[0]]
    lo2 = [int(v) for v in plan.info.grid_lo[1]]
    plan.close()
    return Q1, Q2, lo1, lo2


@pytest.mark.parametrize("kind,n,p,precision", [("periodic", 1531, 4, "fp64"), ("open", 700, 6, "fp64"),
                                                ("slab", 1203, 4, "fp32")])
def test_restrict_noalloc_matches_the_plan_path_twice(kind, n, p, precision):
    import torch
    from paper_2510_05961_b200 import msm
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    w = small_workload(kind, n, seed=100 + n, p=p, precision=precision)
    Q1, Q2, lo1, lo2 = _plan_grids(w, precision)
    # (fp32 plans hold fp32 grids: Q1 is exactly representable, the input is the plan's own)
    dt = torch.float32 if precision == "fp32" else torch.float64
    dev = torch.device("cuda", 0)
    fine = torch.tensor(Q1, dtype=dt, device=dev).contiguous()
    qmax = float(np.abs(w.charges).max())
    scale = max(float(np.abs(Q2).max()), qmax)
    tol = FP32_BOUNDS["Q"] if precision == "fp32" else FP64_RTOL
    # the second call restricts a different input first, so that the shared scratch holds foreign
    # contents when the checked call runs
    other = torch.tensor(np.random.default_rng(5).standard_normal(Q1.shape), dtype=dt, device=dev).contiguous()
    for call in range(2):
        coarse = torch.full(Q2.shape, float("nan"), dtype=dt, device=dev)
        if call == 1:
            msm.restrict_noalloc(other, coarse, p, lo1, lo2, w.periodic)
        msm.restrict_noalloc(fine, coarse, p, lo1, lo2, w.periodic)
        torch.cuda.synchronize()
        got = coarse.cpu().numpy().astype(np.float64)
        assert np.isfinite(got).all(), f"call {call}: output not written in full"
        err = float(np.abs(got - Q2).max()) / scale
        assert err <= tol, f"{w.name} call {call}: restriction differs from the plan path by {err:.3e} > {tol:g}"


def test_restrict_noalloc_rejects_what_does_not_fit():
    """A periodic 256^3 fp64 fine grid needs 96 MiB of scratch: refused, nothing launched."""
    import torch
    from paper_2510_05961_b200 import msm
    dev = torch.device("cuda", 0)
    fine = torch.zeros((256, 256, 256), dtype=torch.float64, device=dev)
    coarse = torch.full((128, 128, 128), 7.0, dtype=torch.float64, device=dev)
    with pytest.raises(msm.MsmError) as e:
        msm.restrict_noalloc(fine, coarse, 4, (0, 0, 0), (0, 0, 0), (1, 1, 1))
    assert e.value.status == 8 and "SCRATCH_LIMIT" in str(e.value)
    torch.cuda.synchronize()
    assert float(coarse.min()) == 7.0 and float(coarse.max()) == 7.0
    # the largest periodic power-of-two case that fits: 128^3 fp64 (12 MiB of the 16 MiB)
    fine = torch.ones((128, 128, 128), dtype=torch.float64, device=dev)
    coarse = torch.zeros((64, 64, 64), dtype=torch.float64, device=dev)
    msm.restrict_noalloc(fine, coarse, 4, (0, 0, 0), (0, 0, 0), (1, 1, 1))
    torch.cuda.synchronize()
    # sum_n J_n = 2 per axis: a constant grid restricts to 8 times the constant
    assert float((coarse - 8.0).abs().max()) <= 1e-13
