"""eps_unbinarity_static: the entry point that allocates nothing (scratch in a file-scope device array of the library).

Collected last on purpose (`pytest --collect-only`): the suite runs with `pytest -x`, and a failure here must not hide the
parity tests.  Passes alone in a fresh process and after the other tests: it depends on no state but the library's own array,
whose contents from earlier calls do not matter (every call writes the slots it reads).
"""
import numpy as np
import pytest
import torch

import oracle as O
from gpu_common import dev, oracle_cfg, rand_C
from paper_2505_03352_b200 import binding as B

pytestmark = pytest.mark.gpu

TOL_U = 1e-5            # the tolerance tests/test_gpu_beta.py uses for u(beta), relative to max(u, 1e-3)


def test_static_unbinarity_matches_the_plan_path_on_two_calls_in_a_row():
    """Two calls in a row with different masks, sizes and beta, so that the second one finds the first one's partial sums in the
    shared array (more of them than it needs): each must equal eps_unbinarity of the same plan -- same sums in the same order,
    so bit for bit, and in any case within the tolerance of the u(beta) tests -- and the float64 oracle within that tolerance.
    The outputs are preallocated: between the two calls nothing is allocated."""
    big = B.make_config(batch=3, mx=150, my=97, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=8.0)       # 3 x 15 partial sums
    small = B.make_config(batch=2, mx=19, my=33, nz=8, z_lo=2.25, z_hi=5.75, filter_kind=1, filter_radius=6.0, filter_sigma=2.0)
    cases = []
    for cfg, beta, seed in ((big, 6.0, 51), (small, 20.0, 52)):
        plan = B.Plan(cfg)
        C = rand_C(cfg, seed)
        u_plan = plan.unbinarity(dev(C), beta).clone()
        phi = plan.stage_filter(dev(C)).clone()
        out = torch.full((cfg.batch,), float("nan"), dtype=torch.float32, device="cuda")
        cases.append((plan, cfg, C, beta, phi, u_plan, out))
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for plan, cfg, C, beta, phi, u_plan, out in cases:                 # the two calls, back to back on one stream
        plan.unbinarity_static(phi, beta, out=out)
    assert torch.cuda.memory_allocated() == before
    torch.cuda.synchronize()
    for plan, cfg, C, beta, phi, u_plan, out in cases:
        assert torch.equal(out, u_plan), (out, u_plan)
        oc = oracle_cfg(cfg)
        for b in range(cfg.batch):
            u_ref = O.unbinarity(oc, C[b], beta)
            assert abs(float(out[b]) - float(u_plan[b])) <= TOL_U * max(float(u_plan[b]), 1e-3)
            assert abs(float(out[b]) - u_ref) < TOL_U * max(u_ref, 1e-3), (float(out[b]), u_ref)
    # again in the other order: the small call first leaves the big one's slots stale
    for plan, cfg, C, beta, phi, u_plan, out in reversed(cases):
        out.fill_(float("nan"))
        plan.unbinarity_static(phi, beta, out=out)
    torch.cuda.synchronize()
    for plan, cfg, C, beta, phi, u_plan, out in cases:
        assert torch.equal(out, u_plan)


def test_static_unbinarity_refuses_what_does_not_fit():
    limit = B.lib().epsgrad_static_scratch_partials()
    assert limit == 4096
    # 17 designs of 1024 x 1024 mask pixels: 17 x 256 partial sums > 4096
    cfg = B.make_config(batch=17, mx=256, my=256, nz=4, z_lo=0.5, z_hi=3.5, filter_radius=4.0)
    plan = B.Plan(cfg)
    phi = torch.zeros(plan.mask_shape, dtype=torch.float32, device="cuda")
    with pytest.raises(B.EpsgradError) as e:
        plan.unbinarity_static(phi, 8.0)
    assert e.value.status == B.EUNSUPPORTED and "4096" in str(e.value)
    # 16 designs fit exactly
    cfg = B.make_config(batch=16, mx=256, my=256, nz=4, z_lo=0.5, z_hi=3.5, filter_radius=4.0)
    plan = B.Plan(cfg)
    C = rand_C(cfg, 53)
    u = plan.unbinarity_static(plan.stage_filter(dev(C)), 8.0)
    assert torch.equal(u, plan.unbinarity(dev(C), 8.0))
    # the morphological filters change the input of the last projection: refused, not silently wrong
    plan = B.Plan(B.make_config(mx=16, my=16, nz=8, z_lo=2.0, z_hi=5.0, filter_radius=4.0, morph_diameter=3.0))
    with pytest.raises(B.EpsgradError) as e:
        plan.unbinarity_static(torch.zeros(plan.mask_shape, dtype=torch.float32, device="cuda"), 8.0)
    assert e.value.status == B.EUNSUPPORTED
    with pytest.raises(B.EpsgradError) as e:                         # beta must be positive and finite
        B.Plan(B.make_config(mx=16, my=16, nz=8, z_lo=2.0, z_hi=5.0)).unbinarity_static(
            torch.zeros((1, 64, 64), dtype=torch.float32, device="cuda"), 0.0)
    assert e.value.status == B.EINVAL
