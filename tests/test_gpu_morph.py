"""GPU parity of the chain with the morphological filters on (Eqs. (4)-(5); readings S17, S18): eps and dF/dC
against the float64 oracle, element by element, through the C ABI -- small regions where every pixel feels a border,
a batch, both filter kinds, s = 4, and the paper-scale region."""
import numpy as np
import pytest
import torch

import oracle as O
from gpu_common import TOL_EPS, TOL_GRAD, check_forward, check_vjp, dev, oracle_cfg, rand_C, rand_fields
from paper_2505_03352_b200 import binding as B

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kw", [
    dict(mx=9, my=7, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0, morph_diameter=3.0),          # every pixel near a border
    dict(batch=2, mx=37, my=29, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0, morph_diameter=4.0),
    dict(mx=24, my=33, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0, morph_diameter=2.0, morph_alpha=35.0),
    dict(mx=20, my=18, nz=8, z_lo=2.25, z_hi=5.75, subpixel=4, filter_radius=3.0, morph_diameter=2.5),
    dict(mx=40, my=40, nz=8, z_lo=2.25, z_hi=5.75, filter_kind=B.FILTER_GAUSSIAN, filter_radius=6.0, filter_sigma=2.0,
         morph_diameter=8.0),                                                                      # widest supported disk at s = 2: R = 8
])
@pytest.mark.parametrize("beta", [6.0, 24.0])
def test_eps_and_gradient_match_oracle_with_filters_on(kw, beta):
    cfg = B.make_config(**kw)
    C = rand_C(cfg, 31)
    EF, EA = rand_fields(cfg, 2, 32)
    plan = B.Plan(cfg)
    check_forward(cfg, C, beta, plan)
    check_vjp(cfg, C, beta, EF, EA, plan)
    eps, g = plan.eps_forward_vjp(dev(C), beta, [dev(f) for f in EF], [dev(f) for f in EA])
    # filter (2 passes when separable), 4 morph, fwd2d, zreduce, extrude, maskgrad, 4 morph^T, filterT (2 passes when separable)
    assert plan.last_launches() == 14 + 2 * (cfg.filter_kind == B.FILTER_GAUSSIAN)
    assert torch.equal(eps, plan.eps_forward(dev(C), beta)) and torch.equal(g, plan.eps_vjp(dev(C), beta, [dev(f) for f in EF], [dev(f) for f in EA]))


def test_uniform_control_stays_uniform_through_the_filters():
    cfg = B.make_config(mx=33, my=20, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0, morph_diameter=4.0)
    plan = B.Plan(cfg)
    beta = 7.0
    for c0 in (0.1, 0.43, 0.8):
        e2 = plan.stage_eps2d(torch.full(plan.ctrl_shape, c0, device="cuda"), beta).cpu().numpy().astype(np.float64)
        rho0 = 0.5 * (1 + np.tanh(beta * (np.float64(np.float32(c0)) - 0.5)))
        rho = 0.5 * (1 + np.tanh(beta * (rho0 - 0.5)))
        ref = rho * cfg.eps_core + (1 - rho) * cfg.eps_clad
        assert np.max(np.abs(e2 - ref)) < 1e-5 * ref


def test_paper_scale_region_with_filters_on():
    cfg = B.make_config(mx=250, my=250, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0, morph_diameter=4.0)
    C = rand_C(cfg, 33)
    EF, EA = rand_fields(cfg, 1, 34)
    plan = B.Plan(cfg)
    err_e = check_forward(cfg, C, 16.0, plan)
    err_g = check_vjp(cfg, C, 16.0, EF, EA, plan)
    print(f"paper scale, d = 4 cells, alpha = 20: eps {err_e:.2e}  dF/dC {err_g:.2e}")


def test_disk_limits_are_reported():
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(mx=64, my=64, nz=8, z_lo=2.0, z_hi=5.0, morph_diameter=17.0))       # R = 17 mask pixels
    assert e.value.status == B.EUNSUPPORTED
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(mx=2, my=8, nz=8, z_lo=2.0, z_hi=5.0, morph_diameter=6.0))          # disk wider than the mask
    assert e.value.status == B.EUNSUPPORTED
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, morph_diameter=2.0, morph_alpha=0.0))
    assert e.value.status == B.EINVAL
