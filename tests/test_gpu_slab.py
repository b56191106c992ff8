"""x-slab sharding of one design (third way) on the GPU path: every "rank" (run here one after
the other on the one GPU -- the ranks exchange nothing until the final sum) builds a plan for its own control rows plus the
halo, holds eps and fields for the rows it owns only (epsgrad_plan_set_slab), and the pieces are compared with the
undivided plan: eps bit for bit (same taps, same interior normalisers, same order, whichever tile of whichever plan a cell
falls in), dF/dC after the sum over ranks."""
import numpy as np
import pytest
import torch

from gpu_common import dev, rand_C, rand_fields
from helpers import rel_inf
from paper_2505_03352_b200 import binding as B, sharding

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kw,world", [
    (dict(mx=61, my=23, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0), 2),
    (dict(mx=61, my=23, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0), 5),
    (dict(batch=2, mx=40, my=31, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=3.0, morph_diameter=2.0), 3),
    (dict(mx=90, my=17, nz=32, z_lo=14.25, z_hi=17.75, filter_kind=1, filter_radius=8.0, filter_sigma=2.5), 4),
    (dict(mx=36, my=20, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0, upsample=1, subpixel=4), 3),
    (dict(mx=250, my=250, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0), 4),
])
def test_slabs_reproduce_the_undivided_plan(kw, world):
    cfg = B.make_config(**kw)
    u, n_pairs, beta = cfg.upsample, 2, 9.0
    Cn = rand_C(cfg, 91)
    EFn, EAn = rand_fields(cfg, n_pairs, 92)
    C, EF, EA = dev(Cn), [dev(f) for f in EFn], [dev(f) for f in EAn]
    full = B.Plan(cfg)
    eps_full, g_full = full.eps_forward_vjp(C, beta, EF, EA)
    gb_full, db_full = full.eps_vjp_beta(C, beta, EF, EA)
    halo = sharding.slab_halo_cells(cfg.filter_radius, cfg.morph_diameter)
    g_sum, db_sum = torch.zeros_like(g_full), torch.zeros_like(db_full)
    for rank in range(world):
        p = sharding.slab_partition(cfg.mx, u, rank, world, halo)
        plan = B.Plan(B.make_config(**dict(kw, mx=p["e1"] - p["e0"])))
        plan.set_slab(p["x_first"], p["x_count"])
        own = slice(u * p["a0"], u * p["a1"])
        assert plan.field_shape == (cfg.batch, 3, p["x_count"], cfg.ny, cfg.nz)
        C_r = C[:, p["e0"]:p["e1"]].clone()                 # (a view into C need not be 16-byte aligned)
        EF_r, EA_r = [f[:, :, own].clone() for f in EF], [f[:, :, own].clone() for f in EA]
        eps_r, g_r = plan.eps_forward_vjp(C_r, beta, EF_r, EA_r)
        assert torch.equal(eps_r, eps_full[:, :, own]), (rank, p)
        assert torch.equal(plan.eps_forward(C_r, beta), eps_r) and torch.equal(plan.eps_vjp(C_r, beta, EF_r, EA_r), g_r)
        g_b, db_r = plan.eps_vjp_beta(C_r, beta, EF_r, EA_r)
        assert torch.equal(g_b, g_r)
        # window-only eps on the slab's own rows: one full call on another design first, then the window call
        buf = plan.eps_forward((1.0 - C_r).contiguous(), beta).clone()
        plan.set_eps_window_only(True)
        plan.eps_forward(C_r, beta, buf)
        plan.set_eps_window_only(False)
        assert torch.equal(buf, eps_r), (rank, p)
        g_sum[:, p["e0"]:p["e1"]] += g_r                 # what sharding.sum_gradients does across ranks
        db_sum += db_r
        # rows of the halo beyond the dependency cone get nothing at all
        far = -(-(2 * halo + 2) // u)
        if p["a0"] - p["e0"] > far:
            assert not g_r[:, : p["a0"] - p["e0"] - far].any()
    err = rel_inf(g_sum.cpu().numpy().astype(np.float64), g_full.cpu().numpy().astype(np.float64))
    assert err < 2e-6, err                                # same terms, summed in another order
    assert torch.allclose(db_sum, db_full, rtol=1e-4, atol=1e-4 * float(g_full.abs().sum()) * 1e-3)


def test_slab_argument_checks():
    plan = B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0))
    with pytest.raises(B.EpsgradError) as e:
        plan.set_slab(10, 8)
    assert e.value.status == B.EINVAL
    plan.set_slab(4, 8)
    with pytest.raises(B.EpsgradError) as e:
        plan.set_embedding(40, 40, 8, 0, 0, 0)
    assert e.value.status == B.EUNSUPPORTED
    plan.set_slab()
    plan.set_embedding(40, 40, 8, 0, 0, 0)
    with pytest.raises(B.EpsgradError) as e:
        plan.set_slab(4, 8)
    assert e.value.status == B.EUNSUPPORTED
