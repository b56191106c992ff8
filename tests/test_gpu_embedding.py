"""The design region embedded in a simulation domain (NEXT-4; "|Omega_D", Fig. 4): eps, E_F, E_A are the solver's
full arrays, the library reads and writes only the block of the design region.  Pure addressing: the results must equal,
bit for bit, those of the region-sized call on the cropped block, and everything outside the block must stay untouched."""
import numpy as np
import pytest
import torch

import oracle as O
from gpu_common import TOL_EPS, TOL_GRAD, dev, max_rel, oracle_cfg, rand_C
from helpers import rel_inf
from paper_2505_03352_b200 import binding as B

pytestmark = pytest.mark.gpu


def full_fields(cfg, shape, n, seed):
    rng = np.random.default_rng([seed, 3])
    out = []
    for _ in range(2 * n):
        a = np.empty(shape, np.complex64)
        rng.standard_normal(out=a.view(np.float32).reshape(-1), dtype=np.float32)
        out.append(a)
    return out[:n], out[n:]


@pytest.mark.parametrize("kw,full,org", [
    (dict(mx=21, my=18, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0), (61, 50, 24), (9, 7, 4)),
    (dict(batch=2, mx=33, my=40, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0), (66, 80, 16), (0, 0, 0)),        # block = domain in x, y, z
    (dict(mx=105, my=105, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0), (430, 450, 64), (110, 120, 0)),     # the model of Fig. 4
    (dict(mx=16, my=20, nz=24, z_lo=8.5, z_hi=13.0, filter_radius=3.0, morph_diameter=3.0), (40, 47, 40), (5, 6, 12)),
])
def test_embedded_calls_equal_region_calls_on_the_cropped_block(kw, full, org):
    cfg = B.make_config(**kw)
    (nxf, nyf, nzf), (i0, j0, k0) = full, org
    shape = (cfg.batch, 3, nxf, nyf, nzf)
    blk = (slice(None), slice(None), slice(i0, i0 + cfg.nx), slice(j0, j0 + cfg.ny), slice(k0, k0 + cfg.nz))
    C = rand_C(cfg, 61)
    EF, EA = full_fields(cfg, shape, 2, 62)
    plan = B.Plan(cfg)
    # region-sized reference calls on the cropped, contiguous block
    cEF, cEA = [dev(np.ascontiguousarray(f[blk])) for f in EF], [dev(np.ascontiguousarray(f[blk])) for f in EA]
    eps_r, g_r = plan.eps_forward_vjp(dev(C), 9.0, cEF, cEA)
    plan.set_embedding(nxf, nyf, nzf, i0, j0, k0)
    assert plan.field_shape == shape
    sentinel = -7.0
    eps_f = torch.full(shape, sentinel, device="cuda")
    dEF, dEA = [dev(f) for f in EF], [dev(f) for f in EA]
    _, g_e = plan.eps_forward_vjp(dev(C), 9.0, dEF, dEA, eps_out=eps_f)
    g_v = plan.eps_vjp(dev(C), 9.0, dEF, dEA)
    eps_f2 = torch.full(shape, sentinel, device="cuda")
    plan.eps_forward(dev(C), 9.0, out=eps_f2)
    torch.cuda.synchronize()
    assert torch.equal(g_e, g_r) and torch.equal(g_v, g_r)
    assert torch.equal(eps_f[blk], eps_r) and torch.equal(eps_f2, eps_f)
    outside = torch.ones(shape, dtype=torch.bool, device="cuda")
    outside[blk] = False
    assert bool((eps_f[outside] == sentinel).all())                    # the rest of the solver's eps is not touched
    # and against the oracle through the crop
    oc = oracle_cfg(cfg)
    for b in range(cfg.batch):
        ref = O.forward(oc, C[b], 9.0)
        assert max_rel(eps_f[blk][b].cpu().numpy().astype(np.float64), ref) < TOL_EPS
        gref = O.vjp(oc, C[b], 9.0, [f[blk][b] for f in EF], [f[blk][b] for f in EA])
        assert rel_inf(g_e[b].cpu().numpy().astype(np.float64), gref) < TOL_GRAD
    # window-only eps (epsgrad_plan_set_eps_window_only) inside the embedded block: after the full call above, a window call on
    # another design leaves the solver's array as a full call would, and still touches nothing outside the block
    C2 = rand_C(cfg, 63)
    eps_w = eps_f.clone()
    eps_full2 = torch.full(shape, sentinel, device="cuda")
    plan.eps_forward(dev(C2), 9.0, out=eps_full2)
    plan.set_eps_window_only(True)
    plan.eps_forward(dev(C2), 9.0, out=eps_w)
    plan.set_eps_window_only(False)
    assert torch.equal(eps_w, eps_full2)
    plan.set_embedding()                                               # back to region-sized arrays
    eps_b, g_b = plan.eps_forward_vjp(dev(C), 9.0, cEF, cEA)
    assert torch.equal(eps_b, eps_r) and torch.equal(g_b, g_r)


def test_embedding_argument_checks():
    plan = B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0))
    with pytest.raises(B.EpsgradError) as e:
        plan.set_embedding(20, 15, 8, 0, 0, 0)              # 16 cells do not fit 15
    assert e.value.status == B.EINVAL
    with pytest.raises(B.EpsgradError) as e:
        plan.set_embedding(20, 20, 16, 1, 1, 2)             # k0 % 4 != 0
    assert e.value.status == B.EUNSUPPORTED
    with pytest.raises(B.EpsgradError) as e:
        plan.set_embedding(20, 20, 18, 1, 1, 4)             # nz_full % 4 != 0
    assert e.value.status == B.EUNSUPPORTED
    plan.set_embedding(20, 20, 16, 2, 3, 4)
    pin = lambda *s: torch.zeros(*s).pin_memory()
    with pytest.raises(B.EpsgradError) as e:
        plan.eps_forward_vjp_host(pin(1, 8, 8), 8.0, [torch.zeros(plan.eps_shape, dtype=torch.complex64).pin_memory()],
                                  [torch.zeros(plan.eps_shape, dtype=torch.complex64).pin_memory()],
                                  pin(*plan.eps_shape), pin(1, 8, 8))
    assert e.value.status == B.EUNSUPPORTED
