"""GPU parity of the coverage paths for grids the fast paths cannot address:
- a non-integer number of Yee cells per control pixel (epsgrad_config_t nx_cells / ny_cells; filter_general.cuh), up to the
  geometry of the paper's own demonstration (Fig. 4): 36 x 36 control variables on a design region of 210 x 210
  cells, embedded at (110, 120, 0) in the 430 x 450 x 64 model, two wavelengths;
- z columns that are not a multiple of 4 cells (scalar3d.cuh).
Each against the float64 oracle (which takes real cells-per-pixel ratios: tests/test_oracle_stages.py pins that by brute
force) at BASELINE.json's tolerances."""
import numpy as np
import pytest
import torch

import oracle as O
from gpu_common import TOL_EPS, TOL_GRAD, check_guard_bands, dev, max_rel, oracle_cfg, rand_C, rand_fields
from helpers import cfg_of, rel_inf, rel_l2
from paper_2505_03352_b200 import binding as B
from paper_2505_03352_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _check(cfg, beta, n_pairs, seed, plan=None):
    C = rand_C(cfg, seed)
    EF, EA = rand_fields(cfg, n_pairs, seed + 1)
    plan = plan or B.Plan(cfg)
    dEF, dEA = [dev(f) for f in EF], [dev(f) for f in EA]
    eps, g = plan.eps_forward_vjp(dev(C), beta, dEF, dEA)
    g2, db = plan.eps_vjp_beta(dev(C), beta, dEF, dEA)
    u = plan.unbinarity(dev(C), beta)
    assert torch.equal(g, g2) and torch.equal(plan.eps_forward(dev(C), beta), eps) and torch.equal(plan.eps_vjp(dev(C), beta, dEF, dEA), g)
    eps, g, db, u = (t.cpu().numpy().astype(np.float64) for t in (eps, g, db, u))
    oc = oracle_cfg(cfg)
    worst = [0.0, 0.0]
    for b in range(cfg.batch):
        f, a = [x[b] for x in EF], [x[b] for x in EA]
        ref = O.forward(oc, C[b], beta)
        gref, dbref = O.vjp_beta(oc, C[b], beta, f, a)
        worst[0] = max(worst[0], max_rel(eps[b], ref))
        worst[1] = max(worst[1], rel_inf(g[b], gref), rel_l2(g[b], gref))
        assert abs(db[b] - dbref) < TOL_GRAD * max(abs(dbref), 1e-3 * np.abs(gref).sum())
        uref = O.unbinarity(oc, C[b], beta)
        assert abs(u[b] - uref) < 1e-5 * max(uref, 1e-3)
    assert worst[0] < TOL_EPS and worst[1] < TOL_GRAD, worst
    return worst


@pytest.mark.parametrize("kw,beta,n_pairs", [
    (dict(mx=7, my=5, nx_cells=41, ny_cells=23, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=6.0), 8.0, 1),          # 5.86 / 4.6 cells per pixel
    (dict(mx=9, my=11, nx_cells=20, ny_cells=31, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0, subpixel=4), 12.0, 2),
    (dict(batch=2, mx=13, my=6, nx_cells=33, ny_cells=47, nz=12, z_lo=0.0, z_hi=7.5, filter_kind=1, filter_radius=9.0, filter_sigma=3.0), 5.0, 1),
    (dict(mx=12, my=12, nx_cells=37, ny_cells=37, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=5.0, morph_diameter=2.5), 10.0, 1),
    (dict(mx=6, my=8, nx_cells=19, ny_cells=18, nz=8, z_lo=1.5, z_hi=6.0, filter_radius=5.0, filter_normalize=0, eta=0.0), 0.7, 3),
    (dict(mx=10, my=10, nx_cells=10, ny_cells=13, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=2.0), 8.0, 1),         # one cell per pixel along x
])
def test_noninteger_cells_per_control_pixel(kw, beta, n_pairs):
    cfg = B.make_config(**kw)
    assert cfg.nx == kw["nx_cells"] and cfg.ny == kw["ny_cells"]
    _check(cfg, beta, n_pairs, 300)
    EF, EA = rand_fields(cfg, n_pairs, 302)
    check_guard_bands(cfg, dev(rand_C(cfg, 301)), [dev(f) for f in EF], [dev(f) for f in EA], beta)


def test_explicit_cell_counts_equal_to_the_integer_ratio_take_the_fast_path_bits():
    kw = dict(mx=21, my=17, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0)
    a, b = B.Plan(B.make_config(**kw)), B.Plan(B.make_config(**kw, nx_cells=42, ny_cells=34))
    cfg = a.cfg
    C = dev(rand_C(cfg, 5))
    EF, EA = rand_fields(cfg, 1, 6)
    ra, rb = a.eps_forward_vjp(C, 8.0, [dev(EF[0])], [dev(EA[0])]), b.eps_forward_vjp(C, 8.0, [dev(EF[0])], [dev(EA[0])])
    assert torch.equal(ra[0], rb[0]) and torch.equal(ra[1], rb[1])


def test_fig4_geometry_embedded_in_the_model_domain():
    """Fig. 4: model 430 x 450 x 64 cells, design region 210 x 210 cells, 36 x 36 control variables, two wavelengths.
    The region sits at (110, 120, 0); eps is written and the fields are read only inside it."""
    w = W.BY_NAME["fig4"]
    cfg = B.config_of(w)
    assert (cfg.nx, cfg.ny, cfg.mx, cfg.my, cfg.nz) == (210, 210, 36, 36, 64) and w.n_pairs == 2
    C = W.make_C(w)
    EF = [W.make_field(w, p, 0) for p in range(w.n_pairs)]
    EA = [W.make_field(w, p, 1) for p in range(w.n_pairs)]
    plan = B.Plan(cfg)
    NXF, NYF, NZF, I0, J0 = 430, 450, 64, 110, 120
    plan.set_embedding(NXF, NYF, NZF, I0, J0, 0)
    shape = (1, 3, NXF, NYF, NZF)
    blk = (slice(None), slice(None), slice(I0, I0 + 210), slice(J0, J0 + 210), slice(0, 64))
    gen = torch.Generator(device="cuda").manual_seed(11)
    full = lambda f: torch.view_as_complex(torch.randn(*shape, 2, device="cuda", generator=gen))
    dEF, dEA = [full(f) for f in EF], [full(f) for f in EA]
    for d, h in zip(dEF + dEA, EF + EA):
        d[blk] = dev(h)[None]
    eps = torch.full(shape, -3.0, device="cuda")
    beta = w.betas[0]
    _, g = plan.eps_forward_vjp(dev(C), beta, dEF, dEA, eps_out=eps)
    torch.cuda.synchronize()
    oc = cfg_of(w)
    ref = O.forward(oc, C[0], beta)
    gref = O.vjp(oc, C[0], beta, EF, EA)
    err_e = max_rel(eps[blk][0].cpu().numpy().astype(np.float64), ref)
    gg = g.cpu().numpy().astype(np.float64)[0]
    err_g = max(rel_inf(gg, gref), rel_l2(gg, gref))
    print(f"fig4 geometry: eps {err_e:.2e}, dF/dC {err_g:.2e}")
    assert err_e < TOL_EPS and err_g < TOL_GRAD
    outside = torch.ones(shape, dtype=torch.bool, device="cuda")
    outside[blk] = False
    assert bool((eps[outside] == -3.0).all())


@pytest.mark.parametrize("kw,beta,n_pairs", [
    (dict(mx=19, my=11, nz=6, z_lo=1.25, z_hi=4.75, filter_radius=4.0), 8.0, 1),
    (dict(mx=8, my=23, nz=9, z_lo=2.5, z_hi=8.25, filter_radius=3.0), 16.0, 2),                 # odd: field columns start on 8-byte boundaries
    (dict(batch=2, mx=12, my=9, nz=13, z_lo=0.0, z_hi=13.0, filter_kind=1, filter_radius=6.0, filter_sigma=2.0, upsample=1, subpixel=4), 6.0, 1),
    (dict(mx=9, my=9, nz=1, z_lo=0.25, z_hi=0.75, filter_radius=2.0), 8.0, 1),                  # a single layer of cells
    (dict(mx=7, my=5, nx_cells=41, ny_cells=23, nz=10, z_lo=2.25, z_hi=5.75, filter_radius=6.0), 8.0, 9),   # both coverage paths; 9 pairs: two launches
])
def test_z_columns_that_are_not_a_multiple_of_four_cells(kw, beta, n_pairs):
    cfg = B.make_config(**kw)
    _check(cfg, beta, n_pairs, 400)
    plan = B.Plan(cfg)
    plan.set_dense_reads(True)                                    # every cell of the column, zero weight outside the slab
    _check(cfg, beta, n_pairs, 400, plan)
    EF, EA = rand_fields(cfg, n_pairs, 402)
    check_guard_bands(cfg, dev(rand_C(cfg, 401)), [dev(f) for f in EF], [dev(f) for f in EA], beta)
    # the host entry point stages such fields whole
    C = rand_C(cfg, 400)
    EF, EA = rand_fields(cfg, n_pairs, 401)
    plan = B.Plan(cfg)
    eps0, g0 = plan.eps_forward_vjp(dev(C), beta, [dev(f) for f in EF], [dev(f) for f in EA])
    pin = lambda a: torch.from_numpy(a).pin_memory()
    eps_h, g_h = torch.empty(plan.eps_shape).pin_memory(), torch.empty(plan.ctrl_shape).pin_memory()
    plan.eps_forward_vjp_host(pin(C), beta, [pin(f) for f in EF], [pin(f) for f in EA], eps_h, g_h)
    torch.cuda.synchronize()
    assert torch.equal(eps_h, eps0.cpu()) and torch.equal(g_h, g0.cpu())


def test_what_the_coverage_paths_refuse():
    gen = B.Plan(B.make_config(mx=7, my=5, nx_cells=41, ny_cells=23, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=6.0))
    with pytest.raises(B.EpsgradError) as e:
        gen.set_slab(0, 10)                                        # x-slabs are cut along control rows
    assert e.value.status == B.EUNSUPPORTED
    with pytest.raises(B.EpsgradError) as e:
        gen.set_fused(1)                                           # the persistent kernel is the fast path's
    assert e.value.status == B.EUNSUPPORTED
    odd = B.Plan(B.make_config(mx=8, my=8, nz=6, z_lo=1.25, z_hi=4.75))
    with pytest.raises(B.EpsgradError) as e:
        odd.set_embedding(40, 40, 8, 4, 4, 0)                      # 16-byte pieces of the domain's arrays
    assert e.value.status == B.EUNSUPPORTED
    with pytest.raises(B.EpsgradError) as e:                       # a cone that leaves mask pixels between the control nodes uncovered
        B.Plan(B.make_config(mx=4, my=4, nx_cells=40, ny_cells=40, nz=8, z_lo=2.0, z_hi=5.0, filter_radius=3.0))
    assert e.value.status == B.EINVAL
