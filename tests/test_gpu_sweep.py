"""GPU parity on a seeded sweep of random configurations: grid sizes around the tile edges (16x16 Yee cells per CTA of
the 2-D kernels, 256 columns per CTA of the 3-D kernels), every supported (upsample, subpixel) pair, both filters with
integer and fractional radii, slabs whose faces fall anywhere in z (on cell edges, inside one cell, on a 16-byte chunk
boundary), batches, several field pairs, the morphological filters on and off, beta from 1 to 64.  Each case checks eps,
dF/dC, dF/dbeta and u(beta) against the float64 oracle at BASELINE.json's tolerances.  The hand-picked cases of
test_gpu_parity.py stay the first line; this one looks for what they did not think of."""
import os

import numpy as np
import pytest

import oracle as O
from gpu_common import TOL_EPS, TOL_GRAD, dev, max_rel, oracle_cfg, rand_C, rand_fields
from helpers import rel_inf, rel_l2
from paper_2505_03352_b200 import binding as B

pytestmark = pytest.mark.gpu

UP_SUB = [(1, 2), (2, 2), (1, 4), (3, 2), (1, 6), (2, 4), (4, 2), (1, 8)]       # upsample * subpixel in {2, 4, 6, 8}
SCALE = int(os.environ.get("EPSGRAD_SWEEP_SCALE", "1"))          # 3: grids up to 216 cells (mask pixels per control pixel <= 4 only: oracle time)
N_CASES = int(os.environ.get("EPSGRAD_SWEEP_CASES", "40"))      # a longer hunt: EPSGRAD_SWEEP_CASES=400 pytest tests/test_gpu_sweep.py


def draw(i: int):
    """Case i of the sweep: (config kwargs, beta, n_pairs).  Sizes are bounded so the oracle takes about a second."""
    rng = np.random.default_rng([20250503, i])
    pairs = UP_SUB if SCALE == 1 else [(1, 2), (2, 2), (1, 4)]
    u, s = pairs[i % len(pairs)]
    cells = int(rng.integers(6, 72)) * SCALE                          # Yee cells along x: below, at and above 16, 32, 48, 64
    mx = max(1, round(cells / u))
    my = max(1, round(int(rng.integers(6, 72)) * SCALE / u))
    nz = 4 * int(rng.integers(1, 11))
    kind = int(rng.random() < 0.3)
    kw = dict(batch=int(rng.integers(1, 4)) if i % 5 == 0 else 1, mx=mx, my=my, nz=nz, upsample=u, subpixel=s, filter_kind=kind)
    if kind == 0:
        # radii the library takes: every mask pixel within reach of a control pixel, R > (u - 1/s)/sqrt(2) (else den = 0 in
        # the normalised Eq. (2): EPSGRAD_EINVAL), and the tap table within shared memory (s >= 6 at one cell per control
        # pixel: R <= 5.5 cells; EPSGRAD_EUNSUPPORTED beyond) -- both limits are checked in test_gpu_parity.py::test_error_codes
        radii = [r for r in [1.0, 2.0, 3.3, 4.0, 5.5, 8.0, 12.0]
                 if r > (u - 1.0 / s) / np.sqrt(2.0) + 0.05 and not (u == 1 and s >= 6 and r > 5.5)]
        kw["filter_radius"] = float(rng.choice(radii))
    else:
        kw["filter_sigma"] = float(rng.choice([0.8, 2.5, 6.0]))
        kw["filter_radius"] = float(np.ceil(3.2 * kw["filter_sigma"]))
    # slab: faces anywhere, sometimes snapped to cell edges, to the ends of the column or into a single cell
    mode = i % 6
    lo, hi = np.sort(rng.uniform(0.0, nz, 2))
    if hi - lo < 0.05:
        hi = min(float(nz), lo + 0.3)
    if mode == 1:
        lo, hi = float(np.floor(lo)), float(np.ceil(hi))             # faces on cell edges
        if hi == lo: hi = lo + 1.0
    elif mode == 2:
        lo = 0.0                                                      # slab from the bottom of the column
    elif mode == 3:
        hi = float(nz)                                                # ... to its top
    elif mode == 4:
        k = int(rng.integers(0, nz)); lo, hi = k + 0.2, k + 0.7      # inside one cell
    kw["z_lo"], kw["z_hi"] = float(lo), float(hi)
    if i % 4 == 3:
        d = float(rng.choice([1.5, 2.5, 4.0]))
        R = int(np.floor(0.5 * d * s))
        if R >= 1 and min(s * u * mx, s * u * my) >= 2 * R + 1:
            kw["morph_diameter"] = d
    if i % 7 == 0:
        kw["eta"] = float(rng.uniform(0.3, 0.7))
    if i % 9 == 0:
        kw["eps_core"], kw["eps_clad"] = 2.1, 12.0                    # inverted contrast
    if i % 3 == 2:
        kw["normal_delta"] = float(rng.choice([1e-8, 1e-5]))          # guard of the normals (S6); the default is 1e-8 too
    beta = float(np.exp(rng.uniform(0.0, np.log(64.0))))
    return kw, beta, int(rng.integers(1, 4))


def errors(kw, beta, n_pairs, i):
    """Run both sides on case i with configuration kw: worst (eps, dF/dC, dF/dbeta, u) errors over the batch, each divided
    by its tolerance (<= 1 passes).  The tolerances are BASELINE.json's up to beta = 17 and grow with beta beyond: float32
    leaves delta Phi ~ 4 roundings at |Phi'| <= 1/2 = 2.4e-7 on the filter output, the projection turns it into
    delta eps/eps <= (|eps_core - eps_clad|/eps_min) (beta/2) delta Phi = 5.8e-7 beta for Si/SiO2, which is
    1e-5 at beta = 17.  (The BASELINE configs stay at 7e-7 even at beta = 64: their filters average 200 control pixels and
    |Phi'| is ten times smaller; a filter of radius 1 does not smooth at all.)"""
    cfg = B.make_config(**kw)
    C = rand_C(cfg, 1000 + i)
    EF, EA = rand_fields(cfg, n_pairs, 2000 + i)
    plan = B.Plan(cfg)
    dEF, dEA = [dev(f) for f in EF], [dev(f) for f in EA]
    eps, g = plan.eps_forward_vjp(dev(C), beta, dEF, dEA)
    g2, db = plan.eps_vjp_beta(dev(C), beta, dEF, dEA)
    u = plan.unbinarity(dev(C), beta)
    eps, g, g2, db, u = (t.cpu().numpy().astype(np.float64) for t in (eps, g, g2, db, u))
    assert np.array_equal(g, g2), kw
    oc = oracle_cfg(cfg)
    amp = max(1.0, beta / 17.0)
    worst = np.zeros(4)
    for b in range(cfg.batch):
        f, a = [x[b] for x in EF], [x[b] for x in EA]
        eps_ref = O.forward(oc, C[b], beta)
        g_ref, db_ref = O.vjp_beta(oc, C[b], beta, f, a)
        u_ref = O.unbinarity(oc, C[b], beta)
        # d F/d beta is a sum of signed per-pixel terms: same scale as tests/test_gpu_beta.py
        scale = max(abs(db_ref), 1e-3 * np.abs(g_ref).sum())
        worst = np.maximum(worst, [max_rel(eps[b], eps_ref) / (TOL_EPS * amp),
                                   max(rel_inf(g[b], g_ref), rel_l2(g[b], g_ref)) / (TOL_GRAD * amp),
                                   abs(db[b] - db_ref) / (TOL_GRAD * amp * scale),
                                   abs(u[b] - u_ref) / (1e-5 * max(u_ref, 1e-3))])
    return worst


# The cases of a 1300-case hunt at the guard SURVEY.md first proposed, delta = 1e-12: there the rounding noise of
# the float32 Sobel differences (noise^2 ~ 1e-14) became normals on flat parts of the mask.  They always run, at the library's
# default guard (1e-8) like every other case, and must pass at the same tolerances.
HARD = [183, 214, 239, 547, 1092, 1239]
AMPLIFIED = []                     # cases whose tolerances were widened by beta / 17 > 1 (printed by the last test)


@pytest.mark.parametrize("i", list(range(N_CASES)) + [i for i in HARD if i >= N_CASES])
def test_random_configuration(i):
    kw, beta, n_pairs = draw(i)
    if beta > 17.0:
        AMPLIFIED.append((i, round(beta, 1)))
    e = errors(kw, beta, n_pairs, i)
    assert np.all(e < 1), (kw, beta, e)


def test_report_amplified_tolerances():
    """How many of the sweep's cases ran with tolerances above BASELINE.json's (beta > 17: the float32 rounding of the filter
    output times beta).  Informational: run with -s to see the list."""
    n = N_CASES + len([i for i in HARD if i >= N_CASES])
    print(f"\nsweep: {len(AMPLIFIED)} of {n} cases ran with tolerances x beta/17 (beta > 17): {AMPLIFIED}")
    assert len(AMPLIFIED) <= n


@pytest.mark.parametrize("i", range(N_CASES))
def test_random_configuration_every_entry_point(i):
    """The same draws through every other way into the library: separate calls, the serial schedule, the TMA and the dense
    field streams, the host entry point (pinned, in-place windows, and staged), CUDA-graph replay, and an embedding in a
    larger simulation domain -- each against eps_forward_vjp on region-sized device arrays (checked against the oracle
    above), bit for bit wherever the arithmetic order is the same."""
    import torch
    kw, beta, n_pairs = draw(i)
    cfg = B.make_config(**kw)
    rng = np.random.default_rng([77, i])
    Cn = rand_C(cfg, 1000 + i)
    EFn, EAn = rand_fields(cfg, n_pairs, 2000 + i)
    C, EF, EA = dev(Cn), [dev(f) for f in EFn], [dev(f) for f in EAn]
    plan = B.Plan(cfg)
    eps0, g0 = plan.eps_forward_vjp(C, beta, EF, EA)
    G0 = plan.stage_zreduce(EF, EA)
    gb0, db0 = plan.eps_vjp_beta(C, beta, EF, EA)
    assert torch.equal(gb0, g0)
    # separate calls; serial schedule
    assert torch.equal(plan.eps_forward(C, beta), eps0) and torch.equal(plan.eps_vjp(C, beta, EF, EA), g0)
    plan.set_overlap(False)
    eps1, g1 = plan.eps_forward_vjp(C, beta, EF, EA)
    gb1, db1 = plan.eps_vjp_beta(C, beta, EF, EA)
    assert torch.equal(eps1, eps0) and torch.equal(g1, g0) and torch.equal(gb1, g0) and torch.equal(db1, db0)
    plan.set_overlap(True)
    # TMA field stream: same windows, same per-column order
    for mode in (1, 2):            # single-stage TMA; persistent TMA ring
        plan.set_tma(mode)
        plan._ws.fill_(255)                # NaN everywhere: a block this mode skipped cannot borrow the previous mode's result
        assert torch.equal(plan.stage_zreduce(EF, EA), G0) and torch.equal(plan.eps_vjp(C, beta, EF, EA), g0), (kw, mode)
    plan.set_tma(0)
    # eps written by bulk copies out of shared memory: the same affine forms
    plan.set_bulk_stores(True)
    assert torch.equal(plan.eps_forward(C, beta), eps0), kw
    plan.set_bulk_stores(False)
    # the persistent dataflow kernel (whole step; 2-D chains only), where it applies: same tiles, the filter's tap rows summed
    # in two groups instead of three
    try:
        plan.set_fused(1)
        fused = True
    except B.EpsgradError as err:
        assert err.status == B.EUNSUPPORTED
        fused = False
    if fused:
        for mode in (1, 2):
            plan.set_fused(mode)
            eps_f, g_f = plan.eps_forward_vjp(C, beta, EF, EA)
            torch.cuda.synchronize()
            assert float(((eps_f - eps0).abs() / eps0.abs()).max()) < 1e-5 * max(1.0, beta / 17.0), (kw, mode)
            assert float((g_f - g0).abs().max()) <= 1e-4 * max(1.0, beta / 17.0) * float(g0.abs().max()) + 1e-30, (kw, mode)
        plan.set_fused(0)
    # dense field stream: the cells outside the slab have zero weight, the order inside a column is the same
    plan.set_dense_reads(True)
    assert torch.equal(plan.eps_vjp(C, beta, EF, EA), g0)
    plan.set_dense_reads(False)
    # field fills with the L2 evict-first policy forced on / off (by default the size of the launch decides): a cache hint only
    for knob in (1, 2):
        plan.set_tuning(5, knob)
        assert torch.equal(plan.stage_zreduce(EF, EA), G0) and torch.equal(plan.eps_vjp(C, beta, EF, EA), g0), (kw, knob)
    plan.set_tuning(5, 0)
    # eps on the design region only: after a full call on another design, the window call gives the full call's array
    try:
        plan.set_eps_window_only(True)
        windowed = True
    except B.EpsgradError as err:
        assert err.status == B.EUNSUPPORTED
        windowed = False
    if windowed:
        plan.set_eps_window_only(False)
        buf = plan.eps_forward((1.0 - C).contiguous(), beta).clone()
        plan.set_eps_window_only(True)
        ew, gw = plan.eps_forward_vjp(C, beta, EF, EA, eps_out=buf)
        assert torch.equal(ew, eps0) and torch.equal(gw, g0), kw
        plan.set_eps_window_only(False)
    # fields on the design region only: the slab window of every z column, packed (where the layout applies)
    try:
        plan.set_packed_fields(True)
        packed = True
    except B.EpsgradError as err:
        assert err.status == B.EUNSUPPORTED
        packed = False
    if packed:
        k0, nk = plan.packed_window()
        pEF = [f[..., k0:k0 + nk].contiguous() for f in EF]
        pEA = [f[..., k0:k0 + nk].contiguous() for f in EA]
        plan._ws.fill_(255)
        assert torch.equal(plan.stage_zreduce(pEF, pEA), G0) and torch.equal(plan.eps_vjp(C, beta, pEF, pEA), g0), kw
        plan.set_packed_fields(False)
    # CUDA graph replay of the fused call
    eps_g, g_g = torch.empty_like(eps0), torch.empty_like(g0)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        plan.eps_forward_vjp(C, beta, EF, EA, eps_out=eps_g, grad_out=g_g)
    torch.cuda.current_stream().wait_stream(s)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        plan.eps_forward_vjp(C, beta, EF, EA, eps_out=eps_g, grad_out=g_g)
    eps_g.zero_(); g_g.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(eps_g, eps0) and torch.equal(g_g, g0)
    # host entry point: pinned buffers (windows gathered by the copy engine; read in place), then staged whole
    pin = lambda a: torch.from_numpy(a).pin_memory()
    eps_h = torch.empty(plan.eps_shape, dtype=torch.float32).pin_memory()
    g_h = torch.empty(plan.ctrl_shape, dtype=torch.float32).pin_memory()
    hC, hEF, hEA = pin(Cn), [pin(f) for f in EFn], [pin(f) for f in EAn]
    for direct in (2, 1, 0):
        plan.set_host_direct(direct)
        eps_h.zero_(); g_h.zero_()
        plan.eps_forward_vjp_host(hC, beta, hEF, hEA, eps_h, g_h)
        torch.cuda.synchronize()
        assert torch.equal(eps_h, eps0.cpu()) and torch.equal(g_h, g0.cpu()), (kw, direct)
    plan.set_host_direct(2)
    # embedded in a larger domain at a random origin (k0 and nz_full multiples of 4)
    i0, j0, k0 = int(rng.integers(0, 9)), int(rng.integers(0, 9)), 4 * int(rng.integers(0, 3))
    nxf, nyf, nzf = cfg.nx + i0 + int(rng.integers(0, 7)), cfg.ny + j0 + int(rng.integers(0, 7)), cfg.nz + k0 + 4 * int(rng.integers(0, 3))
    shape = (cfg.batch, 3, nxf, nyf, nzf)
    blk = (slice(None), slice(None), slice(i0, i0 + cfg.nx), slice(j0, j0 + cfg.ny), slice(k0, k0 + cfg.nz))
    fEF, fEA = [], []
    for f, lst in [(f, fEF) for f in EF] + [(f, fEA) for f in EA]:
        full = torch.view_as_complex(torch.randn(*shape, 2, device="cuda"))      # anything outside the block must not matter
        full[blk] = f
        lst.append(full)
    plan.set_embedding(nxf, nyf, nzf, i0, j0, k0)
    eps_f = torch.full(shape, -7.0, device="cuda")
    _, g_e = plan.eps_forward_vjp(C, beta, fEF, fEA, eps_out=eps_f)
    gb_e, db_e = plan.eps_vjp_beta(C, beta, fEF, fEA)
    torch.cuda.synchronize()
    assert torch.equal(g_e, g0) and torch.equal(eps_f[blk], eps0), (kw, shape, (i0, j0, k0))
    assert torch.equal(gb_e, g0) and torch.equal(db_e, db0)
    outside = torch.ones(shape, dtype=torch.bool, device="cuda")
    outside[blk] = False
    assert bool((eps_f[outside] == -7.0).all())


@pytest.mark.parametrize("i", range(N_CASES))
def test_random_configuration_in_x_slabs(i):
    """The same draws split along x into 2 or 3 slabs with halos: eps of every slab and the sum of the slabs'
    partial gradients against the undivided plan."""
    import torch
    from paper_2505_03352_b200 import sharding
    kw, beta, n_pairs = draw(i)
    cfg = B.make_config(**kw)
    world = 2 + i % 2
    if cfg.mx < world:
        pytest.skip("fewer control rows than slabs")
    C = dev(rand_C(cfg, 1000 + i))
    EFn, EAn = rand_fields(cfg, n_pairs, 2000 + i)
    EF, EA = [dev(f) for f in EFn], [dev(f) for f in EAn]
    eps0, g0 = B.Plan(cfg).eps_forward_vjp(C, beta, EF, EA)
    u = cfg.upsample
    halo = sharding.slab_halo_cells(cfg.filter_radius, cfg.morph_diameter)
    g_sum = torch.zeros_like(g0)
    for rank in range(world):
        p = sharding.slab_partition(cfg.mx, u, rank, world, halo)
        sub = dict(kw, mx=p["e1"] - p["e0"])
        try:
            plan = B.Plan(B.make_config(**sub))
        except B.EpsgradError as e:                    # a slab narrower than the morphological disk
            assert e.status == B.EUNSUPPORTED and cfg.morph_diameter > 0
            pytest.skip("slab narrower than the morphological disk")
        plan.set_slab(p["x_first"], p["x_count"])
        own = slice(u * p["a0"], u * p["a1"])
        eps_r, g_r = plan.eps_forward_vjp(C[:, p["e0"]:p["e1"]].clone(), beta, [f[:, :, own].clone() for f in EF],
                                          [f[:, :, own].clone() for f in EA])
        assert torch.equal(eps_r, eps0[:, :, own]), (kw, rank, p)
        g_sum[:, p["e0"]:p["e1"]] += g_r
    a, b = g_sum.cpu().numpy().astype(np.float64), g0.cpu().numpy().astype(np.float64)
    assert rel_inf(a, b) < 1e-5 * max(1.0, beta / 17.0), (kw, rel_inf(a, b))


@pytest.mark.parametrize("i", range(N_CASES))
def test_random_configuration_writes_stay_inside_their_buffers(i):
    """compute-sanitizer is closed on this GPU pool, so out-of-bounds writes are looked for directly: the
    outputs and the plan's workspace sit between guard bands filled with a sentinel, and the bands must come back untouched
    (and the results unchanged) after every kind of call (gpu_common.check_guard_bands)."""
    from gpu_common import check_guard_bands
    kw, beta, n_pairs = draw(i)
    cfg = B.make_config(**kw)
    EFn, EAn = rand_fields(cfg, n_pairs, 2000 + i)
    check_guard_bands(cfg, dev(rand_C(cfg, 1000 + i)), [dev(f) for f in EFn], [dev(f) for f in EAn], beta)
