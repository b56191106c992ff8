"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by
element on the same seeded inputs.  Small cases span several tiles (16x16 Yee cells per
CTA) with ragged tails; the BASELINE.json configs follow in test_gpu_configs.py."""
import numpy as np
import pytest
import torch

import oracle as O
from gpu_common import (TOL_EPS, TOL_GRAD, check_forward, check_vjp, dev, max_rel, oracle_cfg, rand_C,
                        rand_fields)
from helpers import rel_inf, rel_l2
from paper_2505_03352_b200 import binding as B

pytestmark = pytest.mark.gpu

# name -> (config kwargs, beta)
CASES = {
    "conic_ragged": (dict(mx=37, my=29, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0), 8.0),
    "conic_r8_beta64": (dict(mx=41, my=50, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0), 64.0),
    "conic_r12_beta32": (dict(mx=45, my=39, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=12.0), 32.0),
    "conic_r6_generic_taps": (dict(mx=30, my=41, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=6.0), 10.0),
    "conic_fractional_radius": (dict(mx=24, my=33, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.3), 12.0),
    "subpixel4": (dict(mx=19, my=23, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0, subpixel=4), 10.0),
    "upsample1": (dict(mx=40, my=35, nz=8, z_lo=1.5, z_hi=6.0, filter_radius=2.5, upsample=1), 9.0),
    "upsample3": (dict(mx=13, my=17, nz=12, z_lo=3.25, z_hi=8.5, filter_radius=5.0, upsample=3), 7.0),
    "upsample4": (dict(mx=11, my=9, nz=8, z_lo=2.0, z_hi=6.0, filter_radius=6.0, upsample=4), 6.0),
    "gaussian": (dict(mx=45, my=38, nz=32, z_lo=14.25, z_hi=17.75, filter_kind=1, filter_radius=8.0,
                      filter_sigma=2.5), 8.0),
    "gaussian_wide": (dict(mx=70, my=40, nz=8, z_lo=2.25, z_hi=5.75, filter_kind=1, filter_radius=32.0,
                           filter_sigma=10.0), 8.0),
    "raw_eq2_eq3": (dict(mx=20, my=22, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0, filter_normalize=0,
                         eta=0.0), 0.5),
    "grid_smaller_than_filter": (dict(mx=5, my=7, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=8.0), 8.0),
    "single_control_row": (dict(mx=1, my=40, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0), 8.0),
    "thin_slab_in_one_cell": (dict(mx=18, my=18, nz=8, z_lo=3.6, z_hi=3.9, filter_radius=3.0), 8.0),
    "slab_fills_z": (dict(mx=18, my=18, nz=8, z_lo=0.0, z_hi=8.0, filter_radius=3.0), 8.0),
    "slab_half_cell_faces": (dict(mx=18, my=18, nz=8, z_lo=2.5, z_hi=5.5, filter_radius=3.0), 8.0),
    "batch3": (dict(batch=3, mx=21, my=19, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0), 8.0),
    # tall columns: a window of 256 chunks per column (4 columns per pass of the field stream), a thin slab far up a column
    # longer than a CTA of the store stream, a column length that no power of two divides; long thin regions
    "tall_full_slab": (dict(mx=9, my=7, nz=512, z_lo=0.0, z_hi=512.0, filter_radius=3.0), 9.0),
    "tall_thin_slab": (dict(mx=9, my=7, nz=2048, z_lo=1000.25, z_hi=1007.75, filter_radius=3.0), 9.0),
    "nz36": (dict(mx=9, my=7, nz=36, z_lo=3.5, z_hi=30.0, filter_radius=3.0), 9.0),
    "long_in_x": (dict(mx=300, my=3, nz=12, z_lo=3.5, z_hi=10.0, filter_radius=3.0), 9.0),
    "long_in_y": (dict(mx=3, my=700, nz=12, z_lo=3.5, z_hi=10.0, filter_radius=3.0), 9.0),
}


@pytest.mark.parametrize("name", list(CASES))
def test_forward_matches_oracle(name):
    kw, beta = CASES[name]
    cfg = B.make_config(**kw)
    check_forward(cfg, rand_C(cfg, 11), beta)


@pytest.mark.parametrize("name", list(CASES))
def test_vjp_matches_oracle(name):
    kw, beta = CASES[name]
    cfg = B.make_config(**kw)
    EF, EA = rand_fields(cfg, 1, 5)
    check_vjp(cfg, rand_C(cfg, 11), beta, EF, EA)


@pytest.mark.parametrize("name", ["conic_ragged", "subpixel4", "gaussian", "raw_eq2_eq3", "upsample3"])
def test_stage_filter_and_eps2d(name):
    kw, beta = CASES[name]
    cfg = B.make_config(**kw)
    C = rand_C(cfg, 3)
    plan = B.Plan(cfg)
    oc = oracle_cfg(cfg)
    phi = plan.stage_filter(dev(C)).cpu().numpy().astype(np.float64)
    e2 = plan.stage_eps2d(dev(C), beta).cpu().numpy().astype(np.float64)
    eta0 = cfg.eta if cfg.filter_normalize else 0.0
    for b in range(cfg.batch):
        st = O.forward_stages(oc, C[b], beta)
        # the kernel stores Phi - eta0; fp32 rounding of a sum of <= ~1e3 O(1) terms
        assert np.max(np.abs(phi[b] - (st["Phi"] - eta0))) < 2e-6 * max(1.0, np.max(np.abs(st["Phi"])))
        assert max_rel(e2[b], st["eps2d"]) < TOL_EPS


@pytest.mark.parametrize("n_pairs", [2, 3, 9])
def test_pairs_accumulate(n_pairs):
    # Eq. (1) summed over field pairs (multi-wavelength, BASELINE configs[2]); 9 > EPSGRAD_MAX_PAIRS chains launches
    cfg = B.make_config(mx=17, my=21, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0)
    EF, EA = rand_fields(cfg, n_pairs, 21)
    check_vjp(cfg, rand_C(cfg, 2), 8.0, EF, EA)


def test_zreduce_planes_match_definition():
    cfg = B.make_config(batch=2, mx=9, my=11, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=3.0)
    EF, EA = rand_fields(cfg, 2, 8)
    plan = B.Plan(cfg)
    g = plan.stage_zreduce([dev(f) for f in EF], [dev(f) for f in EA]).cpu().numpy().astype(np.float64)
    G3 = sum(-2.0 * (f.astype(np.complex128) * a.astype(np.complex128)).real for f, a in zip(EF, EA))
    wxy, wz = O.zweights(oracle_cfg(cfg))
    ref = np.stack([G3[:, 0] @ wxy, G3[:, 1] @ wxy, G3[:, 2] @ (wz == 1.0), G3[:, 2, :, :, 5], G3[:, 2, :, :, 9]], axis=1)
    assert rel_inf(g, ref) < 1e-5


def test_tma_field_reads_give_the_same_bits():
    # the TMA variant of the field stream (epsgrad_plan_set_tma) against the LDGSTS kernel: same windows, same per-column sums
    for kw, n_pairs in ((dict(mx=23, my=18, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=4.0), 1),
                        (dict(batch=2, mx=67, my=59, nz=32, z_lo=14.25, z_hi=17.75, filter_radius=4.0), 3),
                        (dict(mx=130, my=131, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0), 9)):
        cfg = B.make_config(**kw)
        C = dev(rand_C(cfg, 4))
        EFn, EAn = rand_fields(cfg, n_pairs, 9)
        EF, EA = [dev(f) for f in EFn], [dev(f) for f in EAn]
        plan = B.Plan(cfg)
        g0, G0 = plan.eps_vjp(C, 16.0, EF, EA), plan.stage_zreduce(EF, EA)
        plan.set_tma(True)
        g1, G1 = plan.eps_vjp(C, 16.0, EF, EA), plan.stage_zreduce(EF, EA)
        plan.set_tma(False)
        plan.set_tuning(5, 2)                                     # field fills without the evict-first L2 policy (the default has it)
        g2, G2 = plan.eps_vjp(C, 16.0, EF, EA), plan.stage_zreduce(EF, EA)
        torch.cuda.synchronize()
        assert torch.equal(G0, G1) and torch.equal(g0, g1) and torch.equal(G0, G2) and torch.equal(g0, g2)


def test_dense_reads_give_the_same_gradient():
    cfg = B.make_config(mx=23, my=18, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=4.0)
    C = rand_C(cfg, 4)
    EF, EA = rand_fields(cfg, 1, 9)
    plan = B.Plan(cfg)
    check_vjp(cfg, C, 16.0, EF, EA, plan=plan)
    plan.set_dense_reads(True)
    check_vjp(cfg, C, 16.0, EF, EA, plan=plan)


def test_profiling_and_timeline_hooks_name_every_kernel():
    cfg = B.make_config(mx=23, my=18, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0)
    C = dev(rand_C(cfg, 4))
    EFn, EAn = rand_fields(cfg, 1, 9)
    EF, EA = [dev(f) for f in EFn], [dev(f) for f in EAn]
    plan = B.Plan(cfg)
    eps0, g0 = plan.eps_forward_vjp(C, 8.0, EF, EA)
    plan.set_profiling(True)                                  # serial schedule, one event after each kernel
    eps1, g1 = plan.eps_forward_vjp(C, 8.0, EF, EA)
    times = plan.last_kernel_times()
    plan.set_profiling(False)
    assert [n for n, _ in times] == ["filter", "fwd2d", "zreduce", "extrude", "maskgrad", "filterT"]
    assert all(ms > 0 for _, ms in times)
    plan.set_timeline(True)                                   # device-clock stamps on both streams
    eps2, g2 = plan.eps_forward_vjp(C, 8.0, EF, EA)
    tl = plan.read_timeline()
    plan.set_timeline(False)
    assert sorted(n for n, _ in tl) == sorted(["begin", "filter", "fwd2d", "zreduce", "extrude", "maskgrad", "filterT"])
    assert all(t >= 0 for _, t in tl)
    assert torch.equal(eps0, eps1) and torch.equal(g0, g1) and torch.equal(eps0, eps2) and torch.equal(g0, g2)


def test_forward_vjp_equals_separate_calls_and_keeps_inputs():
    cfg = B.make_config(mx=30, my=26, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0)
    C = dev(rand_C(cfg, 6))
    EFn, EAn = rand_fields(cfg, 2, 10)
    EF, EA = [dev(f) for f in EFn], [dev(f) for f in EAn]
    C0, F0 = C.clone(), EF[0].clone()
    plan = B.Plan(cfg)
    eps1 = plan.eps_forward(C, 8.0)
    g1 = plan.eps_vjp(C, 8.0, EF, EA)
    eps2, g2 = plan.eps_forward_vjp(C, 8.0, EF, EA)
    torch.cuda.synchronize()
    assert torch.equal(eps1, eps2) and torch.equal(g1, g2)
    assert torch.equal(C, C0) and torch.equal(EF[0], F0)
    assert plan.last_launches() >= 4


@pytest.mark.parametrize("n_pairs", [1, 9, 17])
def test_entry_points_agree_bitwise(n_pairs):
    # eps_forward_vjp, eps_forward and eps_vjp share their kernels; the two-stream schedule and the serial one give the
    # same bits; more than EPSGRAD_MAX_PAIRS pairs are chained through accumulating launches
    cfg = B.make_config(batch=2, mx=27, my=22, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0)
    C = dev(rand_C(cfg, 16))
    EFn, EAn = rand_fields(cfg, n_pairs, 17)
    EF, EA = [dev(f) for f in EFn], [dev(f) for f in EAn]
    plan = B.Plan(cfg)
    eps0, g0 = plan.eps_forward_vjp(C, 8.0, EF, EA)
    assert plan.last_launches() == 5 + (n_pairs + 7) // 8
    eps1 = plan.eps_forward(C, 8.0)
    g1 = plan.eps_vjp(C, 8.0, EF, EA)
    plan.set_overlap(False)
    eps2, g2 = plan.eps_forward_vjp(C, 8.0, EF, EA)
    g3 = plan.eps_vjp(C, 8.0, EF, EA)
    plan.set_overlap(True)
    torch.cuda.synchronize()
    assert torch.equal(eps0, eps1) and torch.equal(g0, g1) and torch.equal(eps0, eps2) and torch.equal(g0, g2) and torch.equal(g0, g3)
    if n_pairs > 1:
        # linearity in the pairs: the sum of single-pair gradients
        gs = sum(plan.eps_vjp(C, 8.0, [f], [a]).double() for f, a in zip(EF, EA))
        assert float((gs - g0.double()).abs().max()) < 1e-5 * float(g0.abs().max())


def test_calls_are_cuda_graph_capturable():
    cfg = B.make_config(mx=25, my=31, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0)
    C = dev(rand_C(cfg, 18))
    EFn, EAn = rand_fields(cfg, 1, 19)
    EF, EA = [dev(f) for f in EFn], [dev(f) for f in EAn]
    plan = B.Plan(cfg)
    eps_ref, g_ref = plan.eps_forward_vjp(C, 8.0, EF, EA)
    eps, g = torch.zeros_like(eps_ref), torch.zeros_like(g_ref)
    torch.cuda.synchronize()
    for overlap in (True, False):
        plan.set_overlap(overlap)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            plan.eps_forward_vjp(C, 8.0, EF, EA, eps, g)
        eps.zero_(); g.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(eps, eps_ref) and torch.equal(g, g_ref)


@pytest.mark.parametrize("z", [
    (3.2, 3.6),        # slab inside one cell: no full E_x/E_y cell, two fractional E_z cells
    (0.0, 8.0),        # slab = the whole grid: every cell full, no face inside the grid for E_x/E_y
    (-1.0, 2.5),       # sticks out below: clipped at the grid
    (6.3, 11.0),       # sticks out above
    (3.0, 5.0),        # faces on cell boundaries: no fractional E_x/E_y cell, two half-filled E_z cells
    (9.0, 10.0),       # entirely outside the grid: eps = eps_clad, dF/dC = 0
])
def test_degenerate_slabs(z):
    cfg = B.make_config(mx=14, my=11, nz=8, z_lo=z[0], z_hi=z[1], filter_radius=3.0)
    C = rand_C(cfg, 71)
    EF, EA = rand_fields(cfg, 2, 72)
    plan = B.Plan(cfg)
    check_forward(cfg, C, 8.0, plan)
    g = plan.eps_vjp(dev(C), 8.0, [dev(f) for f in EF], [dev(f) for f in EA]).cpu().numpy().astype(np.float64)
    ref = O.vjp(oracle_cfg(cfg), C[0], 8.0, [f[0] for f in EF], [f[0] for f in EA])
    if z[0] >= cfg.nz:
        assert np.all(ref == 0.0) and np.all(g == 0.0)
        assert np.all(plan.eps_forward(dev(C), 8.0).cpu().numpy() == np.float32(cfg.eps_clad))
    else:
        assert rel_inf(g[0], ref) < TOL_GRAD and rel_l2(g[0], ref) < TOL_GRAD


def test_real_cotangent_special_case():
    # VJP with an arbitrary (real) field w: E_F = -w/2, E_A = 1
    cfg = B.make_config(mx=12, my=14, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0)
    C = rand_C(cfg, 1)
    w = np.random.default_rng(5).standard_normal((1, 3, cfg.nx, cfg.ny, cfg.nz))
    EF = [(-0.5 * w).astype(np.complex64)]
    EA = [np.ones_like(EF[0])]
    g = B.Plan(cfg).eps_vjp(dev(C), 8.0, [dev(EF[0])], [dev(EA[0])]).cpu().numpy().astype(np.float64)
    ref = O.vjp_real(oracle_cfg(cfg), C[0], 8.0, (-2.0 * (EF[0].astype(np.complex128) * EA[0]).real)[0])
    assert rel_inf(g[0], ref) < TOL_GRAD and rel_l2(g[0], ref) < TOL_GRAD


def test_uniform_control_gives_uniform_mixing_value():
    # north_star invariant, on the GPU path itself
    cfg = B.make_config(mx=33, my=20, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0)
    plan = B.Plan(cfg)
    for c0 in (0.0, 0.43, 1.0):
        e2 = plan.stage_eps2d(torch.full(plan.ctrl_shape, c0, device="cuda"), 8.0).cpu().numpy().astype(np.float64)
        rho = 0.5 * (1 + np.tanh(8.0 * (np.float64(np.float32(c0)) - 0.5)))
        ref = rho * cfg.eps_core + (1 - rho) * cfg.eps_clad
        assert np.max(np.abs(e2 - ref)) < 2e-6 * ref
    eps = plan.eps_forward(torch.rand(plan.ctrl_shape, device="cuda"), 300.0).cpu().numpy()
    assert eps.min() >= np.float32(cfg.eps_clad) * (1 - 1e-6) and eps.max() <= np.float32(cfg.eps_core) * (1 + 1e-6)


def test_host_entry_point_matches_device_entry_point():
    cfg = B.make_config(mx=20, my=24, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0)
    Cn = rand_C(cfg, 12)
    EFn, EAn = rand_fields(cfg, 2, 13)
    plan = B.Plan(cfg)
    eps_d, g_d = plan.eps_forward_vjp(dev(Cn), 8.0, [dev(f) for f in EFn], [dev(f) for f in EAn])
    pin = lambda a: torch.from_numpy(a).pin_memory()
    eps_h = torch.empty(plan.eps_shape, dtype=torch.float32).pin_memory()
    g_h = torch.empty(plan.ctrl_shape, dtype=torch.float32).pin_memory()
    plan.eps_forward_vjp_host(pin(Cn), 8.0, [pin(f) for f in EFn], [pin(f) for f in EAn], eps_h, g_h)
    torch.cuda.synchronize()
    assert torch.equal(eps_h, eps_d.cpu()) and torch.equal(g_h, g_d.cpu())
    # only the slab windows of pinned fields cross the bus: cells 6..9 for x, y (2 chunks of 16 B), 5..9 for z (3 chunks).
    # Default (mode 2): the union window (3 chunks) of every column of every component, gathered by the copy engine
    h2d, d2h = plan.last_copy_bytes()
    ncol = cfg.batch * cfg.nx * cfg.ny
    assert h2d == Cn.nbytes + 2 * 2 * ncol * 3 * 3 * 16 and d2h == eps_h.numel() * 4 + g_h.numel() * 4
    # mode 1: read in place by the kernel, exactly the chunks of each component's window
    plan.set_host_direct(1)
    eps_h.zero_(); g_h.zero_()
    plan.eps_forward_vjp_host(pin(Cn), 8.0, [pin(f) for f in EFn], [pin(f) for f in EAn], eps_h, g_h)
    torch.cuda.synchronize()
    assert torch.equal(eps_h, eps_d.cpu()) and torch.equal(g_h, g_d.cpu())
    assert plan.last_copy_bytes()[0] == Cn.nbytes + 2 * 2 * ncol * (2 + 2 + 3) * 16
    # gradient only: mode 2 behaves as mode 1
    plan.set_host_direct(2)
    g_h.zero_()
    plan.eps_forward_vjp_host(pin(Cn), 8.0, [pin(f) for f in EFn], [pin(f) for f in EAn], None, g_h)
    torch.cuda.synchronize()
    assert torch.equal(g_h, g_d.cpu()) and plan.last_copy_bytes()[0] == Cn.nbytes + 2 * 2 * ncol * (2 + 2 + 3) * 16
    # whole-field staging (also the fallback for pageable buffers) gives the same bits
    plan.set_host_direct(False)
    eps_h.zero_(); g_h.zero_()
    plan.eps_forward_vjp_host(pin(Cn), 8.0, [pin(f) for f in EFn], [pin(f) for f in EAn], eps_h, g_h)
    torch.cuda.synchronize()
    assert torch.equal(eps_h, eps_d.cpu()) and torch.equal(g_h, g_d.cpu())
    h2d, d2h = plan.last_copy_bytes()
    assert h2d == Cn.nbytes + sum(f.nbytes for f in EFn + EAn)
    plan.set_host_direct(2)
    eps_h.zero_(); g_h.zero_()
    plan.eps_forward_vjp_host(torch.from_numpy(Cn), 8.0, [torch.from_numpy(f) for f in EFn], [torch.from_numpy(f) for f in EAn], eps_h, g_h)
    torch.cuda.synchronize()
    assert torch.equal(eps_h, eps_d.cpu()) and torch.equal(g_h, g_d.cpu())
    assert plan.last_copy_bytes()[0] == Cn.nbytes + sum(f.nbytes for f in EFn + EAn)     # pageable: staged whole


def test_error_codes():
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=1.0))
    assert e.value.status == B.EINVAL
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, subpixel=3))
    assert e.value.status == B.EINVAL
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, upsample=5))      # 10 mask pixels per control pixel: no phase table
    assert e.value.status == B.EUNSUPPORTED
    # cone too small to reach the mask pixels midway between control pixels: the normalised Eq. (2) would be 0/0 there
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, upsample=2, subpixel=4, filter_radius=1.0))
    assert e.value.status == B.EINVAL
    B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, upsample=2, subpixel=4, filter_radius=1.0, filter_normalize=0))
    B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, upsample=2, subpixel=4, filter_radius=1.3))
    # tap table of the conic filter beyond shared memory
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(mx=40, my=40, nz=8, z_lo=2.0, z_hi=5.0, upsample=1, subpixel=8, filter_radius=12.0))
    assert e.value.status == B.EUNSUPPORTED
    # field window wider than 512 cells: the scalar field kernel; refused only where that one does not apply (embedded fields)
    cfg = B.make_config(mx=4, my=4, nz=1024, z_lo=3.5, z_hi=1000.0)
    plan = B.Plan(cfg)
    Cw = rand_C(cfg, 1)
    EFw, EAw = rand_fields(cfg, 1, 2)
    gw = plan.eps_vjp(dev(Cw), 8.0, [dev(EFw[0])], [dev(EAw[0])]).cpu().numpy().astype(np.float64)[0]
    gw_ref = O.vjp(oracle_cfg(cfg), Cw[0], 8.0, [EFw[0][0]], [EAw[0][0]])
    assert np.max(np.abs(gw - gw_ref)) < TOL_GRAD * np.max(np.abs(gw_ref))
    plan.set_embedding(8, 8, 1024, 0, 0, 0)
    f = torch.zeros(plan.field_shape, dtype=torch.complex64, device="cuda")
    with pytest.raises(B.EpsgradError) as e:
        plan.eps_vjp(dev(Cw), 8.0, [f], [f])
    assert e.value.status == B.EUNSUPPORTED
    # beyond the 32-bit plane indices: refused at plan creation, before anything is allocated
    with pytest.raises(B.EpsgradError) as e:
        B.Plan(B.make_config(batch=64, mx=4096, my=4096, nz=32, z_lo=14.25, z_hi=17.75))
    assert e.value.status == B.EUNSUPPORTED
    # empty inputs: no design, no control pixel, no field pair
    for kw in (dict(batch=0, mx=8, my=8), dict(mx=0, my=8), dict(mx=8, my=0)):
        with pytest.raises(B.EpsgradError) as e:
            B.Plan(B.make_config(**dict(dict(nz=8, z_lo=2.0, z_hi=5.0), **kw)))
        assert e.value.status == B.EINVAL
    plan = B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0))
    Cd, gd = torch.rand(plan.ctrl_shape, device="cuda"), torch.empty(plan.ctrl_shape, device="cuda")
    assert B.lib().eps_vjp(plan._h, Cd.data_ptr(), 8.0, 0, None, None, gd.data_ptr(), None) == B.EINVAL
    assert B.lib().eps_vjp(plan._h, Cd.data_ptr(), 8.0, 1, None, None, gd.data_ptr(), None) == B.EINVAL
    assert B.lib().eps_forward(plan._h, None, 8.0, gd.data_ptr(), None) == B.EINVAL
    assert B.lib().eps_forward(plan._h, Cd.data_ptr(), float("nan"), gd.data_ptr(), None) == B.EINVAL
    assert B.lib().eps_forward(plan._h, Cd.data_ptr() + 4, 8.0, gd.data_ptr(), None) == B.EINVAL      # misaligned
    with pytest.raises(B.EpsgradError) as e:
        plan.eps_forward(torch.rand(plan.ctrl_shape, device="cuda"), -1.0)
    assert e.value.status == B.EINVAL
    # guard of the normals: 0, a denormal (rcp.approx.ftz would flush it) or NaN would make n^2 = 0/0 on every flat cell and break
    # the uniform-C invariant; non-finite eta or slab faces
    for bad in (dict(normal_delta=0.0), dict(normal_delta=1e-40), dict(normal_delta=float("nan")), dict(normal_delta=-1e-8),
                dict(eta=float("nan")), dict(eta=float("inf")), dict(z_lo=float("-inf"))):
        with pytest.raises(B.EpsgradError) as e:
            B.Plan(B.make_config(**dict(dict(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0), **bad)))
        assert e.value.status == B.EINVAL, bad
    # the smallest guard the library takes keeps a uniform design uniform
    plan = B.Plan(B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, normal_delta=1e-30))
    e1 = plan.eps_forward(torch.full(plan.ctrl_shape, 0.5, device="cuda"), 8.0)
    assert bool(torch.isfinite(e1).all()) and float((e1[:, :, :, :, 3] - 7.0975).abs().max()) < 1e-5


def test_two_plans_on_two_streams_do_not_interfere():
    # a plan carries its own workspace, auxiliary stream and events: calls of different plans interleaved on different streams
    # give the bits each gives alone
    kws = [dict(mx=37, my=29, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0),
           dict(batch=2, mx=45, my=38, nz=32, z_lo=14.25, z_hi=17.75, filter_kind=1, filter_radius=8.0, filter_sigma=2.5)]
    plans, ins, ref = [], [], []
    for k, kw in enumerate(kws):
        cfg = B.make_config(**kw)
        EF, EA = rand_fields(cfg, 2, 70 + k)
        plans.append(B.Plan(cfg))
        ins.append((dev(rand_C(cfg, 60 + k)), [dev(f) for f in EF], [dev(f) for f in EA]))
        ref.append(plans[k].eps_forward_vjp(ins[k][0], 8.0 + k, ins[k][1], ins[k][2]))
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [[], []]
    for rep in range(6):
        for k in (0, 1):
            with torch.cuda.stream(streams[k]):
                outs[k].append(plans[k].eps_forward_vjp(ins[k][0], 8.0 + k, ins[k][1], ins[k][2]))
    torch.cuda.synchronize()
    for k in (0, 1):
        for eps, g in outs[k]:
            assert torch.equal(eps, ref[k][0]) and torch.equal(g, ref[k][1])


@pytest.mark.skipif("PYTEST_XDIST_WORKER" in __import__("os").environ, reason="free device memory is shared with the other workers")
def test_plans_are_released():
    cfg = B.make_config(mx=64, my=64, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0, morph_diameter=2.0)
    C = dev(rand_C(cfg, 3))
    torch.cuda.synchronize()
    free0 = None
    for i in range(60):
        plan = B.Plan(cfg)
        plan.eps_forward(C, 8.0)
        del plan
        torch.cuda.synchronize()
        if i == 9:
            torch.cuda.empty_cache()
            free0 = torch.cuda.mem_get_info()[0]
    torch.cuda.empty_cache()
    assert torch.cuda.mem_get_info()[0] >= free0 - (8 << 20)          # device tables, streams and events go with the plan


@pytest.mark.parametrize("kw,beta", [
    (dict(mx=32, my=32, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0), 8.0),                 # Tiny's geometry: one ragged tile per block
    (dict(mx=67, my=13, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=4.0), 16.0),                 # 2 row blocks (64 + 3), 2 column blocks (8 + 5)
    (dict(batch=3, mx=5, my=70, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=8.0), 64.0),         # fewer control rows than taps; saturated tanh
    (dict(mx=130, my=41, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=8.0, filter_normalize=0, eta=0.0), 1.5),
    (dict(mx=270, my=23, nz=4, z_lo=0.5, z_hi=3.5, filter_radius=12.0), 32.0),                 # streamed weights: 256 + 14 rows
    (dict(batch=2, mx=9, my=9, nz=4, z_lo=0.5, z_hi=3.5, filter_radius=12.0), 8.0),            # a grid smaller than the filter
    (dict(batch=2, mx=500, my=19, nz=4, z_lo=0.5, z_hi=3.5, filter_radius=12.0), 16.0),        # transposed filter: 3 row blocks of 192 staged rows
    (dict(mx=21, my=300, nz=4, z_lo=0.5, z_hi=3.5, filter_radius=8.0), 16.0),                  # 38 column blocks, the last one ragged
])
def test_tensor_core_filter_matches_the_oracle(kw, beta):
    """Eq. (2) by tcgen05 MMAs (filter_tc.cuh, forced on: by default it runs only on large control grids): the filter output
    against the FFMA stencil, and eps / dF/dC against the oracle at BASELINE.json's tolerances."""
    cfg = B.make_config(**kw)
    C = rand_C(cfg, 21)
    plan = B.Plan(cfg)
    plan.set_tensor_cores(0)
    phi0 = plan.stage_filter(dev(C))
    plan.set_tensor_cores(1)
    phi1 = plan.stage_filter(dev(C))
    torch.cuda.synchronize()
    # the tensor core accumulates in float32 with a coarser rounding than FFMA: a few 1e-6 of the largest |Phi|
    assert float((phi1 - phi0).abs().max()) < 8e-6 * max(0.5, float(phi0.abs().max())), float((phi1 - phi0).abs().max())
    check_forward(cfg, C, beta, plan)
    EF, EA = rand_fields(cfg, 2, 22)
    check_vjp(cfg, C, beta, EF, EA, plan)
    # the transposed filter (filterT_tc.cuh) against the FFMA kernel on the same cotangent: two-term tf32 operands, float32 sums
    g1 = plan.eps_vjp(dev(C), beta, [dev(f) for f in EF], [dev(f) for f in EA]).clone()
    plan.set_tensor_cores(0)
    g0 = plan.eps_vjp(dev(C), beta, [dev(f) for f in EF], [dev(f) for f in EA])
    torch.cuda.synchronize()
    assert float((g1 - g0).abs().max()) <= 1e-5 * float(g0.abs().max()), float((g1 - g0).abs().max() / g0.abs().max())
    with pytest.raises(B.EpsgradError) as e:                      # the Gaussian filter is separable: no banded matrices for it
        B.Plan(B.make_config(mx=16, my=16, nz=8, z_lo=2.0, z_hi=5.0, filter_kind=1, filter_radius=6.0, filter_sigma=2.0)).set_tensor_cores(1)
    assert e.value.status == B.EUNSUPPORTED


@pytest.mark.parametrize("kw,beta,n_pairs", [
    (dict(mx=33, my=21, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0), 16.0, 2),          # the paper's slab: cells 26..35 of 64
    (dict(batch=2, mx=17, my=40, nz=32, z_lo=14.25, z_hi=17.75, filter_kind=1, filter_radius=6.0, filter_sigma=2.0), 8.0, 1),   # Wide batch's slab
    (dict(mx=12, my=12, nz=16, z_lo=0.0, z_hi=16.0, filter_radius=4.0), 8.0, 3),                 # the slab is the whole column
    (dict(mx=20, my=9, nz=24, z_lo=3.5, z_hi=4.25, filter_radius=4.0), 32.0, 9),                # a slab inside one cell; more than 8 pairs
    (dict(mx=12, my=14, nx_cells=70, ny_cells=81, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0), 16.0, 2),   # Fig. 4's 5.8 cells per control pixel
    (dict(batch=2, mx=24, my=20, nz=32, z_lo=14.25, z_hi=17.75, filter_radius=6.0, morph_diameter=3.0), 12.0, 1),  # morphological filters on
])
def test_packed_fields_give_the_same_gradient(kw, beta, n_pairs):
    """epsgrad_plan_set_packed_fields: E_F / E_A restricted to the z cells of the slab window (fields on Omega_D only)
    give bit for bit the dF/dC of full columns, through every entry point that reads fields; what lies outside the window
    never mattered (NaNs there change nothing); options that address the fields differently are refused."""
    cfg = B.make_config(**kw)
    C = rand_C(cfg, 31)
    EF, EA = rand_fields(cfg, n_pairs, 32)
    plan = B.Plan(cfg)
    full = lambda fs: [dev(f) for f in fs]
    g0 = plan.eps_vjp(dev(C), beta, full(EF), full(EA)).clone()
    gb0, db0 = plan.eps_vjp_beta(dev(C), beta, full(EF), full(EA))
    gb0, db0 = gb0.clone(), db0.clone()
    z0 = plan.stage_zreduce(full(EF), full(EA)).clone()
    check_vjp(cfg, C, beta, EF, EA, plan)
    k0, n = plan.packed_window()
    assert 0 <= k0 and k0 + n <= cfg.nz and k0 % 2 == 0 and n % 2 == 0
    assert k0 <= int(np.floor(kw["z_lo"])) and k0 + n >= min(cfg.nz, int(np.ceil(kw["z_hi"]))), (k0, n)     # the window holds the slab
    # full columns with NaNs outside the window: same bits
    def poisoned(fs):
        out = []
        for f in fs:
            t = dev(f).clone()
            v = torch.view_as_real(t)
            v[..., :k0, :] = float("nan")
            v[..., k0 + n:, :] = float("nan")
            out.append(t)
        return out
    assert torch.equal(plan.eps_vjp(dev(C), beta, poisoned(EF), poisoned(EA)), g0)
    plan.set_packed_fields(True)
    pack = lambda fs: [dev(f)[..., k0:k0 + n].contiguous() for f in fs]
    assert torch.equal(plan.eps_vjp(dev(C), beta, pack(EF), pack(EA)), g0)
    eps1, g1 = plan.eps_forward_vjp(dev(C), beta, pack(EF), pack(EA))
    assert torch.equal(g1, g0) and tuple(eps1.shape) == plan.eps_shape
    gb1, db1 = plan.eps_vjp_beta(dev(C), beta, pack(EF), pack(EA))
    assert torch.equal(gb1, gb0) and torch.equal(db1, db0)
    assert torch.equal(plan.stage_zreduce(pack(EF), pack(EA)), z0)
    for call in (lambda: plan.set_embedding(cfg.nx + 8, cfg.ny + 8, cfg.nz, 4, 4, 0), lambda: plan.set_slab(0, cfg.nx // 2),
                 lambda: plan.set_dense_reads(True)):
        with pytest.raises(B.EpsgradError) as e:
            call()
        assert e.value.status == B.EUNSUPPORTED
    plan.set_packed_fields(False)
    assert torch.equal(plan.eps_vjp(dev(C), beta, full(EF), full(EA)), g0)
    plan.set_dense_reads(True)
    with pytest.raises(B.EpsgradError) as e:
        plan.set_packed_fields(True)
    assert e.value.status == B.EUNSUPPORTED


@pytest.mark.parametrize("kw,beta", [
    (dict(mx=33, my=21, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0), 16.0),               # the paper's slab: sectors of cells 24..39
    (dict(batch=2, mx=17, my=40, nz=32, z_lo=14.25, z_hi=17.75, filter_kind=1, filter_radius=6.0, filter_sigma=2.0), 8.0),
    (dict(mx=12, my=12, nz=16, z_lo=0.0, z_hi=16.0, filter_radius=4.0), 8.0),                    # the slab is the whole column
    (dict(mx=20, my=9, nz=12, z_lo=3.5, z_hi=4.25, filter_radius=4.0), 32.0),                   # a slab inside one cell; nz/4 odd
    (dict(mx=14, my=10, nz=24, z_lo=20.5, z_hi=24.0, filter_radius=4.0), 8.0),                  # the slab ends at the top of the column
    (dict(mx=12, my=14, nx_cells=70, ny_cells=81, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0), 16.0),
])
def test_eps_window_only_rewrites_the_slab_window_and_nothing_else(kw, beta):
    """epsgrad_plan_set_eps_window_only: after ONE full call, a window call on a NEW design leaves the array bit for bit
    equal to a full call on the new design; on an array of sentinels it writes whole 32-byte sectors around the slab and nothing
    else; the oracle agrees on every cell; eps_forward_vjp does the same and its gradient does not change."""
    cfg = B.make_config(**kw)
    C1, C2 = rand_C(cfg, 61), rand_C(cfg, 62)
    EF, EA = rand_fields(cfg, 1, 63)
    plan = B.Plan(cfg)
    full2 = plan.eps_forward(dev(C2), beta).clone()
    g2 = plan.eps_vjp(dev(C2), beta, [dev(f) for f in EF], [dev(f) for f in EA]).clone()
    buf = plan.eps_forward(dev(C1), beta).clone()                 # the one full call
    assert not torch.equal(buf, full2)
    plan.set_eps_window_only(True)
    plan.eps_forward(dev(C2), beta, buf)
    assert torch.equal(buf, full2)
    ref = np.stack([O.forward(oracle_cfg(cfg), C2[b], beta) for b in range(cfg.batch)])
    assert max_rel(buf.cpu().numpy().astype(np.float64), ref) < TOL_EPS
    # what is written: whole sectors (8 cells) around the slab, nothing else
    SENT = -7.0
    s = torch.full(plan.eps_shape, SENT, dtype=torch.float32, device="cuda")
    plan.eps_forward(dev(C2), beta, s)
    written = (s != SENT)
    per_k = written.reshape(-1, cfg.nz).any(dim=0).cpu().numpy()
    assert (written.reshape(-1, cfg.nz).all(dim=0).cpu().numpy() == per_k).all()      # a z cell is written in every column or in none
    ks = np.nonzero(per_k)[0]
    k_lo, k_hi = int(np.floor(kw["z_lo"])), int(np.ceil(kw["z_hi"]))               # the slab's cells: [k_lo, k_hi)
    assert ks.min() <= k_lo and ks.max() >= min(cfg.nz, k_hi) - 1, (ks.min(), ks.max())
    assert ks.min() % 8 == 0 and ((ks.max() + 1) % 8 == 0 or ks.max() + 1 == cfg.nz), (ks.min(), ks.max())
    assert len(ks) == ks.max() - ks.min() + 1 and len(ks) <= min(cfg.nz, (k_hi - k_lo) + 1 + 16)
    assert torch.equal(s[written], full2[written])
    assert bool((full2[~written] == float(np.float32(cfg.eps_clad))).all())           # everything it skips is cladding
    # the one-call path, and the gradient
    plan.set_eps_window_only(False)
    buf2 = plan.eps_forward(dev(C1), beta).clone()
    plan.set_eps_window_only(True)
    e3, g3 = plan.eps_forward_vjp(dev(C2), beta, [dev(f) for f in EF], [dev(f) for f in EA], buf2)
    assert torch.equal(e3, full2) and torch.equal(g3, g2)
    plan.set_eps_window_only(False)
    assert torch.equal(plan.eps_forward(dev(C2), beta), full2)
    if cfg.nx_cells == 0 and cfg.batch == 1:
        # the host entry point writes its eps buffer whole: refused while the option is on, as with packed fields
        plan.set_eps_window_only(True)
        with pytest.raises(B.EpsgradError) as e:
            plan.eps_forward_vjp_host(torch.from_numpy(C2).pin_memory(), beta, [torch.from_numpy(f).pin_memory() for f in EF],
                                      [torch.from_numpy(f).pin_memory() for f in EA],
                                      torch.empty(plan.eps_shape, dtype=torch.float32).pin_memory(),
                                      torch.empty(plan.ctrl_shape, dtype=torch.float32).pin_memory())
        assert e.value.status == B.EUNSUPPORTED
        plan.set_eps_window_only(False)
    with pytest.raises(B.EpsgradError) as e:                              # columns that are not whole 16-byte pieces
        B.Plan(B.make_config(mx=8, my=8, nz=10, z_lo=2.0, z_hi=5.0, filter_radius=3.0)).set_eps_window_only(True)
    assert e.value.status == B.EUNSUPPORTED
