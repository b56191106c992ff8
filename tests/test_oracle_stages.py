"""Pins of the float64 oracle, stage by stage (CPU only).

Each test checks an oracle stage against something other than the oracle: a closed
form, a hand-made input whose answer is known, a library routine the stage reduces
to, brute force on a tiny input, or the adjoint identity for the transposes.
"""
import math

import numpy as np
import pytest
import torch

import oracle as O
from helpers import small_cfg, torch_average, torch_filter, torch_sobel

RNG = np.random.default_rng(1234)


# ------------------------------------------------------------------ filter, Eq. (2)
@pytest.mark.parametrize("kind,radius,sigma", [(0, 3.0, 0.0), (0, 2.5, 0.0), (1, 4.0, 1.7)])
def test_filter_delta_gives_kernel(kind, radius, sigma):
    cfg = small_cfg(mx=9, my=7, filter_kind=kind, radius=radius, sigma=sigma, normalize=0)
    C = np.zeros((cfg.mx, cfg.my)); C[4, 3] = 1.0
    Phi = O.filter(cfg, C)
    u = cfg.nx / cfg.mx
    for p in range(cfg.px):
        for q in range(cfg.py):
            dx, dy = (p + .5) / cfg.s - u * 4.5, (q + .5) / cfg.s - u * 3.5
            if kind == 0:
                ref = max(0.0, 1 - math.hypot(dx, dy) / radius)
            else:
                ref = math.exp(-(dx * dx + dy * dy) / (2 * sigma ** 2)) if max(abs(dx), abs(dy)) <= radius else 0.0
            assert abs(Phi[p, q] - ref) < 1e-15


@pytest.mark.parametrize("kind", [0, 1])
def test_filter_uniform_is_preserved_including_borders(kind):
    cfg = small_cfg(mx=10, my=6, filter_kind=kind, radius=3.0, sigma=1.5)
    Phi = O.filter(cfg, np.full((cfg.mx, cfg.my), 0.37))
    assert np.max(np.abs(Phi - 0.37)) < 1e-15


@pytest.mark.parametrize("kind,radius,sigma,norm,u,s", [
    (0, 4.0, 0.0, 1, 2, 2), (0, 3.3, 0.0, 0, 2, 2), (1, 5.0, 2.0, 1, 2, 2),
    (0, 4.0, 0.0, 1, 2, 4), (0, 3.0, 0.0, 1, 3, 2), (1, 6.0, 2.5, 0, 1, 2)])
def test_filter_equals_library_transposed_convolution(kind, radius, sigma, norm, u, s):
    cfg = small_cfg(mx=11, my=9, u=u, s=s, filter_kind=kind, radius=radius, sigma=sigma, normalize=norm)
    C = RNG.random((cfg.mx, cfg.my))
    ref = torch_filter(cfg, torch.from_numpy(C)).numpy()
    assert np.max(np.abs(O.filter(cfg, C) - ref)) < 1e-13


def test_filter_brute_force_noninteger_upsampling():
    # Fig. 4 has 210/36 cells per control pixel; the oracle takes ux = nx/mx as a real
    cfg = O.OracleConfig(mx=5, my=4, nx=12, ny=10, nz=4, z_lo=1, z_hi=3, s=2, radius=3.1)
    C = RNG.random((cfg.mx, cfg.my))
    Phi = O.filter(cfg, C)
    ux, uy = cfg.nx / cfg.mx, cfg.ny / cfg.my
    for p in range(cfg.px):
        for q in range(cfg.py):
            num = den = 0.0
            for a in range(cfg.mx):
                for b in range(cfg.my):
                    w = max(0.0, 1 - math.hypot((p + .5) / 2 - ux * (a + .5), (q + .5) / 2 - uy * (b + .5)) / 3.1)
                    num += w * C[a, b]; den += w
            assert abs(Phi[p, q] - num / den) < 1e-14


def test_gaussian_filter_is_separable():
    cfg = small_cfg(mx=12, my=10, filter_kind=1, radius=5.0, sigma=2.0, normalize=0)
    cx, cy = RNG.random(cfg.mx), RNG.random(cfg.my)
    Phi = O.filter(cfg, np.outer(cx, cy))
    assert np.linalg.matrix_rank(Phi, tol=1e-12) == 1


@pytest.mark.parametrize("kind,norm", [(0, 1), (0, 0), (1, 1)])
def test_filter_transpose_adjoint_identity(kind, norm):
    cfg = small_cfg(mx=9, my=8, filter_kind=kind, radius=3.5, sigma=1.6, normalize=norm)
    v, w = RNG.standard_normal((cfg.mx, cfg.my)), RNG.standard_normal((cfg.px, cfg.py))
    lhs = np.sum(O.filter(cfg, v) * w)
    rhs = np.sum(v * O.filter_T(cfg, w))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


# ------------------------------------------------------------------ projection, Eqs. (3)/(6)
def test_projection_closed_forms(golden):
    assert O.project(np.array([0.5]), 8.0, 0.5)[0] == 0.5                       # rho(eta) = 1/2
    assert abs(O.project(np.array([0.5 + 1 / 8]), 8.0, 0.5)[0] - golden["rho_t_plus1"]) < 1e-15
    assert abs(O.project(np.array([-2 / 16]), 16.0, 0.0)[0] - golden["rho_t_minus2"]) < 1e-16
    Phi = np.linspace(-1, 2, 1001)
    rho = O.project(Phi, 64.0, 0.5)
    assert rho.min() >= 0 and rho.max() <= 1 and np.all(np.diff(rho) >= 0)
    assert rho[0] == 0.0 and rho[-1] == 1.0                                     # saturated, beta*delta = 96
    # symmetry rho(eta+x) + rho(eta-x) = 1
    x = RNG.random(50)
    assert np.max(np.abs(O.project(0.5 + x, 7.0, 0.5) + O.project(0.5 - x, 7.0, 0.5) - 1)) < 1e-15


def test_projection_derivative_is_analytic_sech2(golden):
    one = np.ones(1)
    assert abs(O.project_T(np.array([0.5 + 1 / 8]), 8.0, 0.5, one)[0] - golden["drho_dphi_t1_b8"]) < 1e-14
    # stable algebraic form 2 beta t/(1+t)^2, t = exp(-2|x|), in extended precision
    Phi = np.linspace(0.0, 1.0, 201)
    for beta in (4.0, 64.0, 300.0):
        x = np.abs(beta * (Phi.astype(np.longdouble) - 0.5))
        t = np.exp(-2 * x)
        ref = 2 * beta * t / (1 + t) ** 2
        got = O.project_T(Phi, beta, 0.5, np.ones_like(Phi))
        assert np.max(np.abs(got - ref) / ref) < 1e-12
    # and against central differences of the forward
    h = 1e-6
    fd = (O.project(Phi + h, 8.0, 0.5) - O.project(Phi - h, 8.0, 0.5)) / (2 * h)
    assert np.max(np.abs(fd - O.project_T(Phi, 8.0, 0.5, np.ones_like(Phi)))) < 1e-8


def test_mixing_rule(golden):
    cfg = small_cfg()
    e, r = O.mix(cfg, np.array([0.0, 1.0, 0.5, 0.25]))
    assert e[0] == golden["eps_sio2"] and e[1] == golden["eps_si"]
    assert abs(e[2] - golden["half_arithmetic"]) < 1e-15 and abs(e[3] - golden["quarter_arithmetic"]) < 1e-15
    assert np.max(np.abs(r * e - 1)) < 1e-15
    # transpose: d/d rho of sum(a*e + b*r)
    rho = RNG.random(20); a = RNG.standard_normal(20); b = RNG.standard_normal(20)
    e, r = O.mix(cfg, rho)
    got = O.mix_T(cfg, e, a, b, np.zeros(20))
    de = golden["eps_si"] - golden["eps_sio2"]
    assert np.max(np.abs(got - de * (a - b / e ** 2))) < 1e-14


# ------------------------------------------------------------------ averages, Eq. (8)
@pytest.mark.parametrize("s", [2, 4])
def test_average_of_step_masks_gives_fill_fractions(s):
    cfg = small_cfg(mx=4, my=4, u=2, s=s)
    for edge in range(cfg.px + 1):           # vertical step: rho = 1 for p < edge
        f = np.zeros((cfg.px, cfg.py)); f[:edge] = 1.0
        for comp in range(3):
            out = O.average(cfg, f, comp)
            sh = s // 2 if comp == 0 else 0
            for i in range(cfg.nx):
                lo, hi = s * i + sh, s * i + sh + s          # footprint [lo,hi) in pixels
                cnt = sum(1 for p in range(lo, hi) if min(p, cfg.px - 1) < edge)
                assert np.all(np.abs(out[i] - cnt / s) < 1e-15), (edge, comp, i)
    f = np.zeros((cfg.px, cfg.py)); f[:, :3] = 1.0          # horizontal step
    out = O.average(cfg, f, 1)                               # E_y footprint: q in [s j + s/2, ...)
    j0 = [sum(1 for q in range(s * j + s // 2, s * j + s // 2 + s) if min(q, cfg.py - 1) < 3) / s for j in range(cfg.ny)]
    assert np.max(np.abs(out - np.array(j0)[None, :])) < 1e-15


@pytest.mark.parametrize("s", [2, 4])
def test_average_equals_library_avg_pool_on_shifted_mask(s):
    cfg = small_cfg(mx=5, my=6, s=s)
    f = RNG.random((cfg.px, cfg.py))
    for comp in range(3):
        ref = torch_average(cfg, torch.from_numpy(f), comp).numpy()
        assert np.max(np.abs(O.average(cfg, f, comp) - ref)) < 1e-15


def test_average_transpose_adjoint_identity():
    cfg = small_cfg(mx=5, my=4, s=4)
    for comp in range(3):
        v, w = RNG.standard_normal((cfg.px, cfg.py)), RNG.standard_normal((cfg.nx, cfg.ny))
        lhs, rhs = np.sum(O.average(cfg, v, comp) * w), np.sum(v * O.average_T(cfg, w, comp))
        assert abs(lhs - rhs) < 1e-13 * abs(lhs)
        # mass conservation: every cell spreads exactly its value
        assert abs(O.average_T(cfg, w, comp).sum() - w.sum()) < 1e-12


# ------------------------------------------------------------------ Sobel normals
def test_sobel_ramps_and_library_conv():
    cfg = small_cfg(mx=6, my=5)
    i, j = np.meshgrid(np.arange(cfg.nx), np.arange(cfg.ny), indexing="ij")
    gx, gy = O.sobel(cfg, 0.3 * i - 0.7 * j + 2.0)
    assert np.max(np.abs(gx[1:-1, :] - 0.3)) < 1e-14 and np.max(np.abs(gy[:, 1:-1] + 0.7)) < 1e-14
    assert np.max(np.abs(gx[0, :] - 0.15)) < 1e-14            # replicate border halves the slope
    D = RNG.random((cfg.nx, cfg.ny))
    rx, ry = torch_sobel(torch.from_numpy(D))
    gx, gy = O.sobel(cfg, D)
    assert np.max(np.abs(gx - rx.numpy())) < 1e-15 and np.max(np.abs(gy - ry.numpy())) < 1e-15
    gx, gy = O.sobel(cfg, np.full((cfg.nx, cfg.ny), 0.8))
    assert np.max(np.abs(gx)) < 1e-16 and np.max(np.abs(gy)) < 1e-16


def test_sobel_transpose_adjoint_identity():
    cfg = small_cfg(mx=4, my=5)
    D, a, b = (RNG.standard_normal((cfg.nx, cfg.ny)) for _ in range(3))
    gx, gy = O.sobel(cfg, D)
    lhs, rhs = np.sum(gx * a + gy * b), np.sum(D * O.sobel_T(cfg, a, b))
    assert abs(lhs - rhs) < 1e-13 * abs(lhs)


# ------------------------------------------------------------------ Eq. (7)
def _stages_from_mask(cfg, rho):
    e, r = O.mix(cfg, rho)
    out = []
    for c in range(3):
        A, H, D = O.average(cfg, e, c), O.average(cfg, r, c), O.average(cfg, rho, c)
        gx, gy = O.sobel(cfg, D) if c < 2 else (None, None)
        out.append(O.eq7(cfg, c, A, H, gx, gy))
    return out


def test_eq7_vertical_interface_is_textbook_subpixel_smoothing(golden):
    # binary mask with an x-normal interface through the middle of a cell
    cfg = small_cfg(mx=6, my=6, s=2)
    rho = np.zeros((cfg.px, cfg.py)); rho[:11] = 1.0          # edge at x = 5.5 cells
    (exx, n2x), (eyy, n2y), (ezz, _) = _stages_from_mask(cfg, rho)
    # E_z / E_y cell i=5 covers x in [5,6]: half filled
    assert np.max(np.abs(ezz[5] - golden["half_arithmetic"])) < 1e-12          # n_z = 0 -> <eps>
    assert np.max(np.abs(eyy[5] - golden["half_arithmetic"])) < 1e-9           # n_y = 0 -> <eps>
    assert np.max(np.abs(n2y)) < 1e-20
    # E_x cells are shifted by half a cell: cell i=4 covers [4.5,5.5] (full), i=5 covers [5.5,6.5] (empty)
    assert np.max(np.abs(exx[4] - golden["eps_si"])) < 1e-12 and np.max(np.abs(exx[5] - golden["eps_sio2"])) < 1e-12
    rho = np.zeros((cfg.px, cfg.py)); rho[:12] = 1.0          # edge at x = 6: E_x cell i=5 = [5.5,6.5] half filled
    (exx, n2x), _, _ = _stages_from_mask(cfg, rho)
    assert np.max(np.abs(n2x[5] - 1)) < 1e-10                                  # normal along x
    assert np.max(np.abs(exx[5] - golden["half_harmonic"])) < 1e-9             # n_x = 1 -> 1/<1/eps>
    cfg4 = small_cfg(mx=6, my=6, s=4)
    rho = np.zeros((cfg4.px, cfg4.py)); rho[:, :21] = 1.0     # y-normal edge at y = 5.25: fill 1/4 of E_z cell j=5
    (exx, _), (eyy, n2y), (ezz, _) = _stages_from_mask(cfg4, rho)
    assert np.max(np.abs(ezz[:, 5] - golden["quarter_arithmetic"])) < 1e-12
    assert np.max(np.abs(exx[:, 5] - golden["quarter_arithmetic"])) < 1e-9     # tangential component
    # E_y cell j=4 covers [4.5,5.5]: fill 3/4; j=5 covers [5.5,6.5]: empty
    assert np.max(np.abs(eyy[:, 4] - 1 / (0.75 / golden["eps_si"] + 0.25 / golden["eps_sio2"]))) < 1e-9


def test_eq7_diagonal_interface_has_equal_normal_components():
    cfg = small_cfg(mx=8, my=8, s=2)
    p, q = np.meshgrid(np.arange(cfg.px), np.arange(cfg.py), indexing="ij")
    rho = (p + q < cfg.px).astype(float)
    D = O.average(cfg, rho, 2)
    gx, gy = O.sobel(cfg, D)
    assert np.max(np.abs(gx - gy)[2:-2, 2:-2]) < 1e-15
    _, n2 = O.eq7(cfg, 0, D + 1, D + 1, gx, gy)
    edge = np.abs(gx) > 0.1
    assert edge[2:-2, 2:-2].any() and np.max(np.abs(n2[2:-2, 2:-2][edge[2:-2, 2:-2]] - 0.5)) < 1e-10


def test_eq7_bounded_by_harmonic_and_arithmetic_means():
    cfg = small_cfg(mx=10, my=10)
    rho = RNG.random((cfg.px, cfg.py))
    e, r = O.mix(cfg, rho)
    for c in range(2):
        A, H, D = O.average(cfg, e, c), O.average(cfg, r, c), O.average(cfg, rho, c)
        gx, gy = O.sobel(cfg, D)
        eps, n2 = O.eq7(cfg, c, A, H, gx, gy)
        assert np.all(n2 >= 0) and np.all(n2 <= 1)
        assert np.all(eps <= A + 1e-12) and np.all(eps >= 1 / H - 1e-12)
        assert np.all(eps >= cfg.eps_clad) and np.all(eps <= cfg.eps_core)


def test_eq7_transpose_against_finite_differences():
    cfg = small_cfg(mx=3, my=3)
    n = (cfg.nx, cfg.ny)
    A, H = 2 + 5 * RNG.random(n), 0.1 + 0.3 * RNG.random(n)
    gx, gy = 0.2 * RNG.standard_normal(n), 0.2 * RNG.standard_normal(n)
    w = RNG.standard_normal(n)
    for comp in (0, 1):
        Ab, Hb, gxb, gyb = O.eq7_T(cfg, comp, A, H, gx, gy, w)
        f = lambda A, H, gx, gy: np.sum(w * O.eq7(cfg, comp, A, H, gx, gy)[0])
        h = 1e-6
        for k, (arr, bar) in enumerate(((A, Ab), (H, Hb), (gx, gxb), (gy, gyb))):
            for idx in [(0, 0), (2, 3), (5, 1)]:
                args = [A.copy(), H.copy(), gx.copy(), gy.copy()]
                args[k][idx] += h; fp = f(*args)
                args[k][idx] -= 2 * h; fm = f(*args)
                assert abs((fp - fm) / (2 * h) - bar[idx]) < 1e-7 * max(1, abs(bar[idx]))


# ------------------------------------------------------------------ z-extrusion
def test_z_weights_of_the_config_slabs():
    for nz, lo, hi, first in ((16, 6.25, 9.75, 6), (64, 28.25, 35.75, 28), (32, 14.25, 17.75, 14)):
        cfg = small_cfg(nz=nz, z_lo=lo, z_hi=hi)
        wxy, wz = O.zweights(cfg)
        n = int(hi - lo + 0.5)
        exp_xy = np.zeros(nz); exp_xy[first:first + n] = 1; exp_xy[first] = exp_xy[first + n - 1] = 0.75
        exp_z = np.zeros(nz); exp_z[first - 1:first + n] = 1; exp_z[first - 1] = exp_z[first + n - 1] = 0.25
        assert np.array_equal(wxy, exp_xy) and np.array_equal(wz, exp_z)
        assert abs(wxy.sum() - (hi - lo)) < 1e-15 and abs(wz.sum() - (hi - lo)) < 1e-15


def test_extrude_uniform_layer(golden):
    cfg = small_cfg(mx=2, my=2, nz=16, z_lo=6.25, z_hi=9.75)
    eps = O.extrude(cfg, np.full((3, cfg.nx, cfg.ny), golden["uniform_c0_eq3"]))
    assert np.all(eps[:, :, :, :5] == golden["eps_sio2"]) and np.all(eps[:, :, :, 10:] == golden["eps_sio2"])
    assert np.max(np.abs(eps[:2, :, :, 7:9] - golden["uniform_c0_eq3"])) < 1e-15
    assert np.max(np.abs(eps[:2, :, :, [6, 9]] - golden["face_xy_w075"])) < 1e-15
    assert np.max(np.abs(eps[2, :, :, 6:9] - golden["uniform_c0_eq3"])) < 1e-14
    assert np.max(np.abs(eps[2, :, :, [5, 9]] - golden["face_z_w025"])) < 1e-14
    assert np.all(eps[:2, :, :, 5] == golden["eps_sio2"])


def test_extrude_transpose_against_finite_differences():
    cfg = small_cfg(mx=2, my=2, nz=8, z_lo=2.25, z_hi=5.75)
    e2 = 2.5 + 8 * RNG.random((3, cfg.nx, cfg.ny))
    w = RNG.standard_normal((3, cfg.nx, cfg.ny, cfg.nz))
    bar = O.extrude_T(cfg, e2, w)
    h = 1e-6
    for idx in [(0, 0, 0), (1, 2, 3), (2, 1, 1), (2, 3, 0)]:
        ep, em = e2.copy(), e2.copy(); ep[idx] += h; em[idx] -= h
        fd = np.sum(w * (O.extrude(cfg, ep) - O.extrude(cfg, em))) / (2 * h)
        assert abs(fd - bar[idx]) < 1e-8 * max(1, abs(bar[idx]))
