"""Pins of the oracle's morphological filters (Eqs. (4)-(5)) and of the chain with them switched on
(dilate, erode, erode, dilate, then Eq. (6); readings S17, S18 in DESIGN.md): closed forms, the alpha -> infinity
and alpha -> 0 limits against scipy.ndimage, the duality of Eqs. (4) and (5), a library (unfold + logsumexp +
autograd) restatement, the adjoint identity and central finite differences."""
import numpy as np
import pytest
import scipy.ndimage as ndi
import torch

import oracle as O
from helpers import small_cfg, torch_chain, torch_morph


def disk(cfg):
    rp = 0.5 * cfg.morph_diam * cfg.s
    R = int(np.floor(rp))
    d = np.arange(-R, R + 1)
    return (d[:, None] ** 2 + d[None, :] ** 2) <= rp * rp


def test_disk_pixel_counts():
    # lattice points in a circle of radius r: 13 (r = 2), 49 (r = 4), 197 (r = 8): d = 2, 4, 8 cells at s = 2
    for d, n in ((2.0, 13), (4.0, 49), (8.0, 197)):
        assert int(disk(small_cfg(morph_diam=d)).sum()) == n


@pytest.mark.parametrize("erode", [False, True])
def test_constant_field_is_a_fixed_point_everywhere(erode):
    cfg = small_cfg(mx=6, my=7, morph_diam=3.0)
    for c0 in (0.0, 0.3, 1.0):
        y = O.morph(cfg, np.full((cfg.px, cfg.py), c0), erode)
        assert np.max(np.abs(y - c0)) < 1e-13          # also at the borders: unit-sum kernel over in-range pixels


def test_erode_is_the_dual_of_dilate():
    cfg = small_cfg(mx=6, my=5, morph_diam=4.0)
    x = np.random.default_rng(0).random((cfg.px, cfg.py))
    assert np.max(np.abs(O.morph(cfg, x, True) - (1.0 - O.morph(cfg, 1.0 - x, False)))) < 1e-13


def test_large_alpha_tends_to_max_and_min_filters():
    # (1/alpha) log mean exp(alpha x) lies in [max - log(N)/alpha, max]
    cfg = small_cfg(mx=8, my=6, morph_diam=4.0, morph_alpha=400.0)
    x = np.random.default_rng(1).random((cfg.px, cfg.py))
    fp = disk(cfg)
    mx = ndi.maximum_filter(x, footprint=fp, mode="constant", cval=-np.inf)
    mn = ndi.minimum_filter(x, footprint=fp, mode="constant", cval=np.inf)
    tol = np.log(fp.sum()) / cfg.morph_alpha
    D, E = O.morph(cfg, x, False), O.morph(cfg, x, True)
    assert np.all(D <= mx + 1e-12) and np.all(D >= mx - tol - 1e-12)
    assert np.all(E >= mn - 1e-12) and np.all(E <= mn + tol + 1e-12)


def test_small_alpha_tends_to_the_disk_mean():
    cfg = small_cfg(mx=8, my=6, morph_diam=4.0, morph_alpha=1e-5)
    x = np.random.default_rng(2).random((cfg.px, cfg.py))
    fp = disk(cfg).astype(np.float64)
    mean = ndi.convolve(x, fp, mode="constant") / ndi.convolve(np.ones_like(x), fp, mode="constant")
    for erode in (False, True):
        assert np.max(np.abs(O.morph(cfg, x, erode) - mean)) < 1e-5      # second-order term alpha var / 2


def test_jensen_ordering_and_range():
    # unit-sum kernel: disk mean <= dilate <= disk max and disk min <= erode <= disk mean (Jensen)
    cfg = small_cfg(mx=8, my=8, morph_diam=3.0)
    x = np.random.default_rng(3).random((cfg.px, cfg.py))
    fp = disk(cfg)
    mean = ndi.convolve(x, fp.astype(np.float64), mode="constant") / ndi.convolve(np.ones_like(x), fp.astype(np.float64), mode="constant")
    mx = ndi.maximum_filter(x, footprint=fp, mode="constant", cval=-np.inf)
    mn = ndi.minimum_filter(x, footprint=fp, mode="constant", cval=np.inf)
    D, E = O.morph(cfg, x, False), O.morph(cfg, x, True)
    assert np.all(mean <= D + 1e-12) and np.all(D <= mx + 1e-12)
    assert np.all(mn <= E + 1e-12) and np.all(E <= mean + 1e-12)


@pytest.mark.parametrize("erode", [False, True])
def test_matches_library_logsumexp_and_its_autograd(erode):
    cfg = small_cfg(mx=7, my=6, morph_diam=4.0)
    rng = np.random.default_rng(4)
    x = rng.random((cfg.px, cfg.py))
    ybar = rng.standard_normal((cfg.px, cfg.py))
    xt = torch.tensor(x, requires_grad=True)
    yt = torch_morph(cfg, xt, erode)
    assert np.max(np.abs(O.morph(cfg, x, erode) - yt.detach().numpy())) < 1e-12
    (yt * torch.tensor(ybar)).sum().backward()
    g = O.morph_T(cfg, x, erode, ybar)
    assert np.max(np.abs(g - xt.grad.numpy())) < 1e-12 * max(1.0, np.abs(g).max())


@pytest.mark.parametrize("erode", [False, True])
def test_transpose_matches_central_differences(erode):
    cfg = small_cfg(mx=4, my=4, morph_diam=3.0)
    rng = np.random.default_rng(5)
    x = rng.random((cfg.px, cfg.py))
    w = rng.standard_normal((cfg.px, cfg.py))
    g = O.morph_T(cfg, x, erode, w)
    h = 1e-6
    for (p, q) in [(0, 0), (3, 5), (cfg.px - 1, cfg.py - 2), (7, 7)]:
        xp, xm = x.copy(), x.copy()
        xp[p, q] += h; xm[p, q] -= h
        fd = np.sum(w * (O.morph(cfg, xp, erode) - O.morph(cfg, xm, erode))) / (2 * h)
        assert abs(fd - g[p, q]) < 1e-7 * max(1.0, abs(fd))


def test_chain_with_filters_uniform_control_and_bounds():
    cfg = small_cfg(mx=8, my=8, nz=8, morph_diam=3.0, radius=3.0)
    beta = 6.0
    for c0 in (0.2, 0.5, 0.9):
        e2 = O.forward(cfg, np.full((cfg.mx, cfg.my), c0, dtype=np.float32), beta, want_eps2d=True)[1]
        rho0 = 0.5 * (1 + np.tanh(beta * (np.float64(np.float32(c0)) - 0.5)))
        rho = 0.5 * (1 + np.tanh(beta * (rho0 - 0.5)))                     # the filters keep a uniform mask; Eq. (6) follows
        assert np.max(np.abs(e2 - (rho * cfg.eps_core + (1 - rho) * cfg.eps_clad))) < 1e-12
    eps = O.forward(cfg, np.random.default_rng(6).random((cfg.mx, cfg.my)).astype(np.float32), 40.0)
    assert eps.min() >= cfg.eps_clad - 1e-12 and eps.max() <= cfg.eps_core + 1e-12


def test_chain_with_filters_matches_library_autograd_and_finite_differences():
    cfg = small_cfg(mx=6, my=5, nz=8, morph_diam=3.0, radius=3.0)
    rng = np.random.default_rng(7)
    C = rng.random((cfg.mx, cfg.my)).astype(np.float32)
    w = rng.standard_normal((3, cfg.nx, cfg.ny, cfg.nz))
    beta = 5.0
    Ct = torch.tensor(C.astype(np.float64), requires_grad=True)
    eps_t = torch_chain(cfg, Ct, beta)
    eps = O.forward(cfg, C, beta)
    assert np.max(np.abs(eps - eps_t.detach().numpy()) / eps) < 1e-12
    (eps_t * torch.tensor(w)).sum().backward()
    g = O.vjp_real(cfg, C, beta, w)
    assert np.max(np.abs(g - Ct.grad.numpy())) < 1e-10 * np.abs(g).max()
    # central differences of F(C) = sum w eps(C) in float32-representable steps
    h = np.float32(2.0 ** -10)
    for (a, b) in [(0, 0), (2, 3), (5, 4)]:
        Cp, Cm = C.copy(), C.copy()
        Cp[a, b] += h; Cm[a, b] -= h
        fd = np.sum(w * (O.forward(cfg, Cp, beta) - O.forward(cfg, Cm, beta))) / (float(Cp[a, b]) - float(Cm[a, b]))
        assert abs(fd - g[a, b]) < 2e-5 * np.abs(g).max()
