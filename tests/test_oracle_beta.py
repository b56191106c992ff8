"""Pins of the oracle's beta-related pieces (NEXT-2): d eps_hat / d beta, the unbinarity u(beta) (reading S20)
and the beta schedule, Eqs. (14)-(15)."""
import math

import numpy as np
import pytest
import torch

import oracle as O
from helpers import small_cfg, torch_chain


@pytest.mark.parametrize("morph", [0.0, 3.0])
def test_dbeta_matches_central_differences_and_autograd(morph):
    cfg = small_cfg(mx=6, my=5, nz=8, radius=3.0, morph_diam=morph)
    rng = np.random.default_rng(11)
    C = rng.random((cfg.mx, cfg.my)).astype(np.float32)
    w = rng.standard_normal((3, cfg.nx, cfg.ny, cfg.nz))
    beta = 5.0
    g, db = O.vjp_real_beta(cfg, C, beta, w)
    assert np.array_equal(g, O.vjp_real(cfg, C, beta, w))            # the C gradient is untouched
    h = 1e-5
    fd = np.sum(w * (O.forward(cfg, C, beta + h) - O.forward(cfg, C, beta - h))) / (2 * h)
    assert abs(fd - db) < 1e-7 * max(1.0, abs(fd))
    bt = torch.tensor(beta, dtype=torch.float64, requires_grad=True)    # the library chain, differentiated in beta by autograd
    (torch_chain(cfg, torch.tensor(C.astype(np.float64)), bt) * torch.tensor(w)).sum().backward()
    assert abs(float(bt.grad) - db) < 1e-10 * max(1.0, abs(db))


def test_dbeta_from_field_pairs_is_the_real_cotangent_case():
    cfg = small_cfg(mx=5, my=6, nz=8, radius=3.0)
    rng = np.random.default_rng(12)
    C = rng.random((cfg.mx, cfg.my)).astype(np.float32)
    shape = (3, cfg.nx, cfg.ny, cfg.nz)
    EF = [(rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64) for _ in range(2)]
    EA = [(rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64) for _ in range(2)]
    g, db = O.vjp_beta(cfg, C, 7.0, EF, EA)
    G3 = sum(-2.0 * (f.astype(np.complex128) * a.astype(np.complex128)).real for f, a in zip(EF, EA))
    g2, db2 = O.vjp_real_beta(cfg, C, 7.0, G3)
    assert np.allclose(g, g2, rtol=1e-13, atol=0) and abs(db - db2) < 1e-12 * abs(db2)


def test_unbinarity_closed_forms():
    cfg = small_cfg(mx=8, my=8, radius=3.0)
    # uniform C = c0: rho = 1/2 (1 + tanh(beta (c0 - 1/2))) everywhere, u = 4 rho (1 - rho) = sech^2(beta (c0 - 1/2))
    for c0, beta in ((0.5, 9.0), (0.7, 4.0), (0.1, 12.0)):
        u = O.unbinarity(cfg, np.full((cfg.mx, cfg.my), c0, np.float32), beta)
        assert abs(u - 1.0 / math.cosh(beta * (float(np.float32(c0)) - 0.5)) ** 2) < 1e-13
    C = np.random.default_rng(13).random((cfg.mx, cfg.my)).astype(np.float32)
    us = [O.unbinarity(cfg, C, b) for b in (1.0, 4.0, 16.0, 64.0, 1e4)]
    assert all(0.0 <= u <= 1.0 for u in us) and all(a > b for a, b in zip(us, us[1:])) and us[-1] < 1e-2
    # gray pixels are counted on the mask the chain uses: the definition applied to the oracle's own rho
    rho = O.forward_stages(cfg, C, 8.0)["rho"]
    assert abs(O.unbinarity(cfg, C, 8.0) - np.mean(4 * rho * (1 - rho))) < 1e-14


def test_unbinarity_scales_like_one_over_beta_on_a_ramp():
    # a mask that crosses 1/2 linearly: mean sech^2(beta (x - 1/2)) over x in [0,1] = (2/beta) tanh(beta/2): the model
    # u ~ 1/(1 + t beta) behind Eq. (15); checked through project() on a ramp of pixel centres
    n = 4000
    x = (np.arange(n) + 0.5) / n
    for beta in (8.0, 32.0):
        rho = O.project(x, beta, 0.5)
        assert abs(np.mean(4 * rho * (1 - rho)) - 2.0 / beta * math.tanh(beta / 2)) < 1e-6


def test_beta_schedule_eq14():
    bmin, bmax, n = 10.0, 200.0, 100
    assert O.beta_schedule(bmin, bmax, 0, n) == bmin
    assert abs(O.beta_schedule(bmin, bmax, n, n) - bmax) < 1e-12
    b = [O.beta_schedule(bmin, bmax, i, n) for i in range(n + 1)]
    assert all(x < y for x, y in zip(b, b[1:]))
    assert abs(b[50] - (bmin + (bmax - bmin) * (math.exp(0.25) - 1) / (math.e - 1))) < 1e-12


def test_beta_update_eq15_fixed_point():
    # if the mask obeys u = 1/(1 + t* beta), the moving averages converge to t* and to the beta_max at which u = u0
    gamma, u0, tstar = 0.95, 0.01, 0.37
    t, bmax = 1.0, 50.0
    for it in range(2000):
        beta = 10.0 + it * 0.1
        t, bmax = O.beta_update(t, bmax, gamma, 1.0 / (1.0 + tstar * beta), u0, beta)
    assert abs(t - tstar) < 1e-9 and abs(bmax - (1.0 / u0 - 1.0) / tstar) < 1e-6
    t1, b1 = O.beta_update(2.0, 80.0, gamma, 0.2, u0, 16.0)          # one step, by hand
    assert abs(t1 - (0.95 * 2.0 + 0.05 * 4.0 / 16.0)) < 1e-15 and abs(b1 - (0.95 * 80.0 + 0.05 * 99.0 / t1)) < 1e-12


def test_adam_first_step_closed_form_and_library():
    # step 1 from zero moments: Mh = G, Vh = G^2, so C moves by -lr G/(|G| + eps) (Eqs. (10)-(11))
    rng = np.random.default_rng(21)
    C0 = rng.random((7, 9))
    G = rng.standard_normal((7, 9))
    C1, M1, V1 = O.adam_step(C0, np.zeros_like(C0), np.zeros_like(C0), G, 1, lr=1e-3, eps=1e-8)
    assert np.max(np.abs(C1 - (C0 - 1e-3 * G / (np.abs(G) + 1e-8)))) < 1e-15
    assert np.allclose(M1, 0.1 * G, rtol=1e-14) and np.allclose(V1, 0.001 * G * G, rtol=1e-12)
    # 25 steps with fresh gradients against torch.optim.Adam in float64 (same update rule, App. B defaults)
    Ct = torch.tensor(C0.copy(), requires_grad=True)
    opt = torch.optim.Adam([Ct], lr=1e-3, betas=(0.9, 0.999), eps=1e-8)
    C, M, V = C0.copy(), np.zeros_like(C0), np.zeros_like(C0)
    for i in range(1, 26):
        G = rng.standard_normal(C0.shape) * (1.0 + i)
        Ct.grad = torch.tensor(G.copy())
        opt.step()
        C, M, V = O.adam_step(C, M, V, G, i)
        assert np.max(np.abs(C - Ct.detach().numpy())) < 1e-13
