"""Shared pieces of the GPU parity tests: run the CUDA path (through the C ABI binding) and
the float64 oracle on the same seeded inputs and compare.  Tolerances are BASELINE.json's:
relative 1e-5 on eps (element-wise; eps >= eps_clad > 0) and 1e-4 on dF/dC (S14: max-norm
and 2-norm relative error; element-wise is meaningless at sign changes)."""
from __future__ import annotations

import numpy as np
import torch

import oracle as O
from helpers import rel_inf, rel_l2
from paper_2505_03352_b200 import binding as B

TOL_EPS = 1e-5
TOL_GRAD = 1e-4


def oracle_cfg(cfg: B.Config) -> O.OracleConfig:
    return O.OracleConfig(mx=cfg.mx, my=cfg.my, nx=cfg.nx, ny=cfg.ny, nz=cfg.nz, z_lo=cfg.z_lo, z_hi=cfg.z_hi,
                          s=cfg.subpixel, filter_kind=cfg.filter_kind, radius=cfg.filter_radius,
                          sigma=cfg.filter_sigma, normalize=cfg.filter_normalize, eta=cfg.eta,
                          eps_core=cfg.eps_core, eps_clad=cfg.eps_clad, delta=cfg.normal_delta,
                          morph_diam=cfg.morph_diameter, morph_alpha=cfg.morph_alpha)


def rand_C(cfg: B.Config, seed: int) -> np.ndarray:
    return np.random.default_rng(seed).random((cfg.batch, cfg.mx, cfg.my), dtype=np.float32)


def rand_fields(cfg: B.Config, n_pairs: int, seed: int):
    """n_pairs x (E_F, E_A), complex64 [B,3,nx,ny,nz], i.i.d. N(0,1) re and im."""
    rng = np.random.default_rng([seed, 7])
    shape = (cfg.batch, 3, cfg.nx, cfg.ny, cfg.nz)

    def one():
        a = np.empty(shape, np.complex64)
        rng.standard_normal(out=a.view(np.float32).reshape(-1), dtype=np.float32)
        return a
    return [one() for _ in range(n_pairs)], [one() for _ in range(n_pairs)]


def dev(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(a).cuda()


def max_rel(a: np.ndarray, ref: np.ndarray) -> float:
    return float(np.max(np.abs(a - ref) / np.abs(ref)))


def check_forward(cfg: B.Config, C: np.ndarray, beta: float, plan: B.Plan | None = None, tol=TOL_EPS):
    plan = plan or B.Plan(cfg)
    eps = plan.eps_forward(dev(C), beta).cpu().numpy().astype(np.float64)
    oc = oracle_cfg(cfg)
    worst = 0.0
    for b in range(cfg.batch):
        ref = O.forward(oc, C[b], beta)
        worst = max(worst, max_rel(eps[b], ref))
    assert worst < tol, f"eps max relative error {worst:.3e} >= {tol}"
    return worst


def check_vjp(cfg: B.Config, C: np.ndarray, beta: float, EF, EA, plan: B.Plan | None = None, tol=TOL_GRAD):
    plan = plan or B.Plan(cfg)
    g = plan.eps_vjp(dev(C), beta, [dev(f) for f in EF], [dev(f) for f in EA]).cpu().numpy().astype(np.float64)
    oc = oracle_cfg(cfg)
    worst = 0.0
    for b in range(cfg.batch):
        ref = O.vjp(oc, C[b], beta, [f[b] for f in EF], [f[b] for f in EA])
        worst = max(worst, rel_inf(g[b], ref), rel_l2(g[b], ref))
    assert worst < tol, f"dF/dC relative error {worst:.3e} >= {tol}"
    return worst


def check_guard_bands(cfg: B.Config, C, EF, EA, beta: float, guard: int = 4096):
    """Outputs and workspace between guard bands of `guard` bytes (a multiple of 256: alignment kept) filled with a sentinel:
    every kind of call must leave the bands untouched and give the bits it gives with plain buffers.  The sentinel byte 0xFF
    makes every float a NaN, and the workspace is refilled with it before each call: a kernel that read workspace memory no
    kernel of the same call had written (the initcheck case) would propagate NaNs into the result."""
    SENT = 0xFF
    n_pairs = len(EF)
    plan = B.Plan(cfg)
    eps0, g0 = plan.eps_forward_vjp(C, beta, EF, EA)
    gb0, db0 = plan.eps_vjp_beta(C, beta, EF, EA)
    u0 = plan.unbinarity(C, beta)

    def banded(nbytes):
        raw = torch.full((nbytes + 2 * guard,), SENT, dtype=torch.uint8, device="cuda")
        return raw, raw[guard:guard + nbytes]

    def intact(raw, nbytes):
        return bool((raw[:guard] == SENT).all()) and bool((raw[guard + nbytes:] == SENT).all())

    nws = B.lib().epsgrad_workspace_bytes(plan._h)
    ws_raw, ws = banded(nws)
    B._check(B.lib().epsgrad_plan_set_workspace(plan._h, ws.data_ptr(), nws), "epsgrad_plan_set_workspace")
    e_raw, e_mid = banded(eps0.numel() * 4)
    g_raw, g_mid = banded(g0.numel() * 4)
    d_raw, d_mid = banded(db0.numel() * 4)
    eps = e_mid.view(torch.float32).view(eps0.shape)
    g = g_mid.view(torch.float32).view(g0.shape)
    db = d_mid.view(torch.float32).view(db0.shape)
    plan.eps_forward_vjp(C, beta, EF, EA, eps_out=eps, grad_out=g)
    torch.cuda.synchronize()
    assert torch.equal(eps, eps0) and torch.equal(g, g0)
    eps.zero_(); g.zero_(); ws.fill_(SENT)
    plan.eps_forward(C, beta, out=eps)
    ws.fill_(SENT)
    plan.eps_vjp(C, beta, EF, EA, out=g)
    assert torch.equal(eps, eps0) and torch.equal(g, g0)
    g.zero_(); ws.fill_(SENT)
    B._check(B.lib().eps_vjp_beta(plan._h, C.data_ptr(), beta, n_pairs, *plan._fields(EF, EA), g.data_ptr(), db.data_ptr(),
                                  plan._stream()), "eps_vjp_beta")
    ws.fill_(SENT)
    u = plan.unbinarity(C, beta)
    torch.cuda.synchronize()
    assert torch.equal(g, g0) and torch.equal(db, db0) and torch.equal(u, u0)
    for raw, n in ((ws_raw, nws), (e_raw, eps0.numel() * 4), (g_raw, g0.numel() * 4), (d_raw, db0.numel() * 4)):
        assert intact(raw, n), cfg
    plan._ws = ws_raw                                          # keep the banded workspace alive as long as the plan
