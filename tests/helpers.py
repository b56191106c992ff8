"""Test-side helpers: oracle config from a workload, and a float64 torch restatement
of the chain built from LIBRARY primitives (conv_transpose2d, avg_pool2d, conv2d,
autograd) -- the paper's own route to the VJP -- used as a second
opinion on the hand-written oracle.  Not imported by the product."""
from __future__ import annotations

import math

import numpy as np
import torch
import torch.nn.functional as F

import oracle as O


def cfg_of(w, **over) -> O.OracleConfig:
    kw = dict(mx=w.mx, my=w.my, nx=w.nx, ny=w.ny, nz=w.nz, z_lo=w.z_lo, z_hi=w.z_hi, s=w.subpixel,
              filter_kind=w.filter_kind, radius=w.radius, sigma=w.sigma, eta=w.eta,
              eps_core=w.eps_core, eps_clad=w.eps_clad, delta=w.normal_delta,
              morph_diam=getattr(w, "morph_diameter", 0.0), morph_alpha=getattr(w, "morph_alpha", 20.0))
    kw.update(over)
    return O.OracleConfig(**kw)


def small_cfg(mx=8, my=8, u=2, s=2, nz=8, z_lo=2.25, z_hi=5.75, **kw) -> O.OracleConfig:
    return O.OracleConfig(mx=mx, my=my, nx=u * mx, ny=u * my, nz=nz, z_lo=z_lo, z_hi=z_hi, s=s, **kw)


def basis_torch(cfg, dx, dy):
    if cfg.filter_kind == 0:
        return torch.clamp(1.0 - torch.sqrt(dx * dx + dy * dy) / cfg.radius, min=0.0)
    inside = (dx.abs() <= cfg.radius) & (dy.abs() <= cfg.radius)
    return torch.exp(-(dx * dx + dy * dy) / (2 * cfg.sigma ** 2)) * inside


def torch_filter(cfg, C):
    """Eq. (2) as a fractionally-strided (transposed) convolution, float64."""
    u = cfg.nx // cfg.mx
    assert u * cfg.mx == cfg.nx and u * cfg.my == cfg.ny
    s, m = cfg.s, u * cfg.s
    pad = int(math.ceil(s * cfg.radius))
    kt = 2 * pad + m
    d = (torch.arange(kt, dtype=torch.float64) - pad) / s + 0.5 / s - u / 2.0
    b = basis_torch(cfg, d[:, None], d[None, :])[None, None]
    num = F.conv_transpose2d(C[None, None], b, stride=m, padding=pad)[0, 0]
    if not cfg.normalize:
        return num
    den = F.conv_transpose2d(torch.ones_like(C)[None, None], b, stride=m, padding=pad)[0, 0]
    return num / den


def torch_average(cfg, f, comp):
    s = cfg.s
    sp, sq = (s // 2 if comp == 0 else 0), (s // 2 if comp == 1 else 0)
    fp = F.pad(f[None, None], (0, sq, 0, sp), mode="replicate")[:, :, sp:, sq:]
    return F.avg_pool2d(fp, s)[0, 0]


def torch_sobel(D):
    kx = torch.tensor([[-1, -2, -1], [0, 0, 0], [1, 2, 1]], dtype=torch.float64) / 8.0   # d/di
    Dp = F.pad(D[None, None], (1, 1, 1, 1), mode="replicate")
    return F.conv2d(Dp, kx[None, None])[0, 0], F.conv2d(Dp, kx.t().contiguous()[None, None])[0, 0]


def torch_morph(cfg, x, erode):
    """Eqs. (4)-(5) from library primitives: unfold the mask into disk neighbourhoods (outside = -inf, i.e. weight 0),
    torch.logsumexp, minus log of the in-range count (unit-sum kernel, S18)."""
    rp = 0.5 * cfg.morph_diam * cfg.s
    R = int(math.floor(rp))
    d = torch.arange(-R, R + 1, dtype=torch.float64)
    disk = ((d[:, None] ** 2 + d[None, :] ** 2) <= rp * rp).reshape(-1)
    z = cfg.morph_alpha * ((1.0 - x) if erode else x)
    zp = F.pad(z[None, None], (R, R, R, R), value=float("-inf"))
    cols = F.unfold(zp, 2 * R + 1)[0]                                  # [(2R+1)^2, px*py]
    cols = cols[disk]
    n = torch.isfinite(cols).sum(0).to(torch.float64)
    l = ((torch.logsumexp(cols, 0) - torch.log(n)) / cfg.morph_alpha).reshape(x.shape)
    return 1.0 - l if erode else l


def torch_eps2d(cfg, C, beta):
    Phi = torch_filter(cfg, C)
    rho = 0.5 * (1 + torch.tanh(beta * (Phi - cfg.eta)))
    if cfg.morph_diam > 0:                                             # P:L64-74 (S17): dilate, erode, erode, dilate, Eq. (6)
        for erode in (False, True, True, False):
            rho = torch_morph(cfg, rho, erode)
        rho = 0.5 * (1 + torch.tanh(beta * (rho - 0.5)))
    e = rho * cfg.eps_core + (1 - rho) * cfg.eps_clad
    r = 1.0 / e
    out = []
    for c in range(3):
        A, H, D = (torch_average(cfg, f, c) for f in (e, r, rho))
        if c == 2:
            out.append(A)
            continue
        gx, gy = torch_sobel(D)
        gc = gx if c == 0 else gy
        n2 = gc * gc / (gx * gx + gy * gy + cfg.delta)
        out.append(1.0 / (n2 * H + (1 - n2) / A))
    return torch.stack(out)


def torch_chain(cfg, C, beta):
    """eps [3,nx,ny,nz] float64 torch tensor, differentiable in C."""
    e2 = torch_eps2d(cfg, C, beta)
    k = torch.arange(cfg.nz, dtype=torch.float64)
    wxy = torch.clamp(torch.clamp(k + 1, max=cfg.z_hi) - torch.clamp(k, min=cfg.z_lo), min=0)
    wz = torch.clamp(torch.clamp(k + 1.5, max=cfg.z_hi) - torch.clamp(k + 0.5, min=cfg.z_lo), min=0)
    exy = cfg.eps_clad + wxy * (e2[:2, :, :, None] - cfg.eps_clad)
    ezz = 1.0 / (wz / e2[2:, :, :, None] + (1 - wz) / cfg.eps_clad)
    return torch.cat([exy, ezz])


def rel_inf(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(np.asarray(b).ravel()))
