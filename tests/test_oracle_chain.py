"""Pins of the whole oracle chain C -> eps and of its reverse pass (CPU only):
invariants named in BASELINE.json's north_star (uniform C, bounds, mirror symmetry),
the adjoint identity, central finite differences, a float64 library/autograd
restatement (the paper's own route), and the Eq. (1) assembly."""
import numpy as np
import pytest
import torch

import oracle as O
from helpers import cfg_of, rel_inf, small_cfg, torch_chain
from paper_2505_03352_b200 import workloads as W

RNG = np.random.default_rng(99)


def _rand_C(cfg):
    return RNG.random((cfg.mx, cfg.my)).astype(np.float32)


# ------------------------------------------------------------------ invariants
def test_c_zero_gives_average_permittivity(golden):
    # "With C=0 the initial design represents a block of material with a uniform
    # permittivity exactly equal to the average of core and cladding" (Eq. (3) form, eta = 0)
    cfg = small_cfg(mx=6, my=6, nz=16, z_lo=6.25, z_hi=9.75, radius=4.0, eta=0.0)
    eps, e2 = O.forward(cfg, np.zeros((6, 6), np.float32), 10.0, want_eps2d=True)
    assert np.max(np.abs(e2 - golden["uniform_c0_eq3"])) < 1e-14
    assert np.max(np.abs(eps[:2, :, :, 7:9] - golden["uniform_c0_eq3"])) < 1e-14
    assert np.max(np.abs(eps[:2, :, :, [6, 9]] - golden["face_xy_w075"])) < 1e-14
    assert np.max(np.abs(eps[2, :, :, [5, 9]] - golden["face_z_w025"])) < 1e-14
    assert np.all(eps[:, :, :, :5] == golden["eps_sio2"]) and np.all(eps[:, :, :, 10:] == golden["eps_sio2"])


@pytest.mark.parametrize("kind", [0, 1])
def test_uniform_c_gives_uniform_mixing_rule_value(kind):
    cfg = small_cfg(mx=7, my=9, filter_kind=kind, radius=3.0, sigma=1.5)
    for c0 in (0.0, 0.43, 0.5, 1.0):
        _, e2 = O.forward(cfg, np.full((7, 9), c0, np.float32), 8.0, want_eps2d=True)
        rho = 0.5 * (1 + np.tanh(8.0 * (np.float64(np.float32(c0)) - 0.5)))
        ref = rho * cfg.eps_core + (1 - rho) * cfg.eps_clad
        assert np.max(np.abs(e2 - ref)) < 1e-13 * ref


def test_eps_stays_between_cladding_and_core():
    w = W.CONFIGS[0]
    cfg = cfg_of(w)
    for beta in (1.0, 8.0, 64.0, 500.0):
        eps = O.forward(cfg, W.make_C(w)[0], beta)
        assert eps.min() >= cfg.eps_clad * (1 - 1e-15) and eps.max() <= cfg.eps_core * (1 + 1e-15)


def test_mirror_transpose_and_shift_symmetries():
    cfg = small_cfg(mx=10, my=10, radius=3.0, nz=4, z_lo=0.5, z_hi=3.0)
    C = _rand_C(cfg)
    _, e = O.forward(cfg, C, 9.0, want_eps2d=True)
    _, em = O.forward(cfg, C[::-1].copy(), 9.0, want_eps2d=True)           # x-mirror
    nx = cfg.nx
    assert np.max(np.abs(em[2] - e[2][::-1])) < 1e-13                       # E_z: i <-> nx-1-i
    assert np.max(np.abs(em[1] - e[1][::-1])) < 1e-13                       # E_y likewise
    # E_x sits half a cell toward +x: i <-> nx-2-i, away from the clamped last cell
    assert np.max(np.abs(em[0][1:nx - 2] - e[0][nx - 3:0:-1])) < 1e-13
    _, et = O.forward(cfg, C.T.copy(), 9.0, want_eps2d=True)               # transpose
    assert np.max(np.abs(et[0] - e[1].T)) < 1e-13 and np.max(np.abs(et[1] - e[0].T)) < 1e-13
    assert np.max(np.abs(et[2] - e[2].T)) < 1e-13
    # shift by one control pixel = shift by u cells in the interior (far from the borders)
    big = small_cfg(mx=24, my=10, radius=2.0, nz=4, z_lo=0.5, z_hi=3.0)
    Cb = np.full((24, 10), 0.5, np.float32); Cb[8:14] = RNG.random((6, 10)).astype(np.float32)
    Cs = np.roll(Cb, 1, axis=0)
    _, e0 = O.forward(big, Cb, 9.0, want_eps2d=True)
    _, e1 = O.forward(big, Cs, 9.0, want_eps2d=True)
    assert np.max(np.abs(e1[:, 2:] - e0[:, :-2])[:, 8:36]) < 1e-13


# ------------------------------------------------------------------ library / autograd second opinion
CASES = [
    dict(mx=9, my=8, radius=3.0, beta=6.0),
    dict(mx=8, my=9, radius=2.5, beta=20.0, s=4),
    dict(mx=10, my=8, filter_kind=1, radius=5.0, sigma=1.8, beta=8.0),
    dict(mx=8, my=8, radius=3.0, beta=5.0, eta=0.0, normalize=0),
    dict(mx=7, my=8, radius=3.5, beta=12.0, u=3),
]


@pytest.mark.parametrize("case", CASES)
def test_forward_and_vjp_match_float64_library_autograd_chain(case):
    case = dict(case)
    beta = case.pop("beta")
    cfg = small_cfg(nz=8, z_lo=2.25, z_hi=5.75, **case)
    C = _rand_C(cfg) if cfg.normalize else (_rand_C(cfg) - 0.5) * 0.2
    C = C.astype(np.float32)
    Ct = torch.from_numpy(C.astype(np.float64)).requires_grad_(True)
    eps_t = torch_chain(cfg, Ct, beta)
    eps = O.forward(cfg, C, beta)
    assert np.max(np.abs(eps - eps_t.detach().numpy()) / eps) < 1e-12
    wbar = RNG.standard_normal(eps.shape)
    (eps_t * torch.from_numpy(wbar)).sum().backward()
    g = O.vjp_real(cfg, C, beta, wbar)
    assert rel_inf(g, Ct.grad.numpy()) < 1e-11


def test_forward_stages_equal_the_stage_functions_composed():
    cfg = small_cfg(mx=8, my=7, radius=3.0)
    C = _rand_C(cfg)
    st = O.forward_stages(cfg, C, 11.0)
    Phi = O.filter(cfg, C.astype(np.float64))
    rho = O.project(Phi, 11.0, cfg.eta)
    e, r = O.mix(cfg, rho)
    assert np.array_equal(st["Phi"], Phi) and np.array_equal(st["rho"], rho) and np.array_equal(st["e"], e)
    for c in range(3):
        A, H, D = O.average(cfg, e, c), O.average(cfg, r, c), O.average(cfg, rho, c)
        assert np.array_equal(st["A"][c], A) and np.array_equal(st["H"][c], H) and np.array_equal(st["D"][c], D)
        gx, gy = O.sobel(cfg, D) if c < 2 else (None, None)
        if c < 2:
            assert np.array_equal(st["gx"][c], gx) and np.array_equal(st["gy"][c], gy)
        assert np.array_equal(st["eps2d"][c], O.eq7(cfg, c, A, H, gx, gy)[0])
    assert np.array_equal(O.extrude(cfg, st["eps2d"]), O.forward(cfg, C, 11.0))


# ------------------------------------------------------------------ adjoint identity and finite differences
@pytest.mark.parametrize("kind,beta", [(0, 8.0), (1, 8.0), (0, 40.0)])
def test_adjoint_identity_end_to_end(kind, beta):
    # <J v, w> = <v, J^T w> with J v from central differences of the float64 forward
    cfg = small_cfg(mx=8, my=8, filter_kind=kind, radius=3.0, sigma=1.5)
    C = (np.round(_rand_C(cfg) * 4096) / 4096).astype(np.float32)
    v = RNG.standard_normal(C.shape)
    w = RNG.standard_normal((3, cfg.nx, cfg.ny, cfg.nz))
    # C is handed over as fp32, so perturb on an fp32-exact lattice (multiples of 2^-22)
    h = 2.0 ** -16
    dv = (np.round(v * 64) / 64 * h).astype(np.float32)
    Cp, Cm = C + dv, C - dv
    assert np.array_equal((Cp.astype(np.float64) - Cm.astype(np.float64)), 2.0 * dv.astype(np.float64))
    Jv = (O.forward(cfg, Cp, beta) - O.forward(cfg, Cm, beta)) / 2.0       # = J (dv) + O(h^3)
    lhs = np.sum(Jv * w)
    rhs = np.sum(dv.astype(np.float64) * O.vjp_real(cfg, C, beta, w))
    assert abs(lhs - rhs) < 2e-5 * abs(rhs)


def test_vjp_matches_central_finite_differences_on_tiny():
    w0 = W.small_variant(W.CONFIGS[0], 8, 8)
    cfg = cfg_of(w0)
    C = W.make_C(w0)[0]
    wbar = RNG.standard_normal((3, cfg.nx, cfg.ny, cfg.nz))
    g = O.vjp_real(cfg, C, 8.0, wbar)
    h = np.float32(2.0 ** -11)
    for idx in [(0, 0), (3, 4), (7, 7), (2, 6), (5, 0)]:
        Cp, Cm = C.copy(), C.copy()
        Cp[idx] += h; Cm[idx] -= h
        step = float(Cp[idx]) - float(Cm[idx])
        fd = np.sum(wbar * (O.forward(cfg, Cp, 8.0) - O.forward(cfg, Cm, 8.0))) / step
        assert abs(fd - g[idx]) < 1e-5 * np.max(np.abs(g)), (idx, fd, g[idx])


# ------------------------------------------------------------------ Eq. (1) assembly
def test_eq1_assembly_real_imaginary_and_linearity():
    w0 = W.small_variant(W.CONFIGS[0], 8, 8)
    cfg = cfg_of(w0)
    C = W.make_C(w0)[0]
    shape = (3, cfg.nx, cfg.ny, cfg.nz)
    wbar = RNG.standard_normal(shape).astype(np.float32)
    ref = O.vjp_real(cfg, C, 8.0, wbar.astype(np.float64))
    # real-field special case: E_F = -w/2, E_A = 1  =>  -2 Re(E_F E_A) = w
    EF = (-0.5 * wbar).astype(np.complex64); EA = np.ones(shape, np.complex64)
    assert rel_inf(O.vjp(cfg, C, 8.0, [EF], [EA]), ref) < 1e-14
    # purely imaginary pair: (i a)(i b) = -ab flips the sign
    assert rel_inf(O.vjp(cfg, C, 8.0, [1j * EF], [1j * EA]), -ref) < 1e-14
    # general complex pair against numpy's complex product (plain product, no conjugate: P:L35)
    EF = W.make_field(w0, 0, 0); EA = W.make_field(w0, 0, 1)
    G3 = -2.0 * np.real(EF.astype(np.complex128) * EA.astype(np.complex128))
    g1 = O.vjp(cfg, C, 8.0, [EF], [EA])
    assert rel_inf(g1, O.vjp_real(cfg, C, 8.0, G3)) < 1e-14
    assert rel_inf(O.vjp(cfg, C, 8.0, [EF], [np.conj(EA)]), g1) > 1e-2          # a conjugate would change it
    # linearity in the pairs
    EF2 = W.make_field(w0, 1, 0); EA2 = W.make_field(w0, 1, 1)
    g2 = O.vjp(cfg, C, 8.0, [EF2], [EA2])
    assert rel_inf(O.vjp(cfg, C, 8.0, [EF, EF2], [EA, EA2]), g1 + g2) < 1e-13


def test_tiny_config_shapes_and_determinism():
    w = W.CONFIGS[0]
    C = W.make_C(w)
    assert C.shape == (1, 32, 32) and C.dtype == np.float32 and 0 <= C.min() and C.max() < 1
    assert np.array_equal(C, W.make_C(w))
    f = W.make_field(w, 0, 0)
    assert f.shape == (3, 64, 64, 16) and f.dtype == np.complex64
    assert np.array_equal(f, W.make_field(w, 0, 0)) and not np.array_equal(f, W.make_field(w, 0, 1))
    assert abs(f.real.std() - 1) < 0.02 and abs(f.imag.std() - 1) < 0.02
