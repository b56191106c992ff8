"""float64 CPU oracle of the C -> eps_hat chain and its Eq. (1) reverse pass.

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  It shares nothing with ``paper_2505_03352_b200`` (the CUDA path) and
never imports it; the arithmetic lives in ``epsgrad_oracle.c`` (plain C loops,
one function per step of the paper's chain), this file only marshals numpy
arrays into it.  See the header of ``epsgrad_oracle.c`` for citations and pins.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "epsgrad_oracle.c")
_LIB = os.path.join(_HERE, "libepsgrad_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (``-O2 -fopenmp``); returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-Wall", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


class _Cfg(ctypes.Structure):
    _fields_ = [
        ("mx", ctypes.c_int32), ("my", ctypes.c_int32),
        ("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
        ("s", ctypes.c_int32), ("filter_kind", ctypes.c_int32), ("normalize", ctypes.c_int32),
        ("radius", ctypes.c_double), ("sigma", ctypes.c_double),
        ("z_lo", ctypes.c_double), ("z_hi", ctypes.c_double),
        ("eta", ctypes.c_double), ("eps_core", ctypes.c_double), ("eps_clad", ctypes.c_double),
        ("delta", ctypes.c_double), ("morph_diam", ctypes.c_double), ("morph_alpha", ctypes.c_double),
    ]


@dataclass
class OracleConfig:
    """Geometry and materials of one design region (cell units, see the C header)."""
    mx: int
    my: int
    nx: int
    ny: int
    nz: int
    z_lo: float
    z_hi: float
    s: int = 2
    filter_kind: int = 0            # 0 conic, 1 Gaussian (per-axis truncation)
    radius: float = 4.0
    sigma: float = 1.0
    normalize: int = 1
    eta: float = 0.5
    eps_core: float = 12.11
    eps_clad: float = 2.085
    delta: float = 1e-12
    morph_diam: float = 0.0         # d of Eqs. (4)-(5) in Yee cells; 0 = morphological filters off
    morph_alpha: float = 20.0

    def c(self) -> _Cfg:
        return _Cfg(self.mx, self.my, self.nx, self.ny, self.nz, self.s, self.filter_kind,
                    self.normalize, self.radius, self.sigma, self.z_lo, self.z_hi, self.eta,
                    self.eps_core, self.eps_clad, self.delta, self.morph_diam, self.morph_alpha)

    @property
    def px(self) -> int:
        return self.s * self.nx

    @property
    def py(self) -> int:
        return self.s * self.ny


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_weight.restype = ctypes.c_double
        _lib.orc_weight.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_double]
        _lib.orc_num_threads.restype = ctypes.c_int
    return _lib


def _p(a: np.ndarray | None):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f64(a, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ----------------------------------------------------------------- stages
def weight(cfg: OracleConfig, dx: float, dy: float) -> float:
    c = cfg.c()
    return float(lib().orc_weight(ctypes.byref(c), ctypes.c_double(dx), ctypes.c_double(dy)))


def filter(cfg: OracleConfig, C, return_den: bool = False):
    c = cfg.c()
    C = _f64(C, (cfg.mx, cfg.my))
    Phi = np.empty((cfg.px, cfg.py))
    den = np.empty((cfg.px, cfg.py)) if return_den else None
    lib().orc_filter(ctypes.byref(c), _p(C), _p(Phi), _p(den))
    return (Phi, den) if return_den else Phi


def filter_T(cfg: OracleConfig, Phibar):
    c = cfg.c()
    Phibar = _f64(Phibar, (cfg.px, cfg.py))
    Cbar = np.empty((cfg.mx, cfg.my))
    lib().orc_filter_T(ctypes.byref(c), _p(Phibar), _p(Cbar))
    return Cbar


def morph(cfg: OracleConfig, x, erode: bool):
    """Eq. (4) (dilate) or Eq. (5) (erode) on the mask grid"""
    c = cfg.c()
    x = _f64(x, (cfg.px, cfg.py))
    y = np.empty_like(x)
    lib().orc_morph(ctypes.byref(c), _p(x), ctypes.c_int(int(erode)), _p(y))
    return y


def morph_T(cfg: OracleConfig, x, erode: bool, ybar):
    c = cfg.c()
    x = _f64(x, (cfg.px, cfg.py))
    ybar = _f64(ybar, (cfg.px, cfg.py))
    xbar = np.zeros_like(x)
    lib().orc_morph_T(ctypes.byref(c), _p(x), ctypes.c_int(int(erode)), _p(ybar), _p(xbar))
    return xbar


def project(Phi, beta: float, eta: float):
    Phi = _f64(Phi)
    rho = np.empty_like(Phi)
    lib().orc_project(ctypes.c_int64(Phi.size), _p(Phi), ctypes.c_double(beta), ctypes.c_double(eta), _p(rho))
    return rho


def project_T(Phi, beta: float, eta: float, rhobar):
    Phi = _f64(Phi)
    rhobar = _f64(rhobar, Phi.shape)
    out = np.empty_like(Phi)
    lib().orc_project_T(ctypes.c_int64(Phi.size), _p(Phi), ctypes.c_double(beta), ctypes.c_double(eta),
                        _p(rhobar), _p(out))
    return out


def mix(cfg: OracleConfig, rho):
    c = cfg.c()
    rho = _f64(rho)
    e, r = np.empty_like(rho), np.empty_like(rho)
    lib().orc_mix(ctypes.byref(c), ctypes.c_int64(rho.size), _p(rho), _p(e), _p(r))
    return e, r


def mix_T(cfg: OracleConfig, e, ebar, rbar, rhobar):
    """returns rhobar + d(e,r)/d(rho)^T (ebar, rbar)"""
    c = cfg.c()
    e = _f64(e)
    out = _f64(rhobar, e.shape).copy()
    lib().orc_mix_T(ctypes.byref(c), ctypes.c_int64(e.size), _p(e), _p(_f64(ebar, e.shape)),
                    _p(_f64(rbar, e.shape)), _p(out))
    return out


def average(cfg: OracleConfig, f, comp: int):
    c = cfg.c()
    f = _f64(f, (cfg.px, cfg.py))
    out = np.empty((cfg.nx, cfg.ny))
    lib().orc_average(ctypes.byref(c), _p(f), ctypes.c_int(comp), _p(out))
    return out


def average_T(cfg: OracleConfig, outbar, comp: int):
    c = cfg.c()
    outbar = _f64(outbar, (cfg.nx, cfg.ny))
    fbar = np.zeros((cfg.px, cfg.py))
    lib().orc_average_T(ctypes.byref(c), _p(outbar), ctypes.c_int(comp), _p(fbar))
    return fbar


def sobel(cfg: OracleConfig, D):
    c = cfg.c()
    D = _f64(D, (cfg.nx, cfg.ny))
    gx, gy = np.empty_like(D), np.empty_like(D)
    lib().orc_sobel(ctypes.byref(c), _p(D), _p(gx), _p(gy))
    return gx, gy


def sobel_T(cfg: OracleConfig, gxbar, gybar):
    c = cfg.c()
    gxbar = _f64(gxbar, (cfg.nx, cfg.ny))
    gybar = _f64(gybar, (cfg.nx, cfg.ny))
    Dbar = np.zeros((cfg.nx, cfg.ny))
    lib().orc_sobel_T(ctypes.byref(c), _p(gxbar), _p(gybar), _p(Dbar))
    return Dbar


def eq7(cfg: OracleConfig, comp: int, A, H, gx, gy):
    """returns (eps2d_c, n_c^2)"""
    c = cfg.c()
    A = _f64(A, (cfg.nx, cfg.ny))
    H = _f64(H, A.shape)
    gx = None if gx is None else _f64(gx, A.shape)
    gy = None if gy is None else _f64(gy, A.shape)
    out, n2 = np.empty_like(A), np.empty_like(A)
    lib().orc_eq7(ctypes.byref(c), ctypes.c_int(comp), _p(A), _p(H), _p(gx), _p(gy), _p(out), _p(n2))
    return out, n2


def eq7_T(cfg: OracleConfig, comp: int, A, H, gx, gy, eps2dbar):
    """returns (Abar, Hbar, gxbar, gybar)"""
    c = cfg.c()
    A = _f64(A, (cfg.nx, cfg.ny))
    H = _f64(H, A.shape)
    gx = None if gx is None else _f64(gx, A.shape)
    gy = None if gy is None else _f64(gy, A.shape)
    eb = _f64(eps2dbar, A.shape)
    outs = [np.empty_like(A) for _ in range(4)]
    lib().orc_eq7_T(ctypes.byref(c), ctypes.c_int(comp), _p(A), _p(H), _p(gx), _p(gy), _p(eb),
                    *[_p(o) for o in outs])
    return tuple(outs)


def zweights(cfg: OracleConfig):
    c = cfg.c()
    wxy, wz = np.empty(cfg.nz), np.empty(cfg.nz)
    lib().orc_zweights(ctypes.byref(c), _p(wxy), _p(wz))
    return wxy, wz


def extrude(cfg: OracleConfig, eps2d):
    c = cfg.c()
    eps2d = _f64(eps2d, (3, cfg.nx, cfg.ny))
    eps = np.empty((3, cfg.nx, cfg.ny, cfg.nz))
    lib().orc_extrude(ctypes.byref(c), _p(eps2d), _p(eps))
    return eps


def extrude_T(cfg: OracleConfig, eps2d, epsbar):
    c = cfg.c()
    eps2d = _f64(eps2d, (3, cfg.nx, cfg.ny))
    epsbar = _f64(epsbar, (3, cfg.nx, cfg.ny, cfg.nz))
    out = np.empty((3, cfg.nx, cfg.ny))
    lib().orc_extrude_T(ctypes.byref(c), _p(eps2d), _p(epsbar), _p(out))
    return out


# ----------------------------------------------------------------- whole chain
def _c32(C, cfg: OracleConfig) -> np.ndarray:
    C = np.ascontiguousarray(C, dtype=np.float32)
    assert C.shape == (cfg.mx, cfg.my), (C.shape, (cfg.mx, cfg.my))
    return C


def forward(cfg: OracleConfig, C, beta: float, want_eps2d: bool = False):
    """eps [3,nx,ny,nz] float64 from one design's C [mx,my] (fp32 as the GPU sees it)."""
    c = cfg.c()
    C = _c32(C, cfg)
    eps = np.empty((3, cfg.nx, cfg.ny, cfg.nz))
    e2 = np.empty((3, cfg.nx, cfg.ny)) if want_eps2d else None
    lib().orc_forward(ctypes.byref(c), _p(C), ctypes.c_double(beta), _p(eps), _p(e2))
    return (eps, e2) if want_eps2d else eps


def forward_stages(cfg: OracleConfig, C, beta: float) -> dict:
    """every intermediate of the 2-D stage plus eps2d (no z-extrusion)."""
    c = cfg.c()
    C = _c32(C, cfg)
    m, n = (cfg.px, cfg.py), (cfg.nx, cfg.ny)
    st = dict(Phi=np.empty(m), rho=np.empty(m), e=np.empty(m), r=np.empty(m),
              A=np.empty((3,) + n), H=np.empty((3,) + n), D=np.empty((3,) + n),
              gx=np.empty((2,) + n), gy=np.empty((2,) + n), eps2d=np.empty((3,) + n))
    lib().orc_forward_stages(ctypes.byref(c), _p(C), ctypes.c_double(beta),
                             *[_p(st[k]) for k in ("Phi", "rho", "e", "r", "A", "H", "D", "gx", "gy", "eps2d")])
    return st


def vjp_real(cfg: OracleConfig, C, beta: float, epsbar):
    """(d eps/dC)^T epsbar for a real cotangent epsbar [3,nx,ny,nz] -> [mx,my] float64."""
    c = cfg.c()
    C = _c32(C, cfg)
    epsbar = _f64(epsbar, (3, cfg.nx, cfg.ny, cfg.nz))
    out = np.empty((cfg.mx, cfg.my))
    lib().orc_vjp_real(ctypes.byref(c), _p(C), ctypes.c_double(beta), _p(epsbar), _p(out))
    return out


def vjp_real_beta(cfg: OracleConfig, C, beta: float, epsbar):
    """((d eps/dC)^T epsbar [mx,my], epsbar . d eps/d beta) for a real cotangent."""
    c = cfg.c()
    C = _c32(C, cfg)
    epsbar = _f64(epsbar, (3, cfg.nx, cfg.ny, cfg.nz))
    out = np.empty((cfg.mx, cfg.my))
    db = ctypes.c_double(0.0)
    lib().orc_vjp_real_beta(ctypes.byref(c), _p(C), ctypes.c_double(beta), _p(epsbar), _p(out), ctypes.byref(db))
    return out, float(db.value)


def unbinarity(cfg: OracleConfig, C, beta: float) -> float:
    """u(beta): mean of 4 rho (1 - rho) over the projected design mask (S20)."""
    c = cfg.c()
    lib().orc_unbinarity.restype = ctypes.c_double
    return float(lib().orc_unbinarity(ctypes.byref(c), _p(_c32(C, cfg)), ctypes.c_double(beta)))


def beta_schedule(beta_min: float, beta_max: float, i: int, n_iter: int) -> float:
    """Eq. (14)."""
    lib().orc_beta_schedule.restype = ctypes.c_double
    return float(lib().orc_beta_schedule(ctypes.c_double(beta_min), ctypes.c_double(beta_max), ctypes.c_int(i), ctypes.c_int(n_iter)))


def beta_update(t: float, beta_max: float, gamma: float, u: float, u0: float, beta: float):
    """Eq. (15): returns the new (t, beta_max)."""
    ct, cb = ctypes.c_double(t), ctypes.c_double(beta_max)
    lib().orc_beta_update(ctypes.byref(ct), ctypes.byref(cb), ctypes.c_double(gamma), ctypes.c_double(u),
                          ctypes.c_double(u0), ctypes.c_double(beta))
    return float(ct.value), float(cb.value)


def vjp_beta(cfg: OracleConfig, C, beta: float, EF: list, EA: list):
    """Eq. (1) gradient and d F/d beta from field pairs (complex64 [3,nx,ny,nz])."""
    c = cfg.c()
    C = _c32(C, cfg)
    n = len(EF)
    assert n == len(EA) and n >= 1
    keep = [[np.ascontiguousarray(a, dtype=np.complex64) for a in lst] for lst in (EF, EA)]
    for a in keep[0] + keep[1]:
        assert a.shape == (3, cfg.nx, cfg.ny, cfg.nz)
    pf = (ctypes.c_void_p * n)(*[a.ctypes.data for a in keep[0]])
    pa = (ctypes.c_void_p * n)(*[a.ctypes.data for a in keep[1]])
    out = np.empty((cfg.mx, cfg.my))
    db = ctypes.c_double(0.0)
    lib().orc_vjp_beta(ctypes.byref(c), _p(C), ctypes.c_double(beta), ctypes.c_int(n), pf, pa, _p(out), ctypes.byref(db))
    return out, float(db.value)


def adam_step(C, M, V, G, i: int, b1=0.9, b2=0.999, lr=1e-3, eps=1e-8):
    """Eqs. (10)-(11): one Adam step i >= 1 on float64 copies; returns (C, M, V)."""
    C, M, V = (np.array(a, dtype=np.float64, order="C") for a in (C, M, V))
    G = _f64(G)
    lib().orc_adam_step(ctypes.c_int64(C.size), _p(C), _p(M), _p(V), _p(G), ctypes.c_int(i), ctypes.c_double(b1),
                        ctypes.c_double(b2), ctypes.c_double(lr), ctypes.c_double(eps))
    return C, M, V


def vjp(cfg: OracleConfig, C, beta: float, EF: list, EA: list):
    """Eq. (1): -2 Re((d eps/dC)^T (E_F . E_A)) summed over the pairs; fields complex64 [3,nx,ny,nz]."""
    c = cfg.c()
    C = _c32(C, cfg)
    n = len(EF)
    assert n == len(EA) and n >= 1
    shape = (3, cfg.nx, cfg.ny, cfg.nz)
    keep = []
    for lst in (EF, EA):
        arrs = [np.ascontiguousarray(a, dtype=np.complex64) for a in lst]
        for a in arrs:
            assert a.shape == shape, (a.shape, shape)
        keep.append(arrs)
    pf = (ctypes.c_void_p * n)(*[a.ctypes.data for a in keep[0]])
    pa = (ctypes.c_void_p * n)(*[a.ctypes.data for a in keep[1]])
    out = np.empty((cfg.mx, cfg.my))
    lib().orc_vjp(ctypes.byref(c), _p(C), ctypes.c_double(beta), ctypes.c_int(n), pf, pa, _p(out))
    return out


# ---- SOAP, Eqs. (12)-(13): plain numpy, see soap.py
from .soap import soap_accumulate, soap_eigenbasis, soap_step  # noqa: E402,F401
