"""Thin ctypes binding of ``include/epsgrad.h`` -- argument marshalling only.

Every step of the path runs in the CUDA kernels of ``libepsgrad.so``; torch is used for
device memory (tensors, workspace) and the current CUDA stream.  There is no CPU path: a
missing library or a missing CUDA device is a hard error.  Names follow the C ABI.
"""
from __future__ import annotations

import ctypes
import os
from typing import Sequence

from . import build as _build

OK, EINVAL, EUNSUPPORTED, ENOWORKSPACE, ECUDA, ENOMEM = 0, -1, -2, -3, -4, -5
FILTER_CONIC, FILTER_GAUSSIAN = 0, 1

EXPORTS = (
    "epsgrad_plan_create", "epsgrad_plan_destroy", "epsgrad_workspace_bytes",
    "epsgrad_plan_set_workspace", "epsgrad_staging_bytes", "epsgrad_plan_set_staging",
    "epsgrad_plan_set_dense_reads", "epsgrad_plan_last_launches", "epsgrad_plan_last_copy_bytes",
    "epsgrad_plan_set_profiling", "epsgrad_plan_last_kernel_times", "epsgrad_plan_set_overlap", "epsgrad_plan_set_host_direct", "epsgrad_plan_set_embedding", "epsgrad_plan_set_slab", "epsgrad_plan_set_packed_fields", "epsgrad_plan_packed_window", "epsgrad_plan_set_eps_window_only", "epsgrad_plan_set_tma", "epsgrad_plan_set_bulk_stores", "epsgrad_plan_set_pdl", "epsgrad_plan_set_tensor_cores", "epsgrad_plan_set_tuning", "epsgrad_plan_set_fused", "epsgrad_plan_fused_profile", "epsgrad_plan_set_timeline", "epsgrad_plan_read_timeline", 
    "eps_forward", "eps_vjp", "eps_forward_vjp", "eps_forward_vjp_host", "eps_vjp_beta", "eps_unbinarity",
    "eps_unbinarity_static", "epsgrad_static_scratch_partials",
    "epsgrad_beta_schedule", "epsgrad_beta_update", "epsgrad_adam_step",
    "epsgrad_soap_accumulate", "epsgrad_soap_eigh_workspace_bytes", "epsgrad_soap_eigh", "epsgrad_soap_eigh_info",
    "epsgrad_soap_step_workspace_bytes", "epsgrad_soap_step",
    "epsgrad_stage_filter", "epsgrad_stage_eps2d", "epsgrad_stage_zreduce",
    "epsgrad_status_string", "epsgrad_version",
)


class EpsgradError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)} ({status})")


class Embedding(ctypes.Structure):
    """epsgrad_embedding_t (include/epsgrad.h)."""
    _fields_ = [(n, ctypes.c_int32) for n in ("nx_full", "ny_full", "nz_full", "i0", "j0", "k0")]


class Config(ctypes.Structure):
    """epsgrad_config_t (include/epsgrad.h)."""
    _fields_ = [
        ("batch", ctypes.c_int32), ("mx", ctypes.c_int32), ("my", ctypes.c_int32),
        ("upsample", ctypes.c_int32), ("subpixel", ctypes.c_int32), ("nz", ctypes.c_int32),
        ("filter_kind", ctypes.c_int32), ("filter_normalize", ctypes.c_int32),
        ("nx_cells", ctypes.c_int32), ("ny_cells", ctypes.c_int32),
        ("z_lo", ctypes.c_double), ("z_hi", ctypes.c_double),
        ("filter_radius", ctypes.c_double), ("filter_sigma", ctypes.c_double),
        ("eta", ctypes.c_double), ("eps_core", ctypes.c_double), ("eps_clad", ctypes.c_double),
        ("normal_delta", ctypes.c_double), ("morph_diameter", ctypes.c_double), ("morph_alpha", ctypes.c_double),
    ]

    @property
    def nx(self) -> int:
        return self.nx_cells if self.nx_cells > 0 else self.upsample * self.mx

    @property
    def ny(self) -> int:
        return self.ny_cells if self.ny_cells > 0 else self.upsample * self.my


def make_config(*, batch=1, mx, my, nz, z_lo, z_hi, upsample=2, subpixel=2, filter_kind=FILTER_CONIC,
                filter_radius=4.0, filter_sigma=1.0, filter_normalize=1, eta=0.5, eps_core=12.11,
                eps_clad=2.085, normal_delta=1e-8, morph_diameter=0.0, morph_alpha=20.0, nx_cells=0, ny_cells=0) -> Config:
    return Config(batch, mx, my, upsample, subpixel, nz, filter_kind, filter_normalize, nx_cells, ny_cells, z_lo, z_hi,
                  filter_radius, filter_sigma, eta, eps_core, eps_clad, normal_delta, morph_diameter, morph_alpha)


def config_of(w) -> Config:
    """Config of a ``workloads.Workload``."""
    return make_config(batch=w.batch, mx=w.mx, my=w.my, nz=w.nz, z_lo=w.z_lo, z_hi=w.z_hi, upsample=w.upsample,
                       subpixel=w.subpixel, filter_kind=w.filter_kind, filter_radius=w.radius,
                       filter_sigma=w.sigma if w.sigma > 0 else 1.0, eta=w.eta, eps_core=w.eps_core,
                       eps_clad=w.eps_clad, normal_delta=w.normal_delta,
                       morph_diameter=getattr(w, "morph_diameter", 0.0), morph_alpha=getattr(w, "morph_alpha", 20.0),
                       nx_cells=getattr(w, "nx_cells", 0), ny_cells=getattr(w, "ny_cells", 0))


_lib = None


def adam_step(C, M, V, G, step: int, b1=0.9, b2=0.999, lr=1e-3, eps=1e-8) -> None:
    """Eqs. (10)-(11) in place on CUDA float32 tensors of one shape (current stream)."""
    import torch
    for x in (C, M, V, G):
        assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() and x.shape == C.shape
    _check(lib().epsgrad_adam_step(C.data_ptr(), M.data_ptr(), V.data_ptr(), G.data_ptr(), C.numel(), step, b1, b2, lr, eps,
                                   torch.cuda.current_stream(C.device).cuda_stream), "epsgrad_adam_step")


class Soap:
    """State and calls of the SOAP optimizer, Eqs. (12)-(13), for one [mx,my] matrix of control variables on a
    CUDA device: owns M, V', L, R, Q_L, Q_R and the scratch buffers; every step of the arithmetic is a library call."""

    def __init__(self, mx: int, my: int, device=None):
        import torch
        self._torch = torch
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        z = lambda *shape: torch.zeros(*shape, dtype=torch.float32, device=self.device)
        self.mx, self.my = mx, my
        self.M, self.Vp, self.L, self.R = z(mx, my), z(mx, my), z(mx, mx), z(my, my)
        self.QL, self.QR = torch.eye(mx, dtype=torch.float32, device=self.device), torch.eye(my, dtype=torch.float32, device=self.device)
        self.wL, self.wR = z(mx), z(my)
        self._work = torch.empty(lib().epsgrad_soap_step_workspace_bytes(mx, my), dtype=torch.uint8, device=self.device)
        self._ework = None
        self.step = 0

    def _stream(self):
        return self._torch.cuda.current_stream(self.device).cuda_stream

    def _chk(self, *ts):
        t = self._torch
        for x in ts:
            assert x.is_cuda and x.dtype == t.float32 and x.is_contiguous()

    def accumulate(self, G, b2=0.999) -> None:
        """Eq. (12)"""
        self._chk(G)
        assert tuple(G.shape) == (self.mx, self.my)
        with self._torch.cuda.device(self.device):
            _check(lib().epsgrad_soap_accumulate(self.L.data_ptr(), self.R.data_ptr(), G.data_ptr(), self.mx, self.my, b2,
                                                 self._stream()), "epsgrad_soap_accumulate")

    def eigh(self, A, Q, w, check: bool = False) -> None:
        """Q, w <- eigenvectors (columns) and ascending eigenvalues of the symmetric A; check: read the solver's status back
        (synchronises the stream) and raise if it did not converge"""
        t = self._torch
        self._chk(A, Q, w)
        n = A.shape[0]
        assert tuple(A.shape) == (n, n) and tuple(Q.shape) == (n, n) and tuple(w.shape) == (n,)
        with t.cuda.device(self.device):
            need = lib().epsgrad_soap_eigh_workspace_bytes(n)
            if need == 0:
                raise EpsgradError(EUNSUPPORTED, "epsgrad_soap_eigh_workspace_bytes")
            if self._ework is None or self._ework.numel() < need:
                self._ework = t.empty(need, dtype=t.uint8, device=self.device)
            _check(lib().epsgrad_soap_eigh(A.data_ptr(), Q.data_ptr(), w.data_ptr(), n, self._ework.data_ptr(), self._ework.numel(),
                                           self._stream()), "epsgrad_soap_eigh")
            if check:
                info = ctypes.c_int(-1)
                _check(lib().epsgrad_soap_eigh_info(self._ework.data_ptr(), self._ework.numel(), n, self._stream(), ctypes.byref(info)),
                       "epsgrad_soap_eigh_info")
                if info.value != 0:
                    raise RuntimeError(f"epsgrad_soap_eigh: the eigensolver did not converge (info = {info.value})")

    def refresh(self) -> None:
        """Q_L, Q_R <- eigenvectors of L, R"""
        self.eigh(self.L, self.QL, self.wL)
        self.eigh(self.R, self.QR, self.wR)

    def update(self, C, G, b1=0.9, b2=0.999, lr=1e-3, eps=1e-8) -> None:
        """Eq. (13) in place on C with the current bases; counts the step"""
        self._chk(C, G)
        assert tuple(C.shape) == (self.mx, self.my) and tuple(G.shape) == (self.mx, self.my)
        self.step += 1
        with self._torch.cuda.device(self.device):
            _check(lib().epsgrad_soap_step(C.data_ptr(), self.M.data_ptr(), self.Vp.data_ptr(), G.data_ptr(), self.QL.data_ptr(),
                                           self.QR.data_ptr(), self.mx, self.my, self.step, b1, b2, lr, eps,
                                           self._work.data_ptr(), self._work.numel(), self._stream()), "epsgrad_soap_step")


def beta_schedule(beta_min: float, beta_max: float, i: int, n_iter: int) -> float:
    """Eq. (14)."""
    return float(lib().epsgrad_beta_schedule(beta_min, beta_max, i, n_iter))


def beta_update(t: float, beta_max: float, gamma: float, u: float, u0: float, beta: float):
    """Eq. (15): the new (t, beta_max)."""
    ct, cb = ctypes.c_double(t), ctypes.c_double(beta_max)
    _check(lib().epsgrad_beta_update(ctypes.byref(ct), ctypes.byref(cb), gamma, u, u0, beta), "epsgrad_beta_update")
    return float(ct.value), float(cb.value)


def lib() -> ctypes.CDLL:
    """Load (building if stale and nvcc is present) libepsgrad.so; raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.stale():
        try:
            path = _build.build()
        except Exception as e:  # no nvcc on this box: use the shipped library if there is one
            if not os.path.exists(path):
                raise RuntimeError(f"libepsgrad.so is missing and could not be built: {e}") from e
    L = ctypes.CDLL(path)
    vp, i32, f32, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_size_t
    L.epsgrad_plan_create.argtypes = [ctypes.POINTER(Config), i32, ctypes.POINTER(vp)]
    L.epsgrad_plan_destroy.argtypes = [vp]
    L.epsgrad_workspace_bytes.argtypes = [vp]
    L.epsgrad_workspace_bytes.restype = sz
    L.epsgrad_plan_set_workspace.argtypes = [vp, vp, sz]
    L.epsgrad_staging_bytes.argtypes = [vp, i32]
    L.epsgrad_staging_bytes.restype = sz
    L.epsgrad_plan_set_staging.argtypes = [vp, vp, sz]
    L.epsgrad_plan_set_dense_reads.argtypes = [vp, i32]
    L.epsgrad_plan_last_launches.argtypes = [vp]
    L.epsgrad_plan_last_copy_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]
    L.epsgrad_plan_set_profiling.argtypes = [vp, i32]
    L.epsgrad_plan_last_kernel_times.argtypes = [vp, i32, ctypes.POINTER(f32), ctypes.POINTER(ctypes.c_char_p)]
    L.eps_forward.argtypes = [vp, vp, f32, vp, vp]
    L.eps_vjp.argtypes = [vp, vp, f32, i32, vp, vp, vp, vp]
    L.eps_vjp_beta.argtypes = [vp, vp, f32, i32, vp, vp, vp, vp, vp]
    L.eps_unbinarity.argtypes = [vp, vp, f32, vp, vp]
    L.epsgrad_beta_schedule.restype = ctypes.c_double
    L.epsgrad_beta_schedule.argtypes = [ctypes.c_double, ctypes.c_double, i32, i32]
    L.epsgrad_adam_step.argtypes = [vp, vp, vp, vp, sz, i32, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double, vp]
    L.epsgrad_beta_update.argtypes = [vp, vp, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double]
    L.epsgrad_soap_accumulate.argtypes = [vp, vp, vp, i32, i32, ctypes.c_double, vp]
    L.epsgrad_soap_eigh_workspace_bytes.restype = sz
    L.epsgrad_soap_eigh_workspace_bytes.argtypes = [i32]
    L.epsgrad_soap_eigh.argtypes = [vp, vp, vp, i32, vp, sz, vp]
    L.epsgrad_soap_eigh_info.argtypes = [vp, sz, i32, vp, ctypes.POINTER(ctypes.c_int)]
    L.epsgrad_soap_step_workspace_bytes.restype = sz
    L.epsgrad_soap_step_workspace_bytes.argtypes = [i32, i32]
    L.epsgrad_soap_step.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                    ctypes.c_double, vp, sz, vp]
    L.eps_forward_vjp.argtypes = [vp, vp, f32, i32, vp, vp, vp, vp, vp]
    L.eps_forward_vjp_host.argtypes = [vp, vp, f32, i32, vp, vp, vp, vp, vp]
    L.epsgrad_stage_filter.argtypes = [vp, vp, vp, vp]
    L.epsgrad_stage_eps2d.argtypes = [vp, vp, f32, vp, vp]
    L.epsgrad_plan_set_overlap.argtypes = [vp, i32]
    L.epsgrad_plan_set_host_direct.argtypes = [vp, i32]
    L.epsgrad_plan_set_slab.argtypes = [vp, i32, i32]
    L.epsgrad_plan_set_embedding.argtypes = [vp, vp]
    L.epsgrad_plan_set_tma.argtypes = [vp, i32]
    L.epsgrad_plan_set_packed_fields.argtypes = [vp, i32]
    L.epsgrad_plan_set_eps_window_only.argtypes = [vp, i32]
    L.epsgrad_plan_packed_window.argtypes = [vp, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]
    L.epsgrad_plan_set_bulk_stores.argtypes = [vp, i32]
    L.epsgrad_plan_set_pdl.argtypes = [vp, i32]
    L.epsgrad_plan_set_tensor_cores.argtypes = [vp, i32]
    L.epsgrad_plan_set_tuning.argtypes = [vp, i32, i32]
    L.epsgrad_plan_set_fused.argtypes = [vp, i32]
    L.epsgrad_plan_fused_profile.argtypes = [vp, i32, vp]
    L.epsgrad_plan_set_timeline.argtypes = [vp, i32]
    L.epsgrad_plan_read_timeline.argtypes = [vp, i32, vp, vp]
    L.epsgrad_stage_zreduce.argtypes = [vp, i32, vp, vp, vp, vp]
    L.eps_unbinarity_static.argtypes = [vp, vp, ctypes.c_float, vp, vp]
    L.epsgrad_static_scratch_partials.restype = i32
    L.epsgrad_status_string.argtypes = [i32]
    L.epsgrad_status_string.restype = ctypes.c_char_p
    L.epsgrad_version.restype = i32
    _lib = L
    return L


def status_string(status: int) -> str:
    return lib().epsgrad_status_string(int(status)).decode()


def _check(status: int, where: str) -> None:
    if status != OK:
        raise EpsgradError(status, where)


def _ptr_array(tensors: Sequence) -> ctypes.Array:
    return (ctypes.c_void_p * len(tensors))(*[t.data_ptr() for t in tensors])


class Plan:
    """epsgrad_plan_t plus its torch-allocated workspace.  Methods mirror the C entry points."""

    def __init__(self, cfg: Config, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("epsgrad needs a CUDA device (sm_100a); there is no CPU path")
        self._torch = torch
        self.cfg = cfg
        self.device = torch.device("cuda", device)
        self._h = ctypes.c_void_p()
        _check(lib().epsgrad_plan_create(ctypes.byref(cfg), device, ctypes.byref(self._h)), "epsgrad_plan_create")
        nbytes = lib().epsgrad_workspace_bytes(self._h)
        self._ws = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=self.device)
        _check(lib().epsgrad_plan_set_workspace(self._h, self._ws.data_ptr(), self._ws.numel()),
               "epsgrad_plan_set_workspace")
        self._stg = None
        self._stg_pairs = -1
        self._field_shape = None          # set_embedding: shape of the solver's arrays
        self._packed_shape = None         # set_packed_fields: shape of E_F / E_A

    def close(self) -> None:
        if getattr(self, "_h", None):
            lib().epsgrad_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- shapes
    @property
    def eps_shape(self):
        c = self.cfg
        return (c.batch, 3, c.nx, c.ny, c.nz)

    @property
    def field_shape(self):
        """shape of eps / E_F / E_A as the device entry points take them (the solver's arrays when an embedding is set)"""
        return self._field_shape or self.eps_shape

    @property
    def ctrl_shape(self):
        return (self.cfg.batch, self.cfg.mx, self.cfg.my)

    @property
    def mask_shape(self):
        c = self.cfg
        return (c.batch, c.subpixel * c.nx, c.subpixel * c.ny)

    def _stream(self) -> int:
        return self._torch.cuda.current_stream(self.device).cuda_stream

    def _c(self, C):
        t = self._torch
        assert C.is_cuda and C.dtype == t.float32 and C.is_contiguous() and tuple(C.shape) == self.ctrl_shape, \
            (C.shape, self.ctrl_shape)
        return C

    def _fields(self, EF, EA):
        t = self._torch
        assert len(EF) == len(EA) and len(EF) >= 1
        for f in list(EF) + list(EA):
            want = self._packed_shape or self.field_shape
            assert f.is_cuda and f.dtype == t.complex64 and f.is_contiguous() and tuple(f.shape) == tuple(want), (f.shape, f.dtype, want)
        return _ptr_array(EF), _ptr_array(EA)

    def _out(self, out, shape):
        t = self._torch
        if out is None:
            return t.empty(shape, dtype=t.float32, device=self.device)
        assert out.is_cuda and out.dtype == t.float32 and out.is_contiguous() and tuple(out.shape) == tuple(shape)
        return out

    # ---- options
    def set_dense_reads(self, dense: bool) -> None:
        _check(lib().epsgrad_plan_set_dense_reads(self._h, int(bool(dense))), "epsgrad_plan_set_dense_reads")

    def last_launches(self) -> int:
        return int(lib().epsgrad_plan_last_launches(self._h))

    def last_copy_bytes(self):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        _check(lib().epsgrad_plan_last_copy_bytes(self._h, ctypes.byref(a), ctypes.byref(b)), "last_copy_bytes")
        return int(a.value), int(b.value)

    def set_embedding(self, nx_full=None, ny_full=None, nz_full=None, i0=0, j0=0, k0=0) -> None:
        """eps / E_F / E_A become the solver's full arrays [B,3,nx_full,ny_full,nz_full]; no arguments: back to region-sized arrays"""
        if nx_full is None:
            _check(lib().epsgrad_plan_set_embedding(self._h, None), "epsgrad_plan_set_embedding")
            self._field_shape = None
        else:
            e = Embedding(nx_full, ny_full, nz_full, i0, j0, k0)
            _check(lib().epsgrad_plan_set_embedding(self._h, ctypes.byref(e)), "epsgrad_plan_set_embedding")
            self._field_shape = (self.eps_shape[0], 3, nx_full, ny_full, nz_full)

    def set_slab(self, x_first: int = 0, x_count: int = 0) -> None:
        """eps / E_F / E_A hold only Yee rows [x_first, x_first + x_count) of the region: [B,3,x_count,Ny,Nz]; (0, 0): off"""
        _check(lib().epsgrad_plan_set_slab(self._h, x_first, x_count), "epsgrad_plan_set_slab")
        self._field_shape = (self.eps_shape[0], 3, x_count, self.eps_shape[3], self.eps_shape[4]) if x_count > 0 else None

    def set_eps_window_only(self, enable: bool) -> None:
        """eps_forward / eps_forward_vjp rewrite only the z cells of `eps` that depend on the design (the slab window of every
        column); the array must already hold the result of one full call"""
        _check(lib().epsgrad_plan_set_eps_window_only(self._h, int(bool(enable))), "epsgrad_plan_set_eps_window_only")

    def set_packed_fields(self, enable: bool) -> None:
        """E_F / E_A as [B,3,Nx,Ny,n] complex64 holding only z cells packed_window() of every column (fields on Omega_D only)"""
        _check(lib().epsgrad_plan_set_packed_fields(self._h, int(bool(enable))), "epsgrad_plan_set_packed_fields")
        if enable:
            k0, n = self.packed_window()
            self._packed_shape = tuple(self.eps_shape[:4]) + (n,)
        else:
            self._packed_shape = None

    def packed_window(self):
        """(first z cell, number of z cells) of the packed field layout"""
        a, b = ctypes.c_int(0), ctypes.c_int(0)
        _check(lib().epsgrad_plan_packed_window(self._h, ctypes.byref(a), ctypes.byref(b)), "epsgrad_plan_packed_window")
        return int(a.value), int(b.value)

    def set_tma(self, mode) -> None:
        """0: LDGSTS field reads; 1: single-stage TMA; 2: thin persistent TMA read stream"""
        _check(lib().epsgrad_plan_set_tma(self._h, int(mode)), "epsgrad_plan_set_tma")

    def set_tensor_cores(self, mode) -> None:
        """Eq. (2) and its transpose on the tensor cores: 0 / False never, 1 / True wherever it applies, 2 where it measured faster (default)"""
        _check(lib().epsgrad_plan_set_tensor_cores(self._h, int(mode)), "epsgrad_plan_set_tensor_cores")

    def set_pdl(self, enable: bool) -> None:
        _check(lib().epsgrad_plan_set_pdl(self._h, int(bool(enable))), "epsgrad_plan_set_pdl")

    def set_bulk_stores(self, enable: bool) -> None:
        _check(lib().epsgrad_plan_set_bulk_stores(self._h, int(bool(enable))), "epsgrad_plan_set_bulk_stores")

    def set_fused(self, enable) -> None:
        """0 / False: the step as separate kernels (default); 1: one persistent dataflow kernel per call; 2: persistent 2-D chains
        beside the separate stream kernels (measurement switches: both are slower)"""
        _check(lib().epsgrad_plan_set_fused(self._h, int(enable)), "epsgrad_plan_set_fused")

    def fused_profile(self, enable: bool, read: bool = False):
        """cycle accounting of the persistent kernel: dict of per-phase busy cycles / items, wait and total CTA cycles"""
        out = (ctypes.c_uint64 * 20)() if read else None
        _check(lib().epsgrad_plan_fused_profile(self._h, int(bool(enable)), out), "epsgrad_plan_fused_profile")
        if not read:
            return None
        names = ("F1", "F2", "X", "M", "T", "Z")
        return {"busy": {n: int(out[i]) for i, n in enumerate(names)}, "items": {n: int(out[6 + i]) for i, n in enumerate(names)},
                "tickets": int(out[12]), "total": int(out[13]), "wait": int(out[14]), "release": int(out[15]), "zbegin": int(out[16]), "endsync": int(out[17]),
                "raw": [int(x) for x in out]}

    def set_tuning(self, knob: int, value: int) -> None:
        _check(lib().epsgrad_plan_set_tuning(self._h, int(knob), int(value)), "epsgrad_plan_set_tuning")

    def set_host_direct(self, mode) -> None:
        """0 / False: fields staged whole; 1 / True: slab windows read in place by the kernel; 2: gathered by the copy engine"""
        _check(lib().epsgrad_plan_set_host_direct(self._h, int(mode)), "epsgrad_plan_set_host_direct")

    def set_overlap(self, enable: bool) -> None:
        _check(lib().epsgrad_plan_set_overlap(self._h, int(bool(enable))), "epsgrad_plan_set_overlap")

    def set_timeline(self, enable: bool) -> None:
        _check(lib().epsgrad_plan_set_timeline(self._h, int(bool(enable))), "epsgrad_plan_set_timeline")

    def read_timeline(self):
        """[(name, ns since the first stamp)] of the last call (synchronises the device)"""
        ns = (ctypes.c_uint64 * 48)()
        names = (ctypes.c_char_p * 48)()
        n = lib().epsgrad_plan_read_timeline(self._h, 48, ns, names)
        _check(min(n, 0), "epsgrad_plan_read_timeline")
        return [(names[i].decode(), int(ns[i]) - int(ns[0])) for i in range(n)]

    def set_profiling(self, enable: bool) -> None:
        _check(lib().epsgrad_plan_set_profiling(self._h, int(bool(enable))), "epsgrad_plan_set_profiling")

    def last_kernel_times(self):
        """[(kernel name, ms)] of the last call (blocks until its events have completed)."""
        ms = (ctypes.c_float * 24)()
        names = (ctypes.c_char_p * 24)()
        n = lib().epsgrad_plan_last_kernel_times(self._h, 24, ms, names)
        if n < 0:
            raise EpsgradError(n, "epsgrad_plan_last_kernel_times")
        return [(names[i].decode(), float(ms[i])) for i in range(n)]

    # ---- hot path (device tensors)
    def eps_forward(self, C, beta: float, out=None):
        eps = self._out(out, self.field_shape)
        _check(lib().eps_forward(self._h, self._c(C).data_ptr(), beta, eps.data_ptr(), self._stream()), "eps_forward")
        return eps

    def eps_vjp_beta(self, C, beta: float, EF: Sequence, EA: Sequence, out=None):
        """(dF/dC [B,Mx,My], dF/dbeta [B])"""
        pf, pa = self._fields(EF, EA)
        g = self._out(out, self.ctrl_shape)
        db = self._torch.empty(self.ctrl_shape[0], dtype=self._torch.float32, device=self.device)
        _check(lib().eps_vjp_beta(self._h, self._c(C).data_ptr(), beta, len(EF), pf, pa, g.data_ptr(), db.data_ptr(),
                                  self._stream()), "eps_vjp_beta")
        return g, db

    def unbinarity_static(self, phi, beta: float, out=None):
        """u(beta) [B] of a centred filter output the caller holds (stage_filter), partial sums in the library's static device
        array: no workspace, no allocation inside the call (`out` given).  Limit: B * ceil(mask pixels / 4096) <= 4096."""
        t = self._torch
        assert phi.is_cuda and phi.dtype == t.float32 and phi.is_contiguous() and tuple(phi.shape) == self.mask_shape, (phi.shape, self.mask_shape)
        u = out if out is not None else t.empty(self.ctrl_shape[0], dtype=t.float32, device=self.device)
        assert u.is_cuda and u.dtype == t.float32 and u.is_contiguous() and u.numel() == self.ctrl_shape[0]
        rc = lib().eps_unbinarity_static(self._h, phi.data_ptr(), beta, u.data_ptr(), self._stream())
        if rc == EUNSUPPORTED:
            raise EpsgradError(rc, "eps_unbinarity_static (morphological filters on, or B * ceil(mask pixels / 4096) exceeds the static "
                                   f"scratch of {lib().epsgrad_static_scratch_partials()} partial sums)")
        _check(rc, "eps_unbinarity_static")
        return u

    def unbinarity(self, C, beta: float):
        """u(beta) [B]: mean over the design mask of 4 rho (1 - rho) (S20)"""
        u = self._torch.empty(self.ctrl_shape[0], dtype=self._torch.float32, device=self.device)
        _check(lib().eps_unbinarity(self._h, self._c(C).data_ptr(), beta, u.data_ptr(), self._stream()), "eps_unbinarity")
        return u

    def eps_vjp(self, C, beta: float, EF: Sequence, EA: Sequence, out=None):
        pf, pa = self._fields(EF, EA)
        g = self._out(out, self.ctrl_shape)
        _check(lib().eps_vjp(self._h, self._c(C).data_ptr(), beta, len(EF), pf, pa, g.data_ptr(), self._stream()),
               "eps_vjp")
        return g

    def eps_forward_vjp(self, C, beta: float, EF: Sequence, EA: Sequence, eps_out=None, grad_out=None):
        pf, pa = self._fields(EF, EA)
        eps = self._out(eps_out, self.field_shape)
        g = self._out(grad_out, self.ctrl_shape)
        _check(lib().eps_forward_vjp(self._h, self._c(C).data_ptr(), beta, len(EF), pf, pa, eps.data_ptr(),
                                     g.data_ptr(), self._stream()), "eps_forward_vjp")
        return eps, g

    # ---- the same on host (CPU, ideally pinned) tensors; outputs are written asynchronously:
    # synchronise the stream before reading them
    def eps_forward_vjp_host(self, C, beta: float, EF: Sequence, EA: Sequence, eps_out, grad_out):
        t = self._torch
        n = len(EF) if grad_out is not None else 0
        if self._stg is None or self._stg_pairs < n:
            nbytes = lib().epsgrad_staging_bytes(self._h, n)
            self._stg = t.empty(nbytes, dtype=t.uint8, device=self.device)
            self._stg_pairs = n
            _check(lib().epsgrad_plan_set_staging(self._h, self._stg.data_ptr(), nbytes), "epsgrad_plan_set_staging")
        for x in [C, *EF, *EA] + [o for o in (eps_out, grad_out) if o is not None]:
            assert not x.is_cuda and x.is_contiguous()
        pf, pa = _ptr_array(EF), _ptr_array(EA)
        _check(lib().eps_forward_vjp_host(
            self._h, C.data_ptr(), beta, len(EF), pf, pa,
            eps_out.data_ptr() if eps_out is not None else None,
            grad_out.data_ptr() if grad_out is not None else None, self._stream()), "eps_forward_vjp_host")

    # ---- stage taps
    def stage_filter(self, C):
        out = self._out(None, self.mask_shape)
        _check(lib().epsgrad_stage_filter(self._h, self._c(C).data_ptr(), out.data_ptr(), self._stream()),
               "epsgrad_stage_filter")
        return out

    def stage_eps2d(self, C, beta: float):
        c = self.cfg
        out = self._out(None, (c.batch, 3, c.nx, c.ny))
        _check(lib().epsgrad_stage_eps2d(self._h, self._c(C).data_ptr(), beta, out.data_ptr(), self._stream()),
               "epsgrad_stage_eps2d")
        return out

    def stage_zreduce(self, EF: Sequence, EA: Sequence):
        c = self.cfg
        pf, pa = self._fields(EF, EA)
        out = self._out(None, (c.batch, 5, c.nx, c.ny))
        _check(lib().epsgrad_stage_zreduce(self._h, len(EF), pf, pa, out.data_ptr(), self._stream()),
               "epsgrad_stage_zreduce")
        return out
