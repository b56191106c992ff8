"""CPU-only checks of the boundary: libepsgrad.so builds (nvcc cross-compiles sm_100a without a
GPU), loads, exports every function include/epsgrad.h declares, validates configurations
on the host, and fails loudly -- not with a CPU fallback -- when there is no CUDA device."""
import ctypes
import os
import re

import pytest

from paper_2505_03352_b200 import binding as B
from paper_2505_03352_b200 import build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "epsgrad.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b([A-Za-z_][A-Za-z0-9_]*)\s*\(", src)
    return sorted({n for n in names if n.startswith(("eps_", "epsgrad_"))})


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    decl = declared_functions()
    assert len(decl) >= 15 and "eps_forward" in decl and "eps_vjp" in decl and "eps_forward_vjp" in decl
    for name in decl:
        assert hasattr(L, name), f"{name} declared in epsgrad.h but not exported"
    assert sorted(B.EXPORTS) == decl
    assert B.lib().epsgrad_version() >= 100


def test_status_strings():
    for st in (B.OK, B.EINVAL, B.EUNSUPPORTED, B.ENOWORKSPACE, B.ECUDA, B.ENOMEM):
        assert B.status_string(st) and B.status_string(st) != "unknown status"
    assert B.status_string(-99) == "unknown status"


def test_config_struct_layout_matches_header():
    # 10 int32 then 10 doubles, no padding
    assert ctypes.sizeof(B.Config) == 10 * 4 + 10 * 8
    assert B.Config.nx_cells.offset == 32 and B.Config.z_lo.offset == 40 and B.Config.normal_delta.offset == 40 + 7 * 8


def test_host_side_validation_and_no_cpu_fallback():
    import torch
    L = B.lib()
    h = ctypes.c_void_p()
    bad = [
        B.make_config(mx=8, my=8, nz=8, z_lo=3.0, z_hi=2.0),                  # z_hi <= z_lo
        B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, subpixel=3),      # odd subpixel
        B.make_config(mx=0, my=8, nz=8, z_lo=2.0, z_hi=5.0),
        B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, filter_radius=-1.0),
        B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, eps_clad=0.0),
        B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, filter_kind=7),
        B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, normal_delta=0.0),    # n^2 = 0/0 on flat cells
        B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, normal_delta=1e-40),  # denormal: flushed to 0 on the device
        B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, eta=float("nan")),
    ]
    for cfg in bad:
        assert L.epsgrad_plan_create(ctypes.byref(cfg), 0, ctypes.byref(h)) == B.EINVAL
    for cfg in (B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, upsample=5),
                B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, subpixel=10)):
        assert L.epsgrad_plan_create(ctypes.byref(cfg), 0, ctypes.byref(h)) == B.EUNSUPPORTED
    for cfg in (B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, nx_cells=20),                 # only one of the two cell counts
                B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, nx_cells=7, ny_cells=20),     # fewer cells than control pixels
                B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0, nx_cells=-3, ny_cells=20)):
        assert L.epsgrad_plan_create(ctypes.byref(cfg), 0, ctypes.byref(h)) == B.EINVAL
    assert L.epsgrad_plan_create(None, 0, ctypes.byref(h)) == B.EINVAL
    if not torch.cuda.is_available():
        good = B.make_config(mx=8, my=8, nz=8, z_lo=2.0, z_hi=5.0)
        assert L.epsgrad_plan_create(ctypes.byref(good), 0, ctypes.byref(h)) == B.ECUDA
        with pytest.raises(RuntimeError):
            B.Plan(good)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2505_03352_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "epsgrad_oracle" not in text, f


def test_abtest_module_needs_a_gpu_and_names_its_modes(capsys):
    """`python -m paper_2505_03352_b200.abtest`: usage without arguments; no CPU path behind any of its modes."""
    import torch
    from paper_2505_03352_b200 import abtest
    assert abtest.main([]) == 2
    text = capsys.readouterr().out
    for mode in ("streams", "pdl", "fused", "tc"):
        assert mode in text
    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError):
            abtest.main(["pdl", "tiny"])
