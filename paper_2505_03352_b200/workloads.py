"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the float64 oracle, and
therefore holds none of the method's arithmetic: it only names the workloads
(shapes, filter, beta, slab, seeds) and
draws the control variables C and the complex64 fields E_F, E_A from numpy's
PCG64.  The paper measures on no public dataset; every input is synthetic.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    index: int                  # position in BASELINE.json "configs"; also the seed (S16)
    batch: int
    mx: int
    my: int
    nz: int
    z_lo: float
    z_hi: float
    filter_kind: int            # 0 conic, 1 Gaussian with per-axis truncation (S11)
    radius: float               # Yee cells
    sigma: float                # Yee cells (Gaussian only)
    betas: tuple                # one run per beta (S12)
    n_pairs: int
    c_kind: str                 # "uniform" | "blurred" (S13)
    upsample: int = 2           # Yee cells per control pixel
    subpixel: int = 2           # mask pixels per Yee cell (S4)
    eta: float = 0.5
    eps_core: float = 12.11     # Si
    eps_clad: float = 2.085     # SiO2
    normal_delta: float = 1e-8  # guard of the normals (S6): above float32 Sobel-difference noise^2
    morph_diameter: float = 0.0 # d of Eqs. (4)-(5) in Yee cells; 0 = morphological filters off (as in Fig. 4)
    morph_alpha: float = 20.0   # App. B
    nx_cells: int = 0           # Yee cells of the design region when they are not upsample * mx (Fig. 4: 210 cells on 36 controls)
    ny_cells: int = 0

    @property
    def nx(self) -> int:
        return self.nx_cells if self.nx_cells > 0 else self.upsample * self.mx

    @property
    def ny(self) -> int:
        return self.ny_cells if self.ny_cells > 0 else self.upsample * self.my

    @property
    def cells(self) -> int:
        return self.batch * self.nx * self.ny * self.nz

    @property
    def field_shape(self) -> tuple:
        return (self.batch, 3, self.nx, self.ny, self.nz)


CONFIGS = (
    Workload("tiny", 0, 1, 32, 32, 16, 6.25, 9.75, 0, 4.0, 0.0, (8.0,), 1, "uniform"),
    Workload("paper", 1, 1, 250, 250, 64, 28.25, 35.75, 0, 8.0, 0.0, (16.0,), 1, "uniform"),
    Workload("multiwavelength", 2, 1, 250, 250, 64, 28.25, 35.75, 0, 8.0, 0.0, (4.0, 16.0, 64.0), 3, "uniform"),
    Workload("large", 3, 1, 1000, 1000, 64, 28.25, 35.75, 0, 12.0, 0.0, (32.0,), 1, "blurred"),
    Workload("widebatch", 4, 8, 1024, 1024, 32, 14.25, 17.75, 1, 32.0, 10.0, (8.0,), 1, "uniform"),
)
# Not a BASELINE.json config: the paper-scale workload with the morphological filters on (minimum feature size d = 4 cells
# = 100 nm at the 25 nm cells of Fig. 4, alpha = 20 of App. B), for `bench.py --config paper_morph`.
# "fig4": the geometry of the paper's own demonstration (Fig. 4): 36 x 36 control variables on a design region of 210 x 210
# cells (5.83 cells per control pixel), 64 cells in z, two wavelengths = two field pairs; filter radius and beta are not printed:
# R = 8 cells, beta = 16 as at paper scale.
EXTRA = (
    Workload("paper_morph", 1, 1, 250, 250, 64, 28.25, 35.75, 0, 8.0, 0.0, (16.0,), 1, "uniform", morph_diameter=4.0),
    Workload("fig4", 5, 1, 36, 36, 64, 28.25, 35.75, 0, 8.0, 0.0, (16.0,), 2, "uniform", nx_cells=210, ny_cells=210),
)
BY_NAME = {w.name: w for w in CONFIGS + EXTRA}


def make_C(w: Workload) -> np.ndarray:
    """Control variables [B,Mx,My] float32, seed = config index (S16)."""
    rng = np.random.default_rng(w.index)
    if w.c_kind == "uniform":
        return rng.random((w.batch, w.mx, w.my), dtype=np.float32)
    if w.c_kind == "blurred":
        # S13: uniform field blurred in float64 (sigma = 6 control pixels, truncated at
        # 4 sigma, reflect border), rescaled affinely to [0,1], cast to fp32.
        from scipy.ndimage import gaussian_filter
        out = np.empty((w.batch, w.mx, w.my), dtype=np.float32)
        for b in range(w.batch):
            x = gaussian_filter(rng.random((w.mx, w.my)), sigma=6.0, mode="reflect", truncate=4.0)
            out[b] = ((x - x.min()) / (x.max() - x.min())).astype(np.float32)
        return out
    raise ValueError(w.c_kind)


_CHUNK = 1 << 24           # floats per independently seeded chunk (part of the recipe)


def make_field(w: Workload, pair: int, which: int, design: int = 0, out: np.ndarray | None = None) -> np.ndarray:
    """One design's E_F (which=0) or E_A (which=1) of field pair `pair`:
    complex64 [3,Nx,Ny,Nz], real and imaginary parts i.i.d. N(0,1).
    Chunk c of 2^24 floats is drawn from PCG64 seeded [index, pair, which, design, c]
    (chunks are filled by a thread pool; the result does not depend on the thread count)."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    shape = (3, w.nx, w.ny, w.nz)
    if out is None:
        out = np.empty(shape, dtype=np.complex64)
    assert out.shape == shape and out.dtype == np.complex64 and out.flags.c_contiguous
    flat = out.view(np.float32).reshape(-1)

    def fill(c: int) -> None:
        rng = np.random.default_rng([w.index, pair, which, design, c])
        rng.standard_normal(out=flat[c * _CHUNK:(c + 1) * _CHUNK], dtype=np.float32)

    n = (flat.size + _CHUNK - 1) // _CHUNK
    if n == 1:
        fill(0)
    else:
        with ThreadPoolExecutor(max_workers=min(n, len(os.sched_getaffinity(0)))) as ex:
            list(ex.map(fill, range(n)))
    return out


def small_variant(w: Workload, mx: int, my: int, batch: int | None = None) -> Workload:
    """Same recipe on a smaller control grid (parity cases the oracle finishes in seconds)."""
    from dataclasses import replace
    return replace(w, mx=mx, my=my, batch=w.batch if batch is None else batch)
