"""Multi-GPU plumbing (one process per GPU, torch.distributed).  The path shards two ways
(DESIGN.md 8): independent designs of a batch -- no data-path collective at all -- and field pairs
(wavelengths / ports) of one design, whose partial gradients add: one all-reduce (sum) of dF/dC,
B*Mx*My floats (250 KB at paper scale, latency-bound).  No arithmetic of the method lives here."""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int) -> range:
    """Contiguous, balanced share of n units for `rank` of `world` (sizes differ by at most one)."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError((n, rank, world))
    base, extra = divmod(n, world)
    start = rank * base + min(rank, extra)
    return range(start, start + base + (1 if rank < extra else 0))


def sum_gradients(grad, group=None):
    """In-place all-reduce (sum) of a partial dF/dC over the ranks that hold the other field pairs."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(grad, op=dist.ReduceOp.SUM, group=group)
    return grad


def max_over_ranks(value: float, device=None, group=None) -> float:
    """Max of a per-rank scalar (device-timed milliseconds) over all ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def job_throughput(units_per_rank: int, steps: int, ms_max: float, world: int) -> float:
    """Whole-job units/s when every rank processed units_per_rank per step (weak scaling)."""
    return world * units_per_rank * steps / (ms_max * 1e-3)


def slab_halo_cells(filter_radius: float, morph_diameter: float = 0.0) -> int:
    """Yee cells of halo an x-slab needs on either side so that eps on its own rows, and their share of dF/dC, come out as in
    the undivided region: half-cell shift + Sobel ring + averages reach 3 cells, each mask pixel reaches the
    filter radius R -- and must itself sit R cells inside the slab to get the interior normaliser --, and the four morphological
    operations reach 2 d cells more."""
    import math
    return int(math.ceil(filter_radius + 3.0 + 2.0 * morph_diameter))


def slab_partition(mx: int, upsample: int, rank: int, world: int, halo_cells: int) -> dict:
    """Third way to shard: one design split along x.  Returns the control rows this rank owns [a0, a1), the rows
    its plan covers [e0, e1) (own rows plus the halo, clipped at the true borders of the region, where the plan's own border
    handling is the right one) and, in Yee rows of that plan's region, the window of the rows it owns -- the arguments of
    ``Plan.set_slab``."""
    own = shard_range(mx, rank, world)
    a0, a1 = own.start, own.stop
    h = -(-halo_cells // upsample)                     # control rows
    e0, e1 = max(0, a0 - h), min(mx, a1 + h)
    return dict(a0=a0, a1=a1, e0=e0, e1=e1, x_first=upsample * (a0 - e0), x_count=upsample * (a1 - a0))
