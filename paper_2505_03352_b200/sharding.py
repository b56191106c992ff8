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


# ---- one sharded step (bench.py --shard, tests/test_sharding_gloo.py).  Control flow only: `compute` does the arithmetic
# (the CUDA library in bench.py; any implementation of the chain in a test).
def make_shard(mode: str, w, rank: int, world: int) -> dict:
    """This rank's share of workload w (a workloads.Workload) under sharding `mode`:
    "designs": its own batch of designs, nothing shared (weak scaling, no collective);
    "pairs":   field pairs shard_range(n_pairs) of ONE design -- every rank runs the forward chain (its solver needs eps), reads
               only its pairs' fields, and the partial gradients are summed (one all-reduce of B*Mx*My floats);
    "xslab":   control rows [a0, a1) of ONE design plus a halo (slab_partition); eps and the fields hold only the rows it owns;
               the partial gradient covers the slab's control rows and the halo parts add into the neighbours' (all-reduce).
    Returns dict(mode, sub = the Workload of this rank's plan, pairs = range, slab = slab_partition(...) or None)."""
    from dataclasses import replace
    if mode == "designs":
        return dict(mode=mode, sub=w, pairs=range(w.n_pairs), slab=None)
    if mode == "pairs":
        mine = shard_range(w.n_pairs, rank, world)
        return dict(mode=mode, sub=replace(w, n_pairs=len(mine)), pairs=mine, slab=None)
    if mode == "xslab":
        p = slab_partition(w.mx, w.upsample, rank, world, slab_halo_cells(w.radius, w.morph_diameter))
        return dict(mode=mode, sub=replace(w, mx=p["e1"] - p["e0"]), pairs=range(w.n_pairs), slab=p)
    raise ValueError(mode)


def shard_step(shard: dict, compute, C_full, fields, beta: float, grad_full, group=None, C_part=None):
    """One forward + VJP of this rank's share, then the gradient exchange.
    C_full [B,Mx,My]: the whole design's control variables (every rank has them: 250 KB at paper scale);
    fields: (EF, EA) lists of this rank's OWN pairs on its OWN rows (what its solver produced);
    compute(C_part, EF, EA, beta) -> (eps_part, grad_part [B, rows of C_part, My]);
    grad_full: output [B,Mx,My], overwritten with the sum over the ranks;
    C_part: this rank's rows of C_full if the caller has cut them out already (C does not change within a step).
    Returns eps_part (this rank's eps: the whole region, or its rows of it)."""
    EF, EA = fields
    p = shard["slab"]
    if C_part is None:
        C_part = C_full if p is None else C_full[:, p["e0"]:p["e1"]].contiguous()
    eps_part, grad_part = compute(C_part, EF, EA, beta)
    if shard["mode"] == "designs":
        if grad_part is not grad_full:
            grad_full.copy_(grad_part)
        return eps_part
    if p is None:
        if grad_part is None:                       # a rank without pairs adds nothing
            grad_full.zero_()
        elif grad_part is not grad_full:
            grad_full.copy_(grad_part)
    else:
        grad_full.zero_()
        grad_full[:, p["e0"]:p["e1"]].copy_(grad_part)
    sum_gradients(grad_full, group)
    return eps_part
