"""Host-side logic of the N > 1 path on CPU: world_size-2 gloo processes.  Field pairs are sharded
across ranks, each rank forms its partial dF/dC (here with the float64 oracle, the GPU being absent)
and the partials are summed with the same all-reduce helper the GPU path uses; timing is reduced
with the max-over-ranks helper bench.py uses."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2505_03352_b200 import sharding


def test_shard_range_partitions():
    for n in (0, 1, 3, 8, 17):
        for world in (1, 2, 3, 8):
            parts = [sharding.shard_range(n, r, world) for r in range(world)]
            assert [i for p in parts for i in p] == list(range(n))
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_range(4, 2, 2)


def test_job_throughput():
    assert sharding.job_throughput(16_000_000, 10, 2.0, 4) == pytest.approx(4 * 16e6 * 10 / 2e-3)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path[:0] = [root, os.path.join(root, "tests")]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle as O
    from helpers import small_cfg
    cfg = small_cfg(mx=10, my=9, nz=8, z_lo=2.25, z_hi=5.75, radius=3.0)
    rng = np.random.default_rng(7)                      # same stream on every rank: identical inputs
    C = rng.random((cfg.mx, cfg.my)).astype(np.float32)
    n_pairs = 3
    shape = (3, cfg.nx, cfg.ny, cfg.nz)
    mk = lambda: (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)
    EF, EA = [mk() for _ in range(n_pairs)], [mk() for _ in range(n_pairs)]
    mine = sharding.shard_range(n_pairs, rank, world)
    part = O.vjp(cfg, C, 8.0, [EF[p] for p in mine], [EA[p] for p in mine]) if len(mine) else np.zeros((cfg.mx, cfg.my))
    g = sharding.sum_gradients(torch.from_numpy(part.copy()))
    t = sharding.max_over_ranks(10.0 + rank)
    if rank == 0:
        full = O.vjp(cfg, C, 8.0, EF, EA)
        np.save(os.path.join(out_dir, "res.npy"), np.array([np.max(np.abs(g.numpy() - full)) / np.max(np.abs(full)), t]))
    dist.barrier()
    dist.destroy_process_group()


def test_pair_sharded_gradient_sums_to_the_full_gradient(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    err, t = np.load(tmp_path / "res.npy")
    assert err < 1e-12            # linearity of Eq. (1) in the pairs
    assert t == 11.0              # max over ranks


def _slab_worker(rank, world, port, out_dir, morph):
    """x-slab sharding with the oracle as the compute: every rank runs the chain on its own rows plus the halo."""
    import dataclasses
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path[:0] = [root, os.path.join(root, "tests")]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle as O
    from helpers import small_cfg
    cfg = small_cfg(mx=26, my=7, nz=8, z_lo=2.25, z_hi=5.75, radius=3.0, morph_diam=morph)
    u = cfg.nx // cfg.mx
    rng = np.random.default_rng(9)
    C = rng.random((cfg.mx, cfg.my)).astype(np.float32)
    shape = (3, cfg.nx, cfg.ny, cfg.nz)
    mk = lambda: (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)
    EF, EA = [mk()], [mk()]
    p = sharding.slab_partition(cfg.mx, u, rank, world, sharding.slab_halo_cells(3.0, morph))
    sub = dataclasses.replace(cfg, mx=p["e1"] - p["e0"], nx=u * (p["e1"] - p["e0"]))
    rows = slice(p["x_first"], p["x_first"] + p["x_count"])                 # own Yee rows inside the slab's region
    own = slice(u * p["a0"], u * p["a1"])                                  # the same rows in the undivided region
    eps = O.forward(sub, C[p["e0"]:p["e1"]], 8.0)[:, rows]
    # fields: only the own rows exist on this rank; every other row of the slab's region contributes nothing
    f, a = np.zeros((3, sub.nx, sub.ny, sub.nz), np.complex64), np.zeros((3, sub.nx, sub.ny, sub.nz), np.complex64)
    f[:, rows], a[:, rows] = EF[0][:, own], EA[0][:, own]
    part = np.zeros((cfg.mx, cfg.my))
    part[p["e0"]:p["e1"]] = O.vjp(sub, C[p["e0"]:p["e1"]], 8.0, [f], [a])
    g = sharding.sum_gradients(torch.from_numpy(part))
    full_eps = O.forward(cfg, C, 8.0)
    err_eps = np.max(np.abs(eps - full_eps[:, own]) / full_eps[:, own])
    worst = torch.tensor([err_eps])
    dist.all_reduce(worst, op=dist.ReduceOp.MAX)
    if rank == 0:
        full = O.vjp(cfg, C, 8.0, EF, EA)
        np.save(os.path.join(out_dir, "res.npy"), np.array([float(worst), np.max(np.abs(g.numpy() - full)) / np.max(np.abs(full))]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,morph", [(2, 0.0), (3, 0.0), (2, 1.5)])
def test_x_slabs_with_halo_reproduce_the_undivided_region(tmp_path, world, morph):
    mp.spawn(_slab_worker, args=(world, _free_port(), str(tmp_path), morph), nprocs=world, join=True)
    err_eps, err_g = np.load(tmp_path / "res.npy")
    assert err_eps < 1e-12 and err_g < 1e-12, (err_eps, err_g)


def test_slab_partition_covers_the_region_once():
    for mx, u, world, halo in [(26, 2, 3, 6), (250, 2, 8, 11), (5, 1, 4, 7), (1000, 2, 7, 15)]:
        parts = [sharding.slab_partition(mx, u, r, world, halo) for r in range(world)]
        assert parts[0]["a0"] == 0 and parts[-1]["a1"] == mx
        for p, q in zip(parts, parts[1:]):
            assert p["a1"] == q["a0"]
        for p in parts:
            h = -(-halo // u)
            assert p["e0"] == max(0, p["a0"] - h) and p["e1"] == min(mx, p["a1"] + h)
            assert p["x_first"] == u * (p["a0"] - p["e0"]) and p["x_count"] == u * (p["a1"] - p["a0"])
            assert 0 <= p["x_first"] and p["x_first"] + p["x_count"] <= u * (p["e1"] - p["e0"])


# ---- the control flow bench.py --shard runs (sharding.make_shard / shard_step), with the float64 oracle as the compute
def _oracle_compute(w_sub, slab):
    import oracle as O
    from helpers import cfg_of

    def compute(C_part, EF, EA, beta):
        cfg = cfg_of(w_sub)
        C = C_part.numpy()[0]
        eps = O.forward(cfg, C, beta)
        if slab is None:
            g = O.vjp(cfg, C, beta, [f.numpy()[0] for f in EF], [f.numpy()[0] for f in EA]) if len(EF) else None
            return torch.from_numpy(eps)[None], None if g is None else torch.from_numpy(g)[None]
        rows = slice(slab["x_first"], slab["x_first"] + slab["x_count"])
        full = (3, cfg.nx, cfg.ny, cfg.nz)
        fs, as_ = [], []
        for f, a in zip(EF, EA):                    # the rank's arrays hold its own rows only: zero elsewhere in the slab's region
            ff, aa = np.zeros(full, np.complex64), np.zeros(full, np.complex64)
            ff[:, rows], aa[:, rows] = f.numpy()[0], a.numpy()[0]
            fs.append(ff); as_.append(aa)
        g = O.vjp(cfg, C, beta, fs, as_)
        return torch.from_numpy(np.ascontiguousarray(eps[:, rows]))[None], torch.from_numpy(g)[None]
    return compute


def _bench_flow_worker(rank, world, port, out_dir, mode):
    import sys
    from dataclasses import replace
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path[:0] = [root, os.path.join(root, "tests")]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2505_03352_b200 import workloads as W
    w = replace(W.BY_NAME["multiwavelength"], mx=22, my=9, nz=8, z_lo=2.25, z_hi=5.75, radius=3.0)   # 3 pairs
    beta = 8.0
    C = torch.from_numpy(W.make_C(w))
    EF = [torch.from_numpy(W.make_field(w, p, 0))[None] for p in range(w.n_pairs)]
    EA = [torch.from_numpy(W.make_field(w, p, 1))[None] for p in range(w.n_pairs)]
    sh = sharding.make_shard(mode, w, rank, world)
    u = w.upsample
    own = slice(None) if sh["slab"] is None else slice(u * sh["slab"]["a0"], u * sh["slab"]["a1"])
    mine = ([EF[p][:, :, own].contiguous() for p in sh["pairs"]], [EA[p][:, :, own].contiguous() for p in sh["pairs"]])
    grad = torch.full((1, w.mx, w.my), float("nan"), dtype=torch.float64)
    eps = sharding.shard_step(sh, _oracle_compute(sh["sub"], sh["slab"]), C, mine, beta, grad)
    # the 1-rank result of the same flow
    one = sharding.make_shard(mode, w, 0, 1)
    grad1 = torch.empty_like(grad)
    dist_group = dist.new_group([rank])            # a world of one: the all-reduce is the identity
    eps1 = sharding.shard_step(one, _oracle_compute(one["sub"], one["slab"]), C, (EF, EA), beta, grad1, group=dist_group)
    err = torch.tensor([float((grad - grad1).abs().max() / grad1.abs().max()),
                        float(((eps - eps1[:, :, own]).abs() / eps1[:, :, own]).max())])
    dist.all_reduce(err, op=dist.ReduceOp.MAX)
    if rank == 0:
        np.save(os.path.join(out_dir, "res.npy"), err.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("mode,world", [("pairs", 2), ("xslab", 2), ("pairs", 4), ("xslab", 3), ("designs", 2)])
def test_bench_shard_flow_matches_the_one_rank_result(tmp_path, mode, world):
    """bench.py --shard pairs | xslab: partition, per-rank compute, gradient all-reduce -- against the same flow on one rank.
    pairs with 4 ranks leaves one rank without a pair."""
    mp.spawn(_bench_flow_worker, args=(world, _free_port(), str(tmp_path), mode), nprocs=world, join=True)
    err_g, err_e = np.load(tmp_path / "res.npy")
    assert err_g < 1e-12 and err_e < 1e-12, (mode, world, err_g, err_e)
