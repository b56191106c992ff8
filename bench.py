#!/usr/bin/env python
"""bench.py -- eps forward+VJP throughput (Yee-cells/s) and HBM roofline fraction on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config paper] [--impl ours|reference]

A step is one pass of the whole hot path -- eps_forward_vjp: filter, 2-D chain, z-extrusion (eps stores),
Eq. (1) z-reduction (field reads), mask cotangent, transposed filter -- over one batch of
synthetic input (BASELINE.json configs[1] "paper": 250x250 controls -> 500x500x64 Yee cells,
one field pair) that is already resident in HBM.  Field buffers rotate over 3 sets and eps
(192 MB > L2) is rewritten every step, so no step finds its inputs in L2.
One JSON line on stdout (rank 0); see DESIGN.md section 7 for every key.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "eps forward+VJP Yee-cells/s and achieved HBM GB/s vs B200 peak (1 GPU)"
UNIT = "Yee-cells/s"
N_SETS = 3                         # rotating field sets of the paper-scale workloads; see n_sets()


def n_sets(w) -> int:
    """Field sets to rotate over: 3 while they are small enough to matter for L2 (126 MB) and to fit HBM easily; the big
    configs (Large: 24.6 GB, Wide batch: 51.5 GB of fields per set) exceed L2 a hundredfold on their own: one set."""
    return N_SETS if w.cells * 48 * w.n_pairs * N_SETS < 24e9 else 1


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons via NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.002):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.max_mhz = index, period_s, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            pass

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def visible_device_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            pass
    return local_rank


def zreduce_sector_bytes(w, n_pairs: int) -> int:
    """Algorithmic bytes of the Eq. (1) field read: the 32-byte sectors of every z column that hold
    cells with d eps/dC != 0 (x,y: wxy_k > 0; z: wz_k > 0), E_F and E_A, all pairs."""
    import math

    kxy0, kxy1 = int(math.floor(w.z_lo)), int(math.ceil(w.z_hi)) - 1
    kz0, kz1 = int(math.floor(w.z_lo - 0.5)), int(math.ceil(w.z_hi - 0.5)) - 1
    kxy0, kz0 = max(kxy0, 0), max(kz0, 0)
    kxy1, kz1 = min(kxy1, w.nz - 1), min(kz1, w.nz - 1)
    sec = lambda a, b: (b // 4 - a // 4 + 1) * 32          # 4 complex64 cells per 32-byte sector
    per_column = 2 * sec(kxy0, kxy1) + sec(kz0, kz1)
    return w.batch * w.nx * w.ny * per_column * 2 * n_pairs


def crop(w, mx, my):
    """workload w on an mx x my control grid (same cells per control pixel, also when that is not an integer)"""
    from dataclasses import replace
    if w.nx_cells > 0:
        return replace(w, mx=mx, my=my, batch=1, nx_cells=max(mx, round(mx * w.nx_cells / w.mx)), ny_cells=max(my, round(my * w.ny_cells / w.my)))
    return replace(w, mx=mx, my=my, batch=1)


def oracle_cfg(w, mx=None, my=None):
    import oracle as O
    mx, my = mx or w.mx, my or w.my
    wc = crop(w, mx, my)
    return O.OracleConfig(mx=mx, my=my, nx=wc.nx, ny=wc.ny, nz=w.nz, z_lo=w.z_lo, z_hi=w.z_hi,
                          s=w.subpixel, filter_kind=w.filter_kind, radius=w.radius, sigma=w.sigma or 1.0, eta=w.eta,
                          eps_core=w.eps_core, eps_clad=w.eps_clad, delta=w.normal_delta,
                          morph_diam=w.morph_diameter, morph_alpha=w.morph_alpha)


def oracle_step_inputs(w, mx, my):
    from paper_2505_03352_b200 import workloads as W
    ws = crop(w, mx, my)
    C = W.make_C(ws)[0]
    EF = [W.make_field(ws, p, 0) for p in range(w.n_pairs)]
    EA = [W.make_field(ws, p, 1) for p in range(w.n_pairs)]
    return ws, C, EF, EA


def oracle_step(cfg, C, betas, EF, EA, acc=None):
    import oracle as O
    for beta in betas:
        t0 = time.perf_counter()
        O.forward(cfg, C, beta)
        t1 = time.perf_counter()
        O.vjp(cfg, C, beta, EF, EA)
        t2 = time.perf_counter()
        if acc is not None:
            acc["forward"] += t1 - t0
            acc["vjp"] += t2 - t1


def time_oracle(w, budget_s: float, steps: int, warmup: int, split: bool = False):
    """Time the float64 oracle (as it stands) on a crop of workload w sized so that
    (steps + warmup) steps take about budget_s.  Returns (cells/s, seconds/step, sample text, threads) and, with
    split, the forward-only and VJP-only cells/s (O.vjp recomputes the forward chain it differentiates)."""
    import oracle as O
    # calibrate on a 32x32-control crop
    ws, C, EF, EA = oracle_step_inputs(w, min(32, w.mx), min(32, w.my))
    cfg = oracle_cfg(w, ws.mx, ws.my)
    oracle_step(cfg, C, w.betas, EF, EA)
    t0 = time.perf_counter()
    oracle_step(cfg, C, w.betas, EF, EA)
    rate = ws.nx * ws.ny * ws.nz / (time.perf_counter() - t0)          # cells/s, rough
    target_cells = rate * budget_s / max(1, steps + warmup)
    full = w.nx * w.ny * w.nz
    if target_cells >= full:
        mx, my = w.mx, w.my
    else:
        f = (target_cells / full) ** 0.5
        mx, my = max(16, int(w.mx * f)), max(16, int(w.my * f))
    ws, C, EF, EA = oracle_step_inputs(w, mx, my)
    cfg = oracle_cfg(w, mx, my)
    for _ in range(warmup):
        oracle_step(cfg, C, w.betas, EF, EA)
    acc = {"forward": 0.0, "vjp": 0.0}
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_step(cfg, C, w.betas, EF, EA, acc)
    dt = (time.perf_counter() - t0) / steps
    cells = ws.nx * ws.ny * ws.nz                                        # one design of the batch
    sample = (f"{steps} step(s) of forward+VJP on a {mx}x{my}-control crop ({ws.nx}x{ws.ny}x{ws.nz} Yee cells, "
              f"{w.n_pairs} pair(s), {len(w.betas)} beta) of '{w.name}'"
              + (" = the full workload" if (mx, my, w.batch) == (w.mx, w.my, 1) else ""))
    if split:
        parts = {k: cells * len(w.betas) * steps / v for k, v in acc.items()}
        return cells / dt, dt, sample, O.num_threads(), parts
    return cells / dt, dt, sample, O.num_threads()


def base_line(w, args, n_gpus):
    return {
        "metric": METRIC, "unit": UNIT, "n_gpus": n_gpus, "steps": args.steps, "warmup": args.warmup,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "data": "synthetic",
        "config": {"workload": f"{w.name}: C {w.batch}x{w.mx}x{w.my} -> Yee {w.nx}x{w.ny}x{w.nz}, "
                               f"{'conic' if w.filter_kind == 0 else 'gaussian'} R={w.radius:g}, beta={list(w.betas)}, "
                               f"{w.n_pairs} field pair(s), slab [{w.z_lo},{w.z_hi}]"
                               + (f", morphological filters d={w.morph_diameter:g} cells alpha={w.morph_alpha:g}" if w.morph_diameter > 0 else ""),
                   "per_gpu": "one such design batch per GPU (independent designs, no collective)",
                   "launch": "CUDA graph replay of eps_forward_vjp (captured through the C ABI)" if getattr(args, "graph", True)
                             else "eager eps_forward_vjp calls",
                   "cache": f"field buffers rotate over {n_sets(w)} set(s); eps ({w.cells * 12 / 1e6:.0f} MB) rewritten every step"},
    }


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    val, dt, sample, threads = time_oracle(w, 150.0, args.steps, args.warmup)
    line = base_line(w, args, args.gpus)
    line.update({"impl": "reference", "value": val, "ms_per_step": dt * 1e3, "dtype": "f64", "scaling": "weak",
                 "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
                 "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                 "gpu_launches": 0})
    print(json.dumps(line), flush=True)


def run_ours(args, w):
    import torch
    from paper_2505_03352_b200 import binding as B
    from paper_2505_03352_b200 import sharding
    from paper_2505_03352_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the epsgrad path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    from dataclasses import replace
    mode = args.shard
    shard = sharding.make_shard(mode, w, rank, world)
    plan = B.Plan(B.config_of(shard["sub"]), local)
    if shard["slab"] is not None:
        plan.set_slab(shard["slab"]["x_first"], shard["slab"]["x_count"])
    # designs: every rank draws its own designs; pairs / xslab: ONE design, the same C on every rank
    C = torch.from_numpy(W.make_C(replace(w, index=w.index + 1000 * rank) if mode == "designs" else w)).to(dev)
    C_part = C if shard["slab"] is None else C[:, shard["slab"]["e0"]:shard["slab"]["e1"]].contiguous()
    gen = torch.Generator(device=dev)
    gen.manual_seed(1234 + rank)
    shape = plan.field_shape                                   # this rank's rows of eps / E_F / E_A
    n_my = len(shard["pairs"])                                 # this rank's field pairs

    def field():
        return torch.view_as_complex(torch.randn(*shape, 2, device=dev, dtype=torch.float32, generator=gen))
    NS = n_sets(w)
    EF = [[field() for _ in range(n_my)] for _ in range(NS)]
    EA = [[field() for _ in range(n_my)] for _ in range(NS)]
    eps = torch.empty(shape, dtype=torch.float32, device=dev)
    grad = torch.empty((w.batch, w.mx, w.my), dtype=torch.float32, device=dev)         # the whole design's dF/dC
    grad_part = grad if shard["slab"] is None else torch.empty(plan.ctrl_shape, dtype=torch.float32, device=dev)

    def compute(Cp, EFs, EAs, beta):
        if n_my == 0:                                          # more ranks than pairs: forward only, nothing to add
            plan.eps_forward(Cp, beta, eps)
            return eps, None
        plan.eps_forward_vjp(Cp, beta, EFs, EAs, eps, grad_part)
        return eps, grad_part

    def eager_step(i):
        s = i % NS
        for beta in w.betas:
            sharding.shard_step(shard, compute, C, (EF[s], EA[s]), beta, grad, C_part=C_part)

    if mode != "designs" and world > 1:
        args.graph = False                                     # the gradient all-reduce (NCCL) runs between the library calls

    # One CUDA graph per buffer set, captured through the C ABI (the calls enqueue only kernels and
    # fork/join events, so they are capturable); replaying removes the host's launch cost from the step.
    graphs = None
    if args.graph:
        for i in range(3):
            eager_step(i)
        torch.cuda.synchronize()
        graphs = []
        for sset in range(NS):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                eager_step(sset)
            graphs.append(g)

    def step(i):
        if graphs is not None:
            graphs[i % NS].replay()
        else:
            eager_step(i)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    eager_step(0)
    launches_per_step = plan.last_launches() * len(w.betas)
    for i in range(max(args.warmup, 3)):
        step(i)
    sampler = ClockSampler(visible_device_index(local))
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(args.steps):
        step(i)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ms_total = sharding.max_over_ranks(ms_total, device=dev)
    cells_step = w.cells * len(w.betas)
    # designs: every rank processed its own cells (weak scaling); pairs / xslab: the ranks shared ONE design (strong scaling)
    value = sharding.job_throughput(cells_step, args.steps, ms_total, world if mode == "designs" else 1)

    if mode != "designs":
        # ONE design shared by the ranks: whole-job throughput with the gradient exchange inside the timed region.  The
        # per-call breakdown, the per-kernel roofline and the host-buffer leg are those of the default (--shard designs) line.
        if rank == 0:
            peak, peak_src = measured_peak_gbs()
            step_ms = ms_total / args.steps
            step_bytes = (w.cells * 12 * world if mode == "pairs" else w.cells * 12) * len(w.betas) \
                + zreduce_sector_bytes(w, w.n_pairs) * len(w.betas)
            line = base_line(w, args, world)
            line["config"]["per_gpu"] = {
                "pairs": f"field pairs of ONE design over the ranks ({w.n_pairs} pairs / {world} ranks); every rank runs the forward "
                         f"chain and writes its own eps; one all-reduce (sum) of dF/dC, {w.batch * w.mx * w.my * 4} bytes, per step",
                "xslab": f"x-slabs of ONE design over the ranks (halo {sharding.slab_halo_cells(w.radius, w.morph_diameter)} cells); "
                         f"eps and fields hold the own rows only; one all-reduce (sum) of dF/dC, {w.batch * w.mx * w.my * 4} bytes, per step",
            }[mode]
            if not args.graph:
                line["config"]["launch"] = "eager eps_forward_vjp calls (the NCCL all-reduce runs between them)"
            line.update({"value": value, "ms_per_step": step_ms, "dtype": "f32", "scaling": "strong", "shard": mode,
                         "clocks": clocks, "gpu_launches": launches_per_step * args.steps,
                         "e2e": {"skipped": "measured by the default line (--shard designs)"},
                         "roofline": {"bound": "hbm", "kernel": "step", "unit": "GB/s", "peak": peak, "peak_source": peak_src,
                                      "algorithmic_bytes": step_bytes, "achieved": step_bytes / (step_ms * 1e-3) / 1e9,
                                      "frac": step_bytes / (step_ms * 1e-3) / 1e9 / (peak * world), "traffic": None,
                                      "note": "eps stores (every rank's) + touched field sectors of the whole job over the step, "
                                              "against the peak of all ranks' HBM"}})
            print(json.dumps(line), flush=True)
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- the three calls of the ABI, each timed repetition by repetition (median of >= 20 repetitions):
    # forward (eps_forward), vjp (eps_vjp), forward_vjp (the step above).  One CUDA graph per call and buffer set, one event
    # pair per repetition.
    def per_rep_ms(fn, reps):
        gs = None
        if args.graph:
            gs = []
            for sset in range(NS):
                fn(sset)
            torch.cuda.synchronize()
            for sset in range(NS):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    fn(sset)
                gs.append(g)
        run = (lambda i: gs[i % NS].replay()) if gs is not None else (lambda i: fn(i % NS))
        for i in range(3):
            run(i)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(reps + 1)]
        torch.cuda.synchronize()
        ev[0].record()
        for i in range(reps):
            run(i)
            ev[i + 1].record()
        torch.cuda.synchronize()
        return sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(reps))

    def mode_stats(ts, n_calls):
        med = ts[len(ts) // 2]
        return {"ms_median": med, "ms_min": ts[0], "ms_mean": sum(ts) / len(ts), "reps": len(ts),
                "cells_per_s": w.cells * n_calls / (med * 1e-3)}

    reps = max(20, min(args.steps, 200))

    def fwd_call(s):
        for beta in w.betas:
            plan.eps_forward(C, beta, eps)

    def vjp_call(s):
        for beta in w.betas:
            plan.eps_vjp(C, beta, EF[s], EA[s], grad)

    modes = {"forward": mode_stats(per_rep_ms(fwd_call, reps), len(w.betas)),
             "vjp": mode_stats(per_rep_ms(vjp_call, reps), len(w.betas)),
             "forward_vjp": mode_stats(per_rep_ms(eager_step, reps), len(w.betas))}

    # ---- per-kernel durations, live, with CUDA events on the launching stream (the library's hook: one event after
    # each kernel, serial schedule).  A ~150 us spin kernel is enqueued ahead of every profiled step so that the host has
    # queued the whole step before the GPU reaches it: the events then bracket kernel execution, not host launch gaps.
    def kernel_times():
        plan.set_profiling(True)
        acc, n_prof = {}, min(args.steps, 100)
        spin = int(150e-6 * 1.9e9)
        for i in range(n_prof):
            s = i % NS
            for beta in w.betas:
                torch.cuda._sleep(spin)
                plan.eps_forward_vjp(C, beta, EF[s], EA[s], eps, grad)
                for name, ms in plan.last_kernel_times():
                    acc[name] = acc.get(name, 0.0) + ms
        plan.set_profiling(False)
        calls = n_prof * len(w.betas)
        return {k: v / calls for k, v in acc.items()}                   # ms per launch
    kernels = kernel_times()
    peak, peak_src = measured_peak_gbs()
    # the two HBM streams: 12 B written per Yee cell (extrude); the touched 32-byte field sectors read (zreduce)
    alg = {"extrude": w.cells * 12, "zreduce": zreduce_sector_bytes(w, w.n_pairs)}
    dom = max(alg, key=lambda k: kernels[k])

    # the field stream alone (the stage tap of the ABI), cold L2, rotating field sets, two ways of emptying L2 before each
    # repetition: a 256 MB FILL (leaves L2 full of dirty lines, as the eps stores of the previous step do: the stream then
    # also pays for their write-back) and a 256 MB READ (clean lines: nothing to write back)
    flush = torch.empty(64 << 20, dtype=torch.float32, device=dev)
    flush.zero_()

    def z_alone(dirty):
        ts = []
        for i in range(min(reps, 30)):
            if dirty:
                flush.fill_(float(i))
            else:
                flush.sum()
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            plan.stage_zreduce(EF[i % NS], EA[i % NS])
            a1.record()
            torch.cuda.synchronize()
            ts.append(a0.elapsed_time(a1))
        ts.sort()
        return ts[len(ts) // 2]
    flush.sum(); flush.sum()
    z_clean_ms = z_alone(False)
    z_alone_ms = z_alone(True)

    # ---- where the kernels END inside the OVERLAPPED schedule (the per-kernel times above come from the serial one): timeline
    # stamps of the library's hook (a one-thread kernel writing %globaltimer after each kernel, on the stream it ran on), median
    # over a few eager steps, us since the step's first stamp
    plan.set_timeline(True)
    tls = []
    for i in range(8):
        plan.eps_forward_vjp(C, w.betas[-1], EF[i % NS], EA[i % NS], eps, grad)
        tl = plan.read_timeline()
        if i >= 3:
            tls.append(tl)
    plan.set_timeline(False)
    timeline = None
    if tls and all(len(t) == len(tls[0]) for t in tls):
        timeline = [[tls[0][k][0], sorted(t[k][1] for t in tls)[len(tls) // 2] / 1e3] for k in range(len(tls[0]))]

    # ---- the same step with the fields given on the design region only (epsgrad_plan_set_packed_fields: E_F / E_A hold the z
    # cells of the slab window, "restricted to Omega_D"): NOT the BASELINE layout, reported beside the headline only
    packed = None
    try:
        k0, nk = plan.packed_window()
        plan.set_packed_fields(True)
    except B.EpsgradError:
        k0 = nk = 0
    if nk > 0:
        full_EF, full_EA = EF, EA
        EF = [[f[..., k0:k0 + nk].contiguous() for f in s] for s in full_EF]
        EA = [[f[..., k0:k0 + nk].contiguous() for f in s] for s in full_EA]
        pk_bytes = sum(f.numel() * 8 for f in EF[0] + EA[0])
        pk_vjp = mode_stats(per_rep_ms(vjp_call, reps), len(w.betas))
        pk_both = mode_stats(per_rep_ms(eager_step, reps), len(w.betas))
        pk_clean, pk_dirty = z_alone(False), z_alone(True)
        pk_kernels = kernel_times()
        plan.set_packed_fields(False)
        EF, EA = full_EF, full_EA
        packed = {"window_cells": [k0, nk], "bytes_read": pk_bytes,
                  "forward_vjp_ms_median": pk_both["ms_median"], "vjp_ms_median": pk_vjp["ms_median"],
                  "cells_per_s": pk_both["cells_per_s"],
                  "zreduce_in_step_ms": pk_kernels["zreduce"],
                  "zreduce_in_step_frac": pk_bytes / (pk_kernels["zreduce"] * 1e-3) / 1e9 / measured_peak_gbs()[0],
                  "zreduce_alone_ms": pk_clean, "zreduce_alone_frac": pk_bytes / (pk_clean * 1e-3) / 1e9 / measured_peak_gbs()[0],
                  "zreduce_after_fill_ms": pk_dirty,
                  "note": "E_F / E_A as [B,3,Nx,Ny,%d]: only z cells %d..%d of every column, a dense read stream; same dF/dC bit for bit; "
                          "a different input layout from BASELINE.json's full columns, so not the headline" % (nk, k0, k0 + nk - 1)}
    # ---- eps on the design region only (epsgrad_plan_set_eps_window_only): every call after the first rewrites only the z
    # cells of the slab window of every column; with the packed fields beside it, the step a design loop runs once its eps array
    # holds the cladding.  NOT the BASELINE forward (12 B per cell written every call): beside the headline only
    window = None
    try:
        plan.set_eps_window_only(True)
        window_ok = True
    except B.EpsgradError:
        window_ok = False
    if window_ok:
        wn_fwd = mode_stats(per_rep_ms(fwd_call, reps), len(w.betas))
        wn_both = mode_stats(per_rep_ms(eager_step, reps), len(w.betas))
        wn_kernels = kernel_times()
        window = {"forward_ms_median": wn_fwd["ms_median"], "forward_vjp_ms_median": wn_both["ms_median"],
                  "extrude_in_step_ms": wn_kernels["extrude"],
                  "note": "eps_forward rewrites only the slab window of every z column (whole 32-byte sectors); the array holds the "
                          "cladding from one earlier full call; not the BASELINE forward, so not the headline"}
        if nk > 0:
            plan.set_packed_fields(True)
            full_EF, full_EA = EF, EA
            EF = [[f[..., k0:k0 + nk].contiguous() for f in s] for s in full_EF]
            EA = [[f[..., k0:k0 + nk].contiguous() for f in s] for s in full_EA]
            both = mode_stats(per_rep_ms(eager_step, reps), len(w.betas))
            plan.set_packed_fields(False)
            EF, EA = full_EF, full_EA
            window["with_packed_fields_forward_vjp_ms_median"] = both["ms_median"]
            window["with_packed_fields_cells_per_s"] = both["cells_per_s"]
        plan.set_eps_window_only(False)
        plan.eps_forward(C, w.betas[-1], eps)                  # leave a fully written eps behind
    del flush

    # DRAM bytes per launch from the committed ncu --set full capture, if it was taken on THIS build (source hash)
    traffic, traffic_note = None, "no ncu capture of this build under profiles/ (traffic.json names another source hash)"
    try:
        from paper_2505_03352_b200 import build as cuda_build
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            tj = json.load(f)
        ent = tj.get(w.name, {})
        if ent.get("src_sha16") == cuda_build.source_hash():
            traffic, traffic_note = ent.get(dom), "ncu --set full capture of this build (profiles/traffic.json)"
    except Exception:
        pass
    achieved = alg[dom] / (kernels[dom] * 1e-3) / 1e9
    dense_bytes = w.cells * 48 * w.n_pairs                              # every z cell of E_F and E_A: NOT the method's own work
    step_bytes = alg["extrude"] * len(w.betas) + alg["zreduce"] * len(w.betas)
    step_ms = ms_total / args.steps
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_note, "peak_source": peak_src,
                "algorithmic_bytes": alg[dom], "kernel_ms": kernels[dom],
                "kernel_timing": "CUDA events inside the step, serial schedule (one event after each kernel)",
                "kernels_ms": kernels,
                "others": {k: {"algorithmic_bytes": alg[k], "kernel_ms": kernels[k], "GB/s": alg[k] / (kernels[k] * 1e-3) / 1e9,
                               "frac": alg[k] / (kernels[k] * 1e-3) / 1e9 / peak} for k in alg if k != dom},
                "zreduce_alone": {"kernel_ms": z_clean_ms, "frac": alg["zreduce"] / (z_clean_ms * 1e-3) / 1e9 / peak,
                                  "how": "epsgrad_stage_zreduce alone, cold and CLEAN L2 (256 MB read before each repetition), median",
                                  "after_fill_ms": z_alone_ms, "after_fill_frac": alg["zreduce"] / (z_alone_ms * 1e-3) / 1e9 / peak,
                                  "after_fill": "the same after a 256 MB FILL: L2 full of dirty lines, as after the eps stores of the "
                                                "previous step; the difference is their write-back under the read stream"},
                "frac_dense_equiv": {"value": dense_bytes / (kernels["zreduce"] * 1e-3) / 1e9 / peak,
                                     "bytes": dense_bytes,
                                     "note": "48 B per Yee cell and pair as if every z cell were read: not the method's work "
                                             "(d eps/dC = 0 outside the slab); context for the north_star's dense reading only"},
                "step": {"algorithmic_bytes": step_bytes, "ms": step_ms, "GB/s": step_bytes / (step_ms * 1e-3) / 1e9,
                         "frac": step_bytes / (step_ms * 1e-3) / 1e9 / peak,
                         "note": "eps stores + touched field sectors over the whole overlapped step (2-D chain included)"},
                "timeline_us": timeline,
                "timeline": "end of each kernel inside the overlapped two-stream schedule (eager calls, stamps on the kernels' own streams)",
                "packed_fields": packed,
                "eps_window_only": window,
                "modes_frac": {"forward": alg["extrude"] * len(w.betas) / (modes["forward"]["ms_median"] * 1e-3) / 1e9 / peak,
                               "vjp": alg["zreduce"] * len(w.betas) / (modes["vjp"]["ms_median"] * 1e-3) / 1e9 / peak,
                               "vjp_dense_equiv": dense_bytes * len(w.betas) / (modes["vjp"]["ms_median"] * 1e-3) / 1e9 / peak}}

    # ---- end to end through the host-buffer entry point: H2D of C and the fields, D2H of eps and dF/dC
    if w.cells * 48 * w.n_pairs > 8e9:
        # the big parity configs (Large, Wide batch) would pin tens of GB of host memory and stage as much on the device:
        # the end-to-end leg is measured on the paper-scale workloads only
        e2e = {"skipped": "fields of one set exceed 8 GB; e2e is measured on the paper-scale workloads"}
    else:
        pin = lambda t: t.cpu().pin_memory()
        Ch, EFh, EAh = pin(C), [pin(f) for f in EF[0]], [pin(f) for f in EA[0]]
        eps_h = torch.empty(shape, dtype=torch.float32).pin_memory()
        grad_h = torch.empty(plan.ctrl_shape, dtype=torch.float32).pin_memory()
        n_e2e = max(1, min(args.steps, 10))

        def e2e_step():
            for beta in w.betas:
                plan.eps_forward_vjp_host(Ch, beta, EFh, EAh, eps_h, grad_h)
        for _ in range(2):
            e2e_step()
        h2d, d2h = plan.last_copy_bytes()
        barrier()
        e0.record()
        for _ in range(n_e2e):
            e2e_step()
        e1.record()
        barrier()
        ms_e2e = e0.elapsed_time(e1)
        ms_e2e = sharding.max_over_ranks(ms_e2e, device=dev)
        e2e = {"value": sharding.job_throughput(cells_step, n_e2e, ms_e2e, world), "unit": UNIT,
               "h2d_bytes_per_step": h2d * len(w.betas), "d2h_bytes_per_step": d2h * len(w.betas),
               "steps": n_e2e, "ms_per_step": ms_e2e / n_e2e}

    if rank == 0:
        line = base_line(w, args, world)
        line.update({"value": value, "ms_per_step": ms_total / args.steps, "dtype": "f32",
                     "ms_per_step_median": modes["forward_vjp"]["ms_median"], "modes": modes,
                     "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
                     "roofline": roofline})
        if world == 1:
            val, dt, sample, threads, parts = time_oracle(w, 15.0, 3, 1, split=True)
            line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                                    "forward_cells_per_s": parts["forward"], "vjp_cells_per_s": parts["vjp"]}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", default=None, help="workload name (default: paper; multiwavelength / large with --shard pairs / xslab)")
    ap.add_argument("--shard", default="designs", choices=["designs", "pairs", "xslab"],
                    help="how N ranks share the work: independent designs (default, weak scaling, no collective); the field pairs "
                         "of one design; x-slabs of one design (both strong scaling, one all-reduce of dF/dC per step)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-graph", dest="graph", action="store_false",
                    help="launch every step eagerly from Python instead of replaying a captured CUDA graph")
    args = ap.parse_args()
    from paper_2505_03352_b200 import workloads as W
    if args.config is None:
        args.config = {"designs": "paper", "pairs": "multiwavelength", "xslab": "large"}[args.shard]
    w = W.BY_NAME[args.config]
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
