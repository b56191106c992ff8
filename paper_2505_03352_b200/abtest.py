"""A/B timing of a plan's measurement switches on one GPU: which variant of a kernel or of the schedule
is faster on THIS size.  Every variant computes the same path; the switches are the ones `include/epsgrad.h` exports.

    python -m paper_2505_03352_b200.abtest streams [workload]     # eps store stream / field read stream variants
    python -m paper_2505_03352_b200.abtest pdl [workload ...]     # programmatic dependent launch on / off
    python -m paper_2505_03352_b200.abtest fused [workload]       # separate kernels / one persistent dataflow kernel / 2-D chains only
    python -m paper_2505_03352_b200.abtest tc [mx:R ...]          # FFMA stencils against the tensor-core filters (+ cycle accounting)
    python -m paper_2505_03352_b200.abtest replay [workload] [knob=value ...]   # graph replays of the step: a target for ncu

One JSON line per variant: step time of a replayed CUDA graph (us, mean of `steps` replays over rotating field sets), the
event-timed kernels of the serial schedule, and whether the results equal the baseline's bit for bit (or how far they are).
Needs the CUDA extension and a GPU; there is no CPU path.
"""
from __future__ import annotations

import json
import sys
from dataclasses import replace

import torch

from . import binding as B
from . import workloads as W


class _Case:
    def __init__(self, w: W.Workload):
        self.w, self.dev = w, torch.device("cuda", 0)
        self.plan = B.Plan(B.config_of(w), 0)
        self.C = torch.from_numpy(W.make_C(w)).to(self.dev)
        gen = torch.Generator(device=self.dev)
        gen.manual_seed(1)
        shape = self.plan.eps_shape
        self.ns = 3 if w.cells * 48 * w.n_pairs * 3 < 24e9 else 1          # rotating field sets: no step finds its inputs in L2
        field = lambda: torch.view_as_complex(torch.randn(*shape, 2, device=self.dev, dtype=torch.float32, generator=gen))
        self.EF = [[field() for _ in range(w.n_pairs)] for _ in range(self.ns)]
        self.EA = [[field() for _ in range(w.n_pairs)] for _ in range(self.ns)]
        self.beta = w.betas[-1]
        self.eps = torch.empty(shape, dtype=torch.float32, device=self.dev)
        self.g = torch.empty(self.plan.ctrl_shape, dtype=torch.float32, device=self.dev)

    def reset(self):
        p = self.plan
        p.set_bulk_stores(0); p.set_tma(0); p.set_fused(0); p.set_pdl(1); p.set_overlap(True)
        for k in range(8):
            p.set_tuning(k, 0)

    def result(self):
        nan = lambda s: torch.full(s, float("nan"), dtype=torch.float32, device=self.dev)
        e, g = self.plan.eps_forward_vjp(self.C, self.beta, self.EF[0], self.EA[0], nan(self.plan.eps_shape), nan(self.plan.ctrl_shape))
        torch.cuda.synchronize()
        return e, g

    def _replay_us(self, fn, steps):
        for s in range(min(3, self.ns)):
            fn(s)
        torch.cuda.synchronize()
        graphs = []
        for s in range(self.ns):
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr):
                fn(s)
            graphs.append(gr)
        for i in range(6):
            graphs[i % self.ns].replay()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for i in range(steps):
            graphs[i % self.ns].replay()
        b.record()
        torch.cuda.synchronize()
        return round(a.elapsed_time(b) / steps * 1e3, 1)

    def step_us(self, steps=100):
        p = self.plan
        return {"fwd+vjp": self._replay_us(lambda s: p.eps_forward_vjp(self.C, self.beta, self.EF[s], self.EA[s], self.eps, self.g), steps),
                "fwd": self._replay_us(lambda s: p.eps_forward(self.C, self.beta, self.eps), steps),
                "vjp": self._replay_us(lambda s: p.eps_vjp(self.C, self.beta, self.EF[s], self.EA[s], self.g), steps)}

    def kernels_us(self, n=20):
        p, acc = self.plan, {}
        p.set_profiling(True)
        for i in range(n + 3):
            torch.cuda._sleep(int(150e-6 * 1.9e9))            # the host queues the whole step behind a spin kernel
            p.eps_forward_vjp(self.C, self.beta, self.EF[i % self.ns], self.EA[i % self.ns], self.eps, self.g)
            if i >= 3:
                for k, ms in p.last_kernel_times():
                    acc[k] = acc.get(k, 0.0) + ms
        p.set_profiling(False)
        return {k: round(v / n * 1e3, 1) for k, v in acc.items()}


def _agree(e, g, e0, g0):
    if bool(torch.equal(e, e0)) and bool(torch.equal(g, g0)):
        return "bitwise"
    return {"eps_max_rel": float(((e - e0).abs() / e0).max()), "grad_rel": float((g - g0).abs().max() / g0.abs().max()),
            "nan": int(torch.isnan(e).sum()) + int(torch.isnan(g).sum())}


def streams(args):
    c = _Case(W.BY_NAME[args[0] if args else "paper"])
    steps = 100 if c.w.cells < 1e8 else 10
    c.reset()
    e0, g0 = c.result()
    # (name, bulk stores, TMA mode, tuning knobs): knob 0 bulk bytes, 1 store CTAs / SM, 2 ring stages, 3 read CTAs / SM, 5 fill policy
    variants = [("base", 0, 0, ()), ("field fills without the evict-first policy", 0, 0, ((5, 2),)), ("bulk stores", 1, 0, ()), ("bulk 32 KB", 1, 0, ((0, 32768),)), ("bulk 3 CTAs/SM", 1, 0, ((1, 3),)),
                ("TMA ring", 0, 2, ()), ("TMA ring 4 stages", 0, 2, ((2, 4),)), ("TMA ring 4 stages 2 CTAs/SM", 0, 2, ((2, 4), (3, 2))),
                ("TMA per block", 0, 1, ()), ("bulk + TMA ring", 1, 2, ())]
    for name, bulk, tma, tune in variants:
        c.reset()
        c.plan.set_bulk_stores(bulk); c.plan.set_tma(tma)
        for k, v in tune:
            c.plan.set_tuning(k, v)
        e, g = c.result()
        print(json.dumps({"workload": c.w.name, "variant": name, "agree": _agree(e, g, e0, g0), "step_us": c.step_us(steps), "kernels_us": c.kernels_us()}), flush=True)


def pdl(args):
    for name in args or ["tiny", "paper", "large"]:
        c = _Case(W.BY_NAME[name])
        steps = 100 if c.w.cells < 1e8 else 10
        c.reset()
        e0, g0 = c.result()
        for rep in range(2):
            for on in (0, 1):
                c.reset()
                c.plan.set_pdl(on)
                e, g = c.result()
                print(json.dumps({"workload": name, "pdl": on, "agree": _agree(e, g, e0, g0), "step_us": c.step_us(steps)}), flush=True)
        del c
        torch.cuda.empty_cache()


def fused(args):
    c = _Case(W.BY_NAME[args[0] if args else "paper"])
    steps = 100 if c.w.cells < 1e8 else 10
    c.reset()
    e0, g0 = c.result()
    print(json.dumps({"workload": c.w.name, "variant": "separate kernels", "step_us": c.step_us(steps)}), flush=True)
    # knob 4: CTAs / SM of the persistent kernel; knob 6: pipeline lag between producer and consumer phases
    for mode, label in ((1, "one persistent kernel"), (2, "persistent 2-D chains beside the stream kernels")):
        for tune in ((), ((4, 3),), ((4, 2),), ((6, 3),)):
            c.reset()
            c.plan.set_fused(mode)
            for k, v in tune:
                c.plan.set_tuning(k, v)
            e, g = c.result()
            print(json.dumps({"workload": c.w.name, "variant": label, "tuning": tune, "agree": _agree(e, g, e0, g0), "launches": c.plan.last_launches(),
                              "step_us": c.step_us(steps)}), flush=True)
    c.reset()
    c.plan.set_fused(1)
    c.plan.fused_profile(True)
    c.result()
    pr = c.plan.fused_profile(False, read=True)
    tot = max(1, pr["total"])
    print(json.dumps({"workload": c.w.name, "persistent kernel, % of CTA cycles": {k: round(100 * v / tot, 1) for k, v in pr["busy"].items()},
                      "tickets": round(100 * pr["tickets"] / tot, 1), "waiting for bands": round(100 * pr["wait"] / tot, 1),
                      "release": round(100 * pr["release"] / tot, 1), "starting copies": round(100 * pr["zbegin"] / tot, 1), "items": pr["items"]}), flush=True)


_TC_SLOTS = {0: "fwd staging", 1: "fwd wait for accumulator", 2: "fwd read-out + stores", 3: "fwd MMA thread waiting", 4: "fwd MMA issue", 5: "fwd tiles",
             8: "T MMA thread waiting for weights", 9: "T MMA thread waiting for data", 10: "T MMA thread total", 11: "T worker waiting for a free slot",
             12: "T worker waiting for the accumulator", 13: "T read-out", 14: "T overlap-add", 15: "T worker total"}


def tc(args):
    cases = [(int(a), float(b)) for a, b in (x.split(":") for x in args)] if args else [(250, 8.0), (250, 12.0), (375, 8.0), (500, 8.0), (500, 12.0), (1000, 8.0), (1000, 12.0)]
    base = W.BY_NAME["paper"]
    for mx, radius in cases:
        w = replace(base, name=f"{mx}x{mx} R={radius:g}", mx=mx, my=mx, radius=radius, nz=16, z_lo=6.25, z_hi=9.75)
        c = _Case(w)
        c.reset()
        c.plan.set_tensor_cores(0)
        e0, g0 = c.result()
        res = {"control": f"{mx}x{mx}", "R": radius}
        for mode in (0, 1):
            c.plan.set_tensor_cores(mode)
            e, g = c.result()
            k = c.kernels_us()
            res["tensor cores" if mode else "ffma"] = {n: k[n] for n in ("filter", "filterT")}
            if mode:
                res["eps_max_rel_diff"] = float(((e - e0).abs() / e0).max())
                res["grad_rel_diff"] = float((g - g0).abs().max() / g0.abs().max())
        c.plan.fused_profile(True)                              # cycle sums over the CTAs (filter_tc.cuh, filterT_tc.cuh)
        c.result()
        raw = c.plan.fused_profile(False, read=True)["raw"]
        res["cycle_sums_over_ctas"] = {n: raw[i] for i, n in _TC_SLOTS.items() if raw[i]}      # "fwd tiles" is a count
        print(json.dumps(res), flush=True)
        del c
        torch.cuda.empty_cache()


def replay(args):
    """replays CUDA graphs of eps_forward_vjp (3 rotating field sets, 9 replays) with the given tuning knobs: a target for
    `ncu --graph-profiling node --cache-control none`, which then sees every kernel with the L2 state its predecessors left"""
    c = _Case(W.BY_NAME[args[0] if args else "paper"])
    c.reset()
    for kv in args[1:]:
        k, v = kv.split("=")
        c.plan.set_tuning(int(k), int(v))
    print(json.dumps({"workload": c.w.name, "tuning": args[1:], "step_us": c._replay_us(
        lambda s: c.plan.eps_forward_vjp(c.C, c.beta, c.EF[s], c.EA[s], c.eps, c.g), 9)}), flush=True)


def main(argv=None):
    argv = list(sys.argv[1:] if argv is None else argv)
    table = {"streams": streams, "pdl": pdl, "fused": fused, "tc": tc, "replay": replay}
    if not argv or argv[0] not in table:
        print(__doc__)
        return 2
    if not torch.cuda.is_available():
        raise RuntimeError("abtest needs a GPU: the library has no CPU path")
    table[argv[0]](argv[1:])
    return 0


if __name__ == "__main__":
    sys.exit(main())
