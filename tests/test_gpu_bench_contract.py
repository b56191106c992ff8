"""bench.py prints ONE JSON line with the keys the driver's contract names (the tier's roofline / cpu_baseline / e2e objects
included); the reference arm prints its own line with impl = "reference".  Run as the driver runs it, as a subprocess."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_bench_line_has_the_contract_keys():
    d = run_bench("--steps", "5", "--warmup", "3")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] == 3 and d["unit"] == "Yee-cells/s" and d["vs_baseline"] is None
    assert d["dtype"] == "f32" and d["data"] == "synthetic" and "paper" in d["config"]["workload"] and "model" not in d["config"]
    assert d["value"] > 1e10 and abs(d["value"] - 16e6 / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    assert d["gpu_launches"] == 6 * 5
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["kernel"] in ("zreduce", "extrude")
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0.05 < r["frac"] < 1.0
    assert abs(r["achieved"] - r["algorithmic_bytes"] / (r["kernel_ms"] * 1e-3) / 1e9) < 1e-6 * r["achieved"]
    assert r["traffic"] is None or r["traffic"] >= r["algorithmic_bytes"]
    e = d["e2e"]
    assert e["unit"] == d["unit"] and 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] >= 192e6
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and 0 < c["value"] < d["value"] and c["sample"]
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    # the three calls separately, medians of >= 20 repetitions; the slab-only fraction as the headline and the
    # dense-equivalent one beside it; the field stream also timed alone; traffic only from a capture of this very build
    m = d["modes"]
    assert set(m) == {"forward", "vjp", "forward_vjp"}
    for k in m:
        assert m[k]["reps"] >= 20 and m[k]["ms_min"] <= m[k]["ms_median"] and m[k]["cells_per_s"] > 1e10
    assert m["forward"]["ms_median"] < m["forward_vjp"]["ms_median"] and m["vjp"]["ms_median"] < m["forward_vjp"]["ms_median"]
    assert abs(d["ms_per_step_median"] - m["forward_vjp"]["ms_median"]) < 1e-12
    assert r["frac_dense_equiv"]["value"] > r["others"].get("zreduce", r)["frac"] and "not the method's work" in r["frac_dense_equiv"]["note"]
    assert 0.05 < r["zreduce_alone"]["frac"] < 1.0 and 0.05 < r["step"]["frac"] < 1.0
    assert set(r["modes_frac"]) == {"forward", "vjp", "vjp_dense_equiv"} and "traffic_source" in r
    tl = r["timeline_us"]                         # kernel ends inside the overlapped schedule
    assert [n for n, _ in tl][0] == "begin" and {n for n, _ in tl} >= {"filter", "fwd2d", "zreduce", "extrude", "maskgrad", "filterT"}
    assert all(0.0 <= t < 1e4 for _, t in tl)
    wn = r["eps_window_only"]                     # eps rewritten on the slab window only: also beside the headline
    assert 0 < wn["forward_ms_median"] <= m["forward"]["ms_median"] * 1.05 and "not the headline" in wn["note"]
    assert 0 < wn["with_packed_fields_forward_vjp_ms_median"] <= m["forward_vjp"]["ms_median"] * 1.05
    pk = r["packed_fields"]                       # the same step with the fields on the design region only: beside the headline, not it
    assert pk["window_cells"][1] > 0 and pk["bytes_read"] > 0 and "not the headline" in pk["note"]
    assert 0 < pk["zreduce_alone_ms"] <= r["zreduce_alone"]["kernel_ms"] * 1.5 and 0 < pk["forward_vjp_ms_median"] and 0 < pk["zreduce_in_step_frac"] < 1.2
    assert c["forward_cells_per_s"] > 0 and c["vjp_cells_per_s"] > 0


@pytest.mark.parametrize("shard,config", [("pairs", "multiwavelength"), ("xslab", "paper")])
def test_sharded_bench_lines_at_one_rank(shard, config):
    # the N > 1 modes at N = 1: the same control flow (sharding.shard_step) with a world of one
    d = run_bench("--shard", shard, "--config", config, "--steps", "3", "--warmup", "3")
    assert d["shard"] == shard and d["scaling"] == "strong" and d["n_gpus"] == 1 and d["value"] > 1e9
    assert d["gpu_launches"] > 0 and 0.01 < d["roofline"]["frac"] < 1.0 and "all-reduce" in d["config"]["per_gpu"]


def test_reference_arm_times_the_oracle():
    d = run_bench("--impl", "reference", "--steps", "1", "--warmup", "1")
    assert d["impl"] == "reference" and d["dtype"] == "f64" and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["unit"] == "Yee-cells/s" and d["higher_is_better"] is True
