"""bench.py's JSON contract on a small lattice (64^3, a few steps) on the GPU: the keys the driver reads, the roofline /
sustained / e2e / cpu_baseline objects, that the step kernel is the only kernel inside the timed region, and the
--aux and --decomp slab modes.  The numbers themselves mean nothing at this size."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*flags):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + list(flags), cwd=ROOT, capture_output=True,
                       text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    return json.loads(lines[0])


def test_bench_line_has_the_contract_keys():
    d = run_bench("--size", "64", "--steps", "5", "--warmup", "3", "--cpu-seconds", "1")
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline",
                "sustained"):
        assert key in d, key
    assert d["unit"] == "MLUPS" and d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] == 3
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["gpu_launches"] == 5                                     # one step kernel per step, nothing else
    assert abs(d["value"] - 64 ** 3 * 5 / (d["ms_per_step"] * 5e-3) / 1e6) < 1e-6 * d["value"]
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["kernel"] == "step_kernel_tma<TX=64>"
    assert r["algorithmic_bytes_per_launch"] == 2 * 27 * 8 * 64 ** 3
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and r["traffic"] is None      # no ncu capture at this size
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 4 * 64 ** 3 * 8 / 5 == e["d2h_bytes_per_step"] and e["pipelined"]
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["one_core"]["cores"] == 1
    assert c["out_of_cache"]["value"] > 0
    s = d["sustained"]
    assert s["steps"] >= 5 and s["ms_per_step"] > 0 and "clocks" in s
    # the sustained fraction is readable from `roofline` alone, with the clocks it was held at
    assert r["frac_sustained"] == s["frac"] and r["achieved_sustained"] == s["hbm_gbs"] and r["sustained_clocks"] == s["clocks"]
    assert abs(r["frac_sustained"] - 2 * 27 * 8 * 64 ** 3 / (s["ms_per_step"] * 1e-3) / 1e9 / r["peak"]) < 1e-9
    assert "burst" in r["frac_is"] and r["sustained_steps"] == s["steps"]
    assert e["outputs_equal_device_moments"] is True
    assert d["mass_rel_err"] < 1e-12


def test_bench_aux_and_slab_modes():
    a = run_bench("--aux", "--size", "64")["aux"]
    assert set(a) == {"rflbm_moments", "rflbm_stress", "rflbm_snapshot", "rflbm_diagnostics", "rflbm_get_populations",
                      "rflbm_set_populations", "rflbm_init(rho,u)", "rflbm_init(NULL)"}
    assert all(v["ms"] > 0 and v["gbs"] > 0 for v in a.values())
    d = run_bench("--size", "64", "--steps", "4", "--warmup", "3", "--no-cpu", "--no-sustained", "--decomp", "slab")
    assert d["e2e"] is None and "z slabs" in d["config"]["parallelism"]
    assert d["gpu_launches"] == 4 * 5                                 # step + 2 packs + 2 unpacks per step
