"""bench.py's JSON contract on a GPU box (-m gpu): one line, the driver's keys, the tier's roofline /
cpu_baseline / e2e objects, for both solver modes and the reference arm."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args, env=None):
    e = dict(os.environ)
    e.update(env or {})
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args, "--oracle-crop", "96"], capture_output=True, text=True,
                       timeout=900, env=e)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, r.stdout
    return json.loads(lines[0])


def test_bench_line_contract_small_config():
    d = _run("--config", "3", "--nx", "256", "--ny", "192", "--steps", "3", "--warmup", "3")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["unit"] == "cell-updates/s" and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3 and d["higher_is_better"] is True
    assert d["vs_baseline"] is None and "workload" in d["config"] and "model" not in d["config"]
    assert d["value"] > 0 and abs(d["value"] - 256 * 192 * 3 / (d["ms_per_step"] * 3e-3)) <= 1e-6 * d["value"]
    assert d["gpu_launches"] > 0 and d["config"]["status"] == [0, 0]
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["peak"] > 1000 and r["achieved"] > 0
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and "traffic" in r
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == e["d2h_bytes_per_step"] == 8 * (3 * 256 * 192 + 2 * 257 * 193)
    assert e["value"] < d["value"]                  # same step window + host copies: slower than the device leg
    assert e["iters_per_solve"] == d["config"]["iters_per_solve"]   # ... and the same solves
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"] and c["iters_per_solve"] > 0
    assert d["config"]["oracle_crop"] == 96
    assert d["clocks"]["sm_mhz"] and d["clocks"]["sm_max_mhz"] and isinstance(d["clocks"]["reasons"], list)


def test_bench_paper_solver_mode_and_reference_arm():
    d = _run("--config", "3", "--nx", "256", "--ny", "192", "--steps", "3", "--warmup", "3", "--solver", "srj",
             "--srj-eps", "1e-7", "--no-cpu")
    assert "k_srj" in d["roofline"]["kernel"] and d["roofline"]["bytes_per_node_iteration"] == 56.0
    assert "cpu_baseline" not in d and d["config"]["iters_per_solve"] > 1
    ref = _run("--impl", "reference", "--steps", "1", "--warmup", "0")
    assert ref["impl"] == "reference" and ref["value"] > 0 and ref["cpu_baseline"]["kind"] == "oracle"
    assert ref["metric"] == d["metric"] and ref["unit"] == d["unit"]


def test_bench_table2_and_fullruns_modes():
    e = dict(os.environ)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--table2", "64"], capture_output=True,
                       text=True, timeout=600, env=e)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads([l for l in r.stdout.splitlines() if l.strip()][-1])
    row = d["table2"][0]
    assert row["n"] == 64 and all(k in row for k in ("swe", "nh_1e-3", "nh_1e-4", "nh_1e-5"))
    assert all(row[k]["t_end"] >= 1.0 and row[k]["seconds"] > 0 for k in ("swe", "nh_1e-3", "nh_1e-4", "nh_1e-5"))
    assert row["swe"]["sweeps_per_solve"] == 0.0
    assert row["nh_1e-3"]["sweeps_per_solve"] <= row["nh_1e-4"]["sweeps_per_solve"] <= row["nh_1e-5"]["sweeps_per_solve"]
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--fullruns", "1,2"], capture_output=True,
                       text=True, timeout=600, env=e)
    assert r.returncode == 0, r.stderr[-2000:]
    rows = [json.loads(l) for l in r.stdout.splitlines() if l.strip()]
    assert [x["config"] for x in rows] == [1, 2] and all(x["status"] == 0 and x["finite"] for x in rows)
    assert rows[0]["steps"] == 200 and rows[1]["steps"] == 1000 and rows[1]["iters_per_solve"] == 0.0
    assert abs(rows[0]["mass_rel_change"]) < 1e-12 and rows[1]["mass_rel_change"] == 0.0


def test_bench_streammix_mode():
    # the measurement hook behind profiles/r03c: plain streaming kernels with the solver's plane mixes
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--streammix", "--config", "3", "--nx", "1024",
                        "--ny", "1024"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads([l for l in r.stdout.splitlines() if l.strip()][-1])
    assert set(d["GBs"]) == {"1R+1W", "5R+1W", "8R+4W", "6R+1W"} and all(v > 100.0 for v in d["GBs"].values())
    assert d["nodes"] == 1025 * 1025 and d["bicgstab_floor_ms_per_iteration"] > 0
    from paper_1706_04551_b200 import nh
    with pytest.raises(nh.NHError):
        nh.stream_mix_rate(3, 3, 1024)        # a mix the hook has no kernel for
