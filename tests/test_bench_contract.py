"""bench.py's reference arm runs on CPU (it times the oracle): check the JSON line it prints against the contract
(keys, metric, unit, config) for both lens models, and that ranks other than 0 print nothing."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(extra, env=None):
    e = dict(os.environ)
    e.update(env or {})
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "3",
                        "--cpu-seconds", "0.2"] + extra, capture_output=True, text=True, env=e, timeout=600)
    assert r.returncode == 0, r.stderr
    return r.stdout.strip()


@pytest.mark.parametrize("extra,workload", [([], "cfg3_4096x4096_1000"), (["--config", "1"], "cfg1_1024x1024_100"), (["--model", "sie"], "sie_paper_6730x6730_702"),
                                            (["--model", "nfw"], "nfw_512x512_64_n2048")])
def test_reference_arm_line(extra, workload):
    out = _run(extra)
    lines = [l for l in out.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "lens_pixel_gradient_evals_per_s" and d["unit"] == "lens*pixel/s"
    assert d["higher_is_better"] is True and d["n_gpus"] == 1 and d["steps"] == 1 and d["warmup"] == 3
    assert d["config"]["workload"] == workload and d["value"] > 0 and d["ms_per_step"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["sample"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert d["gpu_launches"] == 0 and d["data"] == "synthetic"


def test_reference_arm_ignores_the_launchers_omp_default():
    """torch.distributed.run exports OMP_NUM_THREADS=1 to its ranks; the reference arm must time the oracle on the same
    cores at every N, so it reports (and uses) the cores of the process, not OpenMP's default."""
    d = json.loads(_run([], env={"OMP_NUM_THREADS": "1", "RANK": "0", "WORLD_SIZE": "2"}))
    assert d["cpu_baseline"]["cores"] == len(os.sched_getaffinity(0))


def test_reference_arm_other_ranks_are_silent():
    assert _run([], env={"RANK": "1", "WORLD_SIZE": "2"}) == ""


@pytest.mark.gpu
def test_our_arm_line_on_the_gpu():
    """The line bench.py prints for our arm, with its defaults: the largest single-GPU configuration, every key of the
    contract (value, e2e with its byte counts, gpu_launches, clocks, roofline with bound / achieved / peak / frac /
    traffic, cpu_baseline), the other modes, the other configs, and per mode the parity against the oracle with its
    tolerance."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3", "--warmup", "3", "--cpu-seconds", "0.5"],
                       capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline",
              "modes", "configs", "parity"):
        assert k in d, k
    assert d["metric"] == "lens_pixel_gradient_evals_per_s" and d["dtype"] == "f64" and d["scaling"] == "weak"
    assert d["config"]["workload"] == "cfg3_4096x4096_1000" and d["vs_baseline"] is None
    assert d["value"] > 1e10 and d["gpu_launches"] >= 2 * d["steps"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 1000 * 56 and e["d2h_bytes_per_step"] == 4096 * 4096 * 16
    rf = d["roofline"]
    assert rf["bound"] == "alu" and rf["unit"] == "TFLOP/s" and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert 0 < rf["frac"] < 1 and 0 < rf["executed"]["frac_of_floor"] < 1
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["sample"]
    assert set(d["modes"]) == {"fp64", "fp32", "mixed"}
    assert "sm_mhz" in d["clocks"] and "reasons" in d["clocks"]
    assert set(d["configs"]) == {"cfg1_1024x1024_100", "cfg2_2048x2048_500", "cfg4_stress_2048x2048_200",
                                 "sie_paper_6730x6730_702"}
    for block in [d] + list(d["configs"].values()):
        for mode in ("fp64", "fp32", "mixed"):
            p = block["parity"][mode]
            assert p["pass"] and p["max_err_rel"] < p["tol"] and p["n_sampled"] >= 19000, (mode, p)
        assert block["parity"]["mixed"]["flagged_bit_equal_to_fp64_mode"]
    for name, cfg in d["configs"].items():
        for mode in ("fp64", "fp32", "mixed"):
            assert cfg[mode]["value"] > 1e10, (name, mode)


@pytest.mark.gpu
def test_strong_scaling_arm_on_one_gpu():
    """--shard rows under one rank: the row-block arm runs, says so, and reports the same metric as strong scaling."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--shard", "rows", "--gather", "--config", "2",
                        "--mode", "mixed", "--steps", "3", "--warmup", "3", "--no-extras"],
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr
    d = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][0])
    assert d["scaling"] == "strong" and d["config"]["parallelism"].startswith("rows/1")
    assert d["shard"]["rows_per_rank"] == [2048] and len(d["shard"]["ms_per_rank"]) == 1 and d["value"] > 1e10


def test_parity_block_of_the_bench_line_on_cpu():
    """bench.py's parity leg (oracle_parity) needs no GPU for its own logic: fed with the oracle's `double` map as the
    "device" values it must report a tiny error that passes, with the sample it promises; fed with a map that is off by
    2e-5 of max|alpha| in one pixel it must fail fp32's tolerance."""
    import numpy as np
    sys.path.insert(0, ROOT)
    import bench
    from oracle import lt_oracle as O
    from paper_1902_03252_b200 import workloads
    W = workloads.make(0)
    i, j = bench.parity_sample(W)
    assert len(i) == 20000 + 8 and i.min() >= 0 and i.max() < W.nx and j.max() < W.ny
    g = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, precision=O.DOUBLE)
    got = g[j, i]
    flags = np.zeros(len(i), np.uint8)
    flags[:100] = 2
    sampled = {"fp64": got, "fp32": got.astype(np.float32).astype(np.float64), "mixed": got.copy()}
    p = bench.oracle_parity(W, sampled, flags, (3.26, 0.0104 / 0.03, 6.0, 0.3, 15.0))
    assert p["fp64"]["pass"] and p["fp64"]["max_err_rel"] < 1e-13 and p["fp64"]["tol"] == 1e-12
    assert p["fp32"]["pass"] and 1e-9 < p["fp32"]["max_err_rel"] < 1e-6 and p["fp32"]["n_sampled"] == len(i)
    assert p["mixed"]["flagged_bit_equal_to_fp64_mode"] and p["mixed"]["n_flagged_in_sample"] == 100
    bad = dict(sampled)
    bad["fp32"] = got.copy()
    bad["fp32"][7, 1] += 2e-5 * np.abs(g).max()
    assert not bench.oracle_parity(W, bad, flags, (3.26, 0.0104 / 0.03, 6.0, 0.3, 15.0))["fp32"]["pass"]
