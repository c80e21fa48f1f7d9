"""bench.py's one-line JSON contract: the reference arm (the oracle on host cores; CPU test) and our arm on a
small pool (GPU test).  Checks keys and types, not numbers."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "cpu_baseline", "gpu_launches"}


def run_bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         cwd=ROOT, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.strip().splitlines() if ln.startswith("{")]
    assert len(lines) == 1, "exactly one JSON line on stdout"
    return json.loads(lines[0])


def test_reference_arm_prints_the_contract_line():
    line = run_bench("--impl", "reference", "--steps", "2", "--warmup", "1")
    assert BASE_KEYS <= set(line), BASE_KEYS - set(line)
    # the reference arm honours --steps / --warmup and times the oracle on OUR arm's workload -- same shape, the full
    # 512-page prefix per step, same byte convention -- and states the pool it really ran on (a host pool bounded by
    # RAM), not our arm's 96 GiB device pool
    assert line["steps"] == 2 and line["warmup"] == 1
    sys.path.insert(0, ROOT)
    import argparse

    import bench
    from paper_2606_31093_b200 import workloads as W

    ours = bench.bench_config(argparse.Namespace(prefix_tokens=8192, pool_order="nhd", pool_pages=65536, kernel="auto"), W.QWEN3_OMNI)
    own = {"pool_pages", "pool_GiB", "kernel", "pool"}
    assert {k: v for k, v in line["config"].items() if k not in own} == {k: v for k, v in ours.items() if k not in own}
    assert ours["pages_per_step"] == 512
    assert line["config"]["pool_pages"] == bench.ORACLE_POOL_PAGES and line["config"]["pool_GiB"] == 6.0
    assert line["config"]["kernel"].startswith("n/a") and "host-resident" in line["config"]["pool"]
    assert "full 512-page prefix" in line["cpu_baseline"]["sample"]
    assert line["impl"] == "reference" and line["metric"] == "kv_pack_unpack_GBps" and line["unit"] == "GB/s"
    assert line["value"] > 0 and line["higher_is_better"] is True and line["vs_baseline"] is None
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["cpu_baseline"]["value"] == line["value"] == line["e2e"]["value"]
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in line["config"] and "model" not in line["config"]


@pytest.mark.gpu
def test_our_arm_prints_the_contract_line():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    line = run_bench("--steps", "3", "--warmup", "3", "--pool-pages", "2048", "--e2e-steps", "2")
    assert BASE_KEYS | {"roofline", "clocks"} <= set(line)
    assert "impl" not in line or line["impl"] != "reference"
    assert line["n_gpus"] == 1 and line["steps"] == 3 and line["warmup"] == 3 and line["scaling"] == "weak"
    assert line["gpu_launches"] == 6  # one launch per kv_pack / kv_unpack in the timed device leg
    r = line["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and 0 < r["frac"] == pytest.approx(r["achieved"] / r["peak"])
    assert r["algorithmic_bytes"] == 2 * 512 * 48 * 2 * 16384
    e = line["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] >= 512 * 1572864 and e["d2h_bytes_per_step"] == 512 * 1572864
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] > 0
    assert set(line["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert line["config"]["workload"].startswith("configs[1]")
    assert line["bit_exact"] is True  # the timed region's last step, checked with torch indexing
    assert r["traffic"] is None  # a profile figure: emitted only for a profiled configuration (a pool of at least 12 GiB)
    # the host-link roofline is measured in the same run: peaks and fractions for offload, reload and both at once
    assert r["host"]["offload"] == line["roofline_host"]["offload"] and 0 < r["host"]["duplex"]["frac"]
    assert e["offload_frac"] == r["host"]["offload"]["frac"] and e["reload_frac"] == r["host"]["reload"]["frac"]
    h = line["roofline_host"]
    for k in ("offload", "reload", "duplex"):
        assert 0 < h[k]["frac"] == pytest.approx(h[k]["achieved"] / h[k]["peak"])
    assert h["peaks"]["h2d_GBps"] > 0 and h["peaks"]["d2h_GBps"] > 0 and h["peaks"]["duplex_GBps"] > 0
    # the e2e leg's steps one by one, and the link peaks' medians beside their best-of-20 figures
    sm = e["step_ms"]
    assert 0 < sm["best"] <= sm["median"] <= sm["worst"] and sm["best"] <= sm["mean"] <= sm["worst"]
    assert h["duplex"]["frac_best_step"] >= h["duplex"]["frac_median_step"] > 0
    assert h["duplex"]["frac_of_median_memcpy"] >= h["duplex"]["frac"] > 0
    assert 0 < h["peaks"]["median"]["duplex_GBps"] <= h["peaks"]["duplex_GBps"]
    assert r["kernel"].startswith("kv_move_shot_plain")  # the plain single-request case takes the short kernel
    assert "per_config" not in line  # needs the 96 GiB pool
    assert line["peer"]["available"] in (True, False)
    if line["peer"]["available"]:
        assert line["peer"]["push"]["bit_exact"] and line["peer"]["pull"]["bit_exact"]


@pytest.mark.gpu
def test_two_replicas_aggregate_on_rank_zero():
    """The N > 1 plumbing of our arm (barrier, max over ranks of the device-timed interval, sum of units) with two
    ranks sharing this box's one GPU over gloo: replicas never wait on one another's kernels, only the hosts
    meet at barriers.  Rank 0 prints the whole-job line, rank 1 prints nothing."""
    import socket
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK="0", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), KV_BENCH_BACKEND="gloo")
        procs.append(subprocess.Popen([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3",
                                       "--warmup", "3", "--pool-pages", "2048", "--e2e-steps", "2", "--no-cpu-baseline"],
                                      env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = [p.communicate(timeout=600) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    assert outs[1][0].strip() == ""
    line = json.loads([ln for ln in outs[0][0].strip().splitlines() if ln.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and line["value"] > 0
    # whole-job value = 2 replicas' bytes over the slower replica's time
    assert line["value"] == pytest.approx(2 * 4 * 512 * 1572864 * 3 / (line["ms_per_step"] * 3 * 1e-3) / 1e9, rel=1e-6)
