"""bench.py on a GPU: the JSON line carries every key of the contract, and the torchrun launch path works."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parent.parent


def parse(stdout):
    lines = [l for l in stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, stdout
    return json.loads(lines[0])


def check_line(d, n_gpus=1, scaling="weak"):
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "gpu_launches", "roofline", "clocks", "e2e"):
        assert key in d, key
    assert d["n_gpus"] == n_gpus and d["value"] > 0 and d["dtype"] == "f32" and d["scaling"] == scaling
    assert d["gpu_launches"] > 0 and d["warmup"] >= 3 and d["vs_baseline"] is None
    r = d["roofline"]
    assert r["bound"] in ("alu", "hbm") and r["achieved"] > 0 and r["peak"] > 0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert "workload" in d["config"] and "model" not in d["config"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0 and e["value"] != d["value"]
    assert set(("sm_mhz", "sm_max_mhz", "reasons")) <= set(d["clocks"])


def test_bench_small_config_single_process():
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--config", "1", "--steps", "2", "--warmup", "3",
                        "--cpu-templates", "8"], capture_output=True, text=True, cwd=ROOT, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    d = parse(r.stdout)
    check_line(d)
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0


def test_bench_under_torchrun_one_rank():
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "1",
                        "--master-addr", "127.0.0.1", "--master-port", "29731", str(ROOT / "bench.py"), "--gpus", "1",
                        "--config", "1", "--steps", "1", "--warmup", "3", "--no-cpu-baseline"],
                       capture_output=True, text=True, cwd=ROOT, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    check_line(parse(r.stdout))


def test_bench_two_ranks_functional():
    """The N > 1 path (barriers, max over ranks, per-rank banks, rank 0 prints): two ranks share the one GPU of the test
    box, so this checks function, not speed (bench.py switches the timing exchange to gloo when ranks outnumber GPUs)."""
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29733", str(ROOT / "bench.py"), "--gpus", "2",
                        "--config", "1", "--steps", "1", "--warmup", "3", "--no-cpu-baseline"],
                       capture_output=True, text=True, cwd=ROOT, timeout=240,
                       env=dict(os.environ, GLOO_SOCKET_IFNAME="lo", SPIIR_BENCH_BACKEND="gloo"))
    assert r.returncode == 0, r.stderr[-2000:]
    d = parse(r.stdout)                     # exactly one line: only rank 0 prints
    check_line(d, n_gpus=2)
    assert d.get("functional_only") is True           # two ranks on one GPU: marked, not a multi-GPU number


def test_bench_two_ranks_shard_one_bank():
    """--shard: ONE bank split over the ranks by shard_templates ("scaling": "strong"), per-rank filter counts in the line."""
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29735", str(ROOT / "bench.py"), "--gpus", "2",
                        "--config", "1", "--steps", "1", "--warmup", "3", "--no-cpu-baseline", "--shard"],
                       capture_output=True, text=True, cwd=ROOT, timeout=240,
                       env=dict(os.environ, GLOO_SOCKET_IFNAME="lo", SPIIR_BENCH_BACKEND="gloo"))
    assert r.returncode == 0, r.stderr[-2000:]
    d = parse(r.stdout)
    check_line(d, n_gpus=2, scaling="strong")
    sh = d["shard"]
    assert sum(sh["filters_per_rank"]) == 64 * 256 and sh["imbalance_max_over_mean"] < 1.01


def test_bench_default_run_reports_every_config():
    """The driver's command: cfg3 as the headline plus a per_config leg for cfg0, cfg1 (one-shot and chunked), cfg2, cfg4."""
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--steps", "1", "--warmup", "3", "--cpu-templates", "4"],
                       capture_output=True, text=True, cwd=ROOT, timeout=1500)
    assert r.returncode == 0, r.stderr[-2000:]
    d = parse(r.stdout)
    check_line(d)
    assert d["e2e"].get("last_chunk_bitwise_equal_to_device_run") is True
    per = d["per_config"]
    assert set(per) == {"cfg0", "cfg1_oneshot", "cfg1_chunked", "cfg2", "cfg4", "small_templates_32", "small_templates_8"}
    for name, leg in per.items():
        assert leg["value"] > 0 and leg["bound"] in ("alu", "hbm") and 0 < leg["frac"] < 1.2, name
        assert leg["p50_us"] > 0 and leg["p99_us"] >= leg["p50_us"] and "reasons" in leg["clocks"], name
    assert per["cfg4"]["bound"] == "hbm" and per["cfg4"]["path"] == 3 and per["cfg0"]["path"] == 2
