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


def check_line(d, n_gpus=1):
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "gpu_launches", "roofline", "clocks", "e2e"):
        assert key in d, key
    assert d["n_gpus"] == n_gpus and d["value"] > 0 and d["dtype"] == "f32" and d["scaling"] == "weak"
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
