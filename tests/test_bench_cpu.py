"""CPU-side tests of bench.py: the reference arm (the oracle timed on the host cores), the flop model,
and the N > 1 path (replicas) with a world_size-2 gloo job."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--ref-size", "16",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300, check=True)
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "cell-updates/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["higher_is_better"] is True and d["gpu_launches"] == 0


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, env=env, check=True)
    assert out.stdout.strip() == ""


def test_flop_model_is_the_oracle_count():
    sys.path.insert(0, ROOT)
    import bench
    fm = bench.flop_model(256)
    # SURVEY.md 8(d) hand count: ~8600 flop per cell-step, ~2860 per stage; the oracle's own count must be near it
    assert 8000 < fm["step"] < 9500
    assert abs(fm["step"] - (3 * fm["rhs"] + 3 * 20)) / fm["step"] < 0.02      # + RK combination (20 flop per stage)
    assert fm["prim"] < fm["grad"] < fm["rhs"]


def test_two_rank_gloo_aggregation():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "tests", "_gloo_worker.py")]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert d["max"] == [15.0, 100.0]                      # max over the two ranks, element-wise
    assert d["value"] == 2 * 1000 * 4 / 15.0e-3           # all ranks' cells x steps / slowest rank's time
