"""N > 1 path of bench.py on CPU: two ranks over gloo (replicas only, no data-path
collective; the only cross-rank traffic is the timing barrier and the max-over-ranks reduction)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _run(nproc, extra):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"),
           "--gpus", str(nproc)] + extra
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout          # rank 0 alone prints ONE JSON line
    return json.loads(lines[0])


def test_two_ranks_take_the_max_time_and_sum_the_work():
    d = _run(2, ["--plumbing-test", "--steps", "4", "--warmup", "3"])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak"
    # fake timings: rank r reports 10 (r + 1) ms -> max = 20 ms; 2 ranks x 1000 units x 4 steps / 20 ms
    assert abs(d["ms_per_step"] - 5.0) < 1e-9
    assert abs(d["value"] - 2 * 1000 * 4 / 0.020) < 1e-6


def test_single_rank_plumbing_needs_no_process_group():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--plumbing-test", "--steps", "2"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads(out.stdout.strip().splitlines()[-1])
    assert d["n_gpus"] == 1 and abs(d["value"] - 1000 * 2 / 0.010) < 1e-6


def test_reference_arm_prints_only_on_rank0():
    """--impl reference under torchrun: rank 0 runs the oracle on a tiny sample, the other rank exits 0 silently."""
    d = _run(2, ["--impl", "reference", "--config", "1", "--steps", "2", "--warmup", "1"])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
