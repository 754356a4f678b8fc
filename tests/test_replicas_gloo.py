"""The N > 1 path (independent replicas + barrier + max-over-ranks timing) on CPU with gloo, world_size 2."""
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parents[1]


def test_two_replicas_report_max_time_and_whole_job_value():
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                          "127.0.0.1", "--master-port", "29577", str(ROOT / "tests" / "gloo_worker.py")],
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("RESULT")][0]
    assert "world=2" in line and "ms=2.0" in line and "value=1000000.0" in line, line


def test_single_process_is_identity():
    from paper_2606_19025_b200 import replicas
    assert replicas.world() == 1 and replicas.max_over_ranks(3.5) == 3.5
    assert replicas.whole_job_tokens_per_s(8192, 0.5) == 8192 / 0.5e-3
