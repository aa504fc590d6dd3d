"""N > 1 plumbing on the CPU (gloo, world_size 2): the path has no exchange step (replicas
only), so what N > 1 adds is the launch contract of bench.py -- barrier, max over ranks, whole-job aggregate, rank 0
prints -- and that is what runs here without a GPU."""
import json
import os
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent

_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
r = bench.Ranks(world, "gloo", None)
r.barrier()
local_ms = 10.0 * (rank + 1)                    # rank 1 is the slow one
worst = r.max(local_ms)
value = r.whole_job_value(1000, 3, local_ms)
r.barrier()
sys.stdout.write("RESULT %d %r %r\n" % (rank, worst, value)); sys.stdout.flush()
r.close()
"""


def _torchrun(args, timeout=600):
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29533"] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_ranks_max_and_whole_job_value_over_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=str(ROOT)))
    p = _torchrun([str(script)])
    assert p.returncode == 0, p.stderr[-2000:]
    import re

    rows = re.findall(r"RESULT (\d) ([0-9.e+]+) ([0-9.e+]+)", p.stdout + p.stderr)   # ranks may share a line
    assert sorted(r[0] for r in rows) == ["0", "1"], p.stdout
    for rank, worst, value in rows:
        assert float(worst) == 20.0                          # max over ranks, on every rank
        assert abs(float(value) - 1000 * 3 * 2 / 20e-3) < 1e-6    # both replicas' cells over the slowest rank's time


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    p = _torchrun([str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                   "--grid", "24", "12", "12"])
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
