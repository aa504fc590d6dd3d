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


# ---------------------------------------------------------------------------------------------------------------
# halo exchange: the transfer of paper_2403_05910_b200/halo.py over torch.distributed, world
# size 2 over gloo with CPU tensors standing for the packed face buffers (the pack / unpack kernels and the decomposed
# time stepping are verified on the GPU by tests/test_gpu_halo.py with the in-process transport).
# ---------------------------------------------------------------------------------------------------------------
_HALO_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2403_05910_b200 import halo
dist.init_process_group("gloo")
rank = dist.get_rank()

class FakeBlock:      # what DistTransport touches of a halo.Block
    def __init__(self, spec, m):
        self.spec, self.S = spec, torch.zeros(1, dtype=torch.float64)
        self.send = {{k: torch.full((m,), 100.0 * spec.coord[0] + 10.0 * k[0] + k[1] + 1000.0 * spec.coord[1], dtype=torch.float64)
                     for k, o in spec.neighbour.items() if o is not None}}
        self.recv = {{k: torch.full((m,), -1.0, dtype=torch.float64) for k in self.send}}

ok = True
# (a) x periodic and split in two: BOTH faces of a block border the same neighbour -> two messages per pair, matched by order
for procs, bc, d in (((2, 1, 1), (0, 0, 1, 1, 1, 1), 0), ((1, 2, 1), (1, 1, 3, 1, 0, 0), 1)):
    dec = halo.Decomposition((16, 12, 8), procs, bc)
    spec = dec.block(dec.coord_of(rank))
    b = FakeBlock(spec, 7)
    tr = halo.DistTransport(dec, b, dist)
    tr.exchange(d)
    for (dd, side), other in spec.neighbour.items():
        if other is None:
            continue
        # my ghost layers on `side` hold the neighbour's border on ITS opposite side
        want = 100.0 * other[0] + 10.0 * dd + (1 - side) + 1000.0 * other[1]
        ok = ok and bool((b.recv[(dd, side)] == want).all())
    n_faces = sum(o is not None for o in spec.neighbour.values())
    ok = ok and n_faces == (2 if procs[0] == 2 else 1)
    ok = ok and tr.max([1.0 + rank, 0.5]) == 2.0
sys.stdout.write("HALO %d %s\n" % (rank, ok)); sys.stdout.flush()
dist.destroy_process_group()
"""


def test_halo_transfer_over_gloo(tmp_path):
    script = tmp_path / "halo_worker.py"
    script.write_text(_HALO_WORKER.format(root=str(ROOT)))
    p = _torchrun([str(script)])
    assert p.returncode == 0, p.stderr[-2000:]
    import re

    rows = re.findall(r"HALO (\d) (True|False)", p.stdout + p.stderr)
    assert sorted(rows) == [("0", "True"), ("1", "True")], p.stdout + p.stderr[-1500:]


def test_decomposition_bookkeeping():
    from paper_2403_05910_b200 import halo

    dec = halo.Decomposition((50, 31, 12), (3, 2, 1), (3, 1, 0, 0, 2, 2))
    specs = [dec.block(c) for c in dec.coords]
    assert [dec.rank_of(s.coord) for s in specs] == list(range(6)) and all(dec.coord_of(dec.rank_of(s.coord)) == s.coord for s in specs)
    assert sum(s.n[0] * s.n[1] * s.n[2] for s in specs) == 50 * 31 * 12
    assert sorted({(s.offset[0], s.n[0]) for s in specs}) == [(0, 17), (17, 17), (34, 16)]
    first, last = dec.block((0, 0, 0)), dec.block((2, 1, 0))
    assert first.bc == (3, 4, 4, 4, 2, 2) and last.bc == (4, 1, 4, 4, 2, 2)          # physical faces keep their kind
    assert first.neighbour[(1, 0)] == (0, 1, 0) and first.neighbour[(0, 0)] is None   # y periodic wraps, x does not
    import pytest

    with pytest.raises(ValueError):
        halo.Decomposition((8, 8, 1), (1, 1, 2), (0,) * 6)
    with pytest.raises(ValueError):
        halo.Decomposition((8, 8, 8), (4, 1, 1), (0,) * 6)
