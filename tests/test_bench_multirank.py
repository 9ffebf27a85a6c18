"""Host-side logic of bench.py's N > 1 path on CPU: two `gloo` ranks (world_size 2).

The path shards by DM trials with no data-path collective, so what there is
to test is the plumbing: per-rank workloads differ, the step time is the max over ranks, the
value is the whole-job aggregate, and the reference arm runs on rank 0 only."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
from workloads import get_workload, draw_pulses
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
w = bench.rank_workload(get_workload(3).scaled(8, 65536, 4), rank)
ms = bench.max_over_ranks(10.0 * (rank + 1))
out = dict(rank=rank, world=world, seed=w.seed, first_pulse=draw_pulses(w)[0].t0, ms=ms,
           value=bench.whole_job_value(world, w.n_samples, ms))
dist.barrier()
dist.destroy_process_group()
print("RESULT " + json.dumps(out), flush=True)
"""


def _torchrun(code_or_args, port, capture=True):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + code_or_args
    env = dict(os.environ, OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=capture, text=True, timeout=300)


def test_two_gloo_ranks_max_time_and_aggregate(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    res = _torchrun([str(script)], 29541)
    assert res.returncode == 0, res.stdout[-2000:] + res.stderr[-4000:]
    # the two ranks share stdout: their lines may run together
    dec = json.JSONDecoder()
    rows = [dec.raw_decode(part)[0] for part in res.stdout.split("RESULT ")[1:]]
    assert sorted(r["rank"] for r in rows) == [0, 1]
    r0, r1 = sorted(rows, key=lambda r: r["rank"])
    assert r0["world"] == r1["world"] == 2
    assert r0["seed"] != r1["seed"] and r0["first_pulse"] != r1["first_pulse"]  # each rank has its own DM trials
    assert r0["ms"] == r1["ms"] == 20.0                                         # max over ranks
    assert r0["value"] == r1["value"] == pytest.approx(2 * 8 * 65536 / 20e-3)   # whole-job samples/s


def test_reference_arm_runs_on_rank0_only():
    res = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                     "--workload", "1", "--cpu-seconds", "0.2"], 29543)
    assert res.returncode == 0, res.stdout[-2000:] + res.stderr[-4000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0


def test_single_process_helpers():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_value(4, 1000, 2.0) == pytest.approx(2e6)
