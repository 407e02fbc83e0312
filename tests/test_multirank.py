"""The N > 1 path of bench.py on CPU: two `gloo` ranks.  Multi-GPU here means independent
replicas (`north_star` fixes one GPU, no sharding, no collectives), so the only
thing ranks exchange is the elapsed time: the job's time is the maximum over ranks and the value
is world * units / that time.  Also checks that `--impl reference` leaves all work to rank 0."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")        # rank 1 is the slow one
val = bench.aggregate_value(1000.0, 4, ms, dist.get_world_size())
print(json.dumps({{"rank": rank, "ms": ms, "value": val}}))
dist.destroy_process_group()
"""


def _free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.timeout(300)
def test_max_over_ranks_with_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 15.0                                      # the slowest rank's time, on every rank
        assert o["value"] == pytest.approx(2 * 1000.0 * 4 / 15e-3)   # whole-job units / that time


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.aggregate_value(10.0, 2, 4.0, 1) == pytest.approx(10.0 * 2 / 4e-3)


@pytest.mark.timeout(600)
def test_reference_arm_runs_on_rank_zero_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 prints the line, rank 1 exits 0 silently"""
    outs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2")
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2",
                            "--warmup", "1", "--config", "0"], env=env, capture_output=True, text=True, timeout=500)
        assert r.returncode == 0, r.stderr[-2000:]
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
