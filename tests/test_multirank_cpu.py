"""The N > 1 path of bench.py on CPU: world_size 2 over gloo ("replicas only").

The step itself does not shard (north_star: one GPU), so what N > 1 adds is host logic only: the max-over-ranks
of the timed region, the whole-job unit count, and "rank 0 alone prints" for the reference arm.  These tests run
that logic in two real processes with a gloo group on 127.0.0.1.
"""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


_WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
import torch
import torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%(port)d", rank=rank, world_size=world)
# rank r "measured" (r + 1) * 10 ms: the job's time is the slowest rank's
ms = bench.max_over_ranks(10.0 * (rank + 1), world, torch.device("cpu"))
value = bench.whole_job_value(32, 2, 5, world, ms * 1e-3)
dist.barrier()
print(json.dumps({"rank": rank, "ms": ms, "value": value}))
dist.destroy_process_group()
"""


def test_max_over_ranks_and_whole_job_value_gloo_world2(tmp_path):
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % {"root": ROOT, "port": port})
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 20.0                                   # max(10, 20) on both ranks
        assert o["value"] == pytest.approx(32 ** 3 * 2 * 5 * 2 / 0.020, rel=1e-15)


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(3.5, 1, None) == 3.5
    assert bench.whole_job_value(4, 1, 2, 1, 0.5) == 4 ** 3 * 2 / 0.5


def test_reference_arm_under_torchrun_rank0_alone_prints():
    """`--impl reference` launched the way the driver launches N > 1: rank 0 times the oracle and prints one
    JSON line, the other rank exits 0 without work."""
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "cfg0_chaotic32"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["e2e"]["value"] == line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
