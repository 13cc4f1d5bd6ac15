"""N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- the job's time is the max over ranks of the
device-timed region and the work is the sum over ranks; rank 0 alone runs the reference arm."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
local_ms = 10.0 if rank == 0 else 25.0          # the slower rank sets the job time
local_flop = 4.0e9 if rank == 0 else 6.0e9
ms, gfl = bench.job_throughput(local_ms, local_flop, world, dist, "cpu")
sys.stdout.write(json.dumps({{"rank": rank, "ms": ms, "gflops": gfl}}) + "\n")     # one write: the two ranks share a pipe
sys.stdout.flush()
dist.destroy_process_group()
"""


def _free_port():
    import socket
    with socket.socket(socket.AF_INET, socket.SOCK_STREAM) as s:
        s.bind(("127.0.0.1", 0))
        return str(s.getsockname()[1])


def test_job_throughput_world_size_2(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(WORKER.format(root=ROOT))
    for attempt in range(3):      # rendezvous on a shared box can fail for reasons outside this code (port taken, resolver hiccup): retry
        port = _free_port()
        # gloo on the loopback interface: the container hostname may not resolve (or only intermittently)
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=port, OMP_NUM_THREADS="1")
        if os.path.isdir("/sys/class/net/lo") and attempt < 2:
            env["GLOO_SOCKET_IFNAME"] = "lo"
        r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                            "--master-addr", "127.0.0.1", "--master-port", port, str(script)],
                           capture_output=True, text=True, env=env, timeout=300)
        if r.returncode == 0:
            break
    assert r.returncode == 0, r.stderr[-2000:]
    # (two processes write to one pipe: tolerate two records on one line)
    rows = [json.loads(l) for l in r.stdout.replace("}{", "}\n{").splitlines() if l.startswith("{")]
    assert len(rows) == 2
    for row in rows:
        assert row["ms"] == pytest.approx(25.0)
        assert row["gflops"] == pytest.approx(10.0e9 / 25.0e-3 / 1e9)


def test_job_throughput_single_rank():
    sys.path.insert(0, ROOT)
    import bench
    ms, gfl = bench.job_throughput(2.0, 4.0e9, 1)
    assert ms == 2.0 and gfl == pytest.approx(2000.0)


def test_reference_arm_prints_on_rank0_only(tmp_path):
    """--impl reference under torchrun: ranks other than 0 exit 0 without work (no GPU needed: the oracle is numpy)."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "cfg2"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
