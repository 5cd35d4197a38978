"""Multi-GPU path on CPU: world_size 2, gloo backend (tier rule 5: the path shards by replicas, with no
data-path collective; torch.distributed only brackets and reduces the timing).  Checks the host logic
bench.py uses under torchrun: frame sharding, per-rank seeds, barrier, MAX/SUM over ranks, whole-job
throughput, and that the reference arm runs on rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2602_17938_b200 import replicas  # noqa: E402


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_shard_partitions_the_frames():
    for n in (0, 1, 7, 64):
        for world in (1, 2, 3, 8):
            parts = [replicas.shard(n, r, world) for r in range(world)]
            flat = sorted(i for p in parts for i in p)
            assert flat == list(range(n))                       # complete and disjoint
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        replicas.shard(4, 2, 2)
    assert replicas.rank_seed(3, 0) == 3 and replicas.rank_seed(3, 5) != replicas.rank_seed(3, 4)
    assert replicas.max_over_ranks(2.5, 1) == 2.5 and replicas.job_throughput(4, 2.0, 1) == 2000.0


_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
from paper_2602_17938_b200 import replicas
rank, local_rank, world = replicas.env_rank_world()
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=world)
mine = replicas.shard(7, rank, world)                 # 7 frames over 2 ranks: 4 + 3
ms = 10.0 + 5.0 * rank                                # rank 1 is the slow one
replicas.barrier(world)
out = dict(rank=rank, world=world, mine=mine, seed=replicas.rank_seed(3, rank),
           max_ms=replicas.max_over_ranks(ms, world), units=replicas.sum_over_ranks(len(mine), world),
           fps=replicas.job_throughput(len(mine), ms, world))
replicas.barrier(world)
dist.destroy_process_group()
print("RESULT " + json.dumps(out))
"""


def test_two_ranks_gloo(tmp_path):
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    res = {}
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        line = [ln for ln in out.splitlines() if ln.startswith("RESULT ")][-1]
        r = json.loads(line[7:])
        res[r["rank"]] = r
    assert res[0]["mine"] == [0, 2, 4, 6] and res[1]["mine"] == [1, 3, 5]
    assert res[0]["seed"] != res[1]["seed"]
    for r in res.values():
        assert r["world"] == 2
        assert r["max_ms"] == 15.0                              # MAX over ranks, seen by both
        assert r["units"] == 7.0
        assert abs(r["fps"] - 7 * 1e3 / 15.0) < 1e-9            # whole-job units / slowest rank


def test_reference_arm_runs_on_rank_zero_only():
    """bench.py --impl reference under torchrun: ranks other than 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--workload", "config0"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""


_STREAM_WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
from paper_2602_17938_b200 import replicas
rank, local_rank, world = replicas.env_rank_world()
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=world)

def run_shard(mine):        # stands in for the CUDA call: 2 timed steps over this rank's frames, 3 ms per frame
    return 2 * len(mine), 2 * 3.0 * len(mine) * (1.0 + 0.5 * rank)

job = bench.stream_job(9, rank, world, run_shard)       # bench.py's own sharding + reduction code path
dist.destroy_process_group()
print("RESULT " + json.dumps(dict(rank=rank, **job)))
"""


def test_bench_stream_job_two_ranks_gloo(tmp_path):
    """bench.py --workload stream: the sharding (frame i -> rank i mod N) and the SUM/MAX reduction are bench.py's
    own code (stream_job); here with world_size 2 on gloo and a stub in place of the CUDA call."""
    port = _free_port()
    script = tmp_path / "stream_worker.py"
    script.write_text(_STREAM_WORKER.format(root=ROOT, port=port))
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    res = {}
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        r = json.loads([ln for ln in out.splitlines() if ln.startswith("RESULT ")][-1][7:])
        res[r["rank"]] = r
    assert res[0]["indices_this_rank"] == [0, 2, 4, 6, 8] and res[1]["indices_this_rank"] == [1, 3, 5, 7]
    # rank 0: 10 frame-steps in 30 ms; rank 1: 8 frame-steps in 36 ms -> 18 units over the slowest rank's 36 ms
    for r in res.values():
        assert r["frames_total"] == 18 and r["ms_slowest_rank"] == 36.0
        assert abs(r["frames_per_s"] - 18 * 1e3 / 36.0) < 1e-9


def test_bench_gpus_n_starts_n_ranks(monkeypatch):
    """`python bench.py --gpus 2` outside torchrun must launch 2 ranks (torch.distributed.run, 127.0.0.1)."""
    import bench
    seen = {}
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: seen.setdefault("cmd", cmd) and 0)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "2", "--steps", "3", "--warmup", "3"])
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    assert bench.main() == 0
    cmd = seen["cmd"]
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node" in cmd
    assert cmd[cmd.index("--nproc-per-node") + 1] == "2" and cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-6:] == ["--gpus", "2", "--steps", "3", "--warmup", "3"] and cmd[-7].endswith("bench.py")
    # under torchrun (RANK set) it must NOT respawn: the ranks come from the environment
    monkeypatch.setenv("RANK", "0")
    monkeypatch.setenv("WORLD_SIZE", "2")
    monkeypatch.setattr(bench, "run_cuda", lambda a: 17)
    assert bench.main() == 17
