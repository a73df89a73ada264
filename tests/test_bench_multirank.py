"""N > 1 plumbing of bench.py on CPU (gloo, world_size 2): the path shards by independent streams
(replicas, no data-path collective), so what needs covering is the rank bookkeeping:
max-over-ranks timing, the whole-job aggregate, and that only rank 0 of the reference arm prints."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from workloads import CONFIGS
    ms_local = 1.0 + rank                      # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, world)
    wl = CONFIGS["llava_ov_7b"]
    val = bench.job_value(wl, world, wl.n_streams, ms)
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms": ms, "value": val, "env": bench.dist_env()}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world2(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / f"r{i}.json")) for i in range(2)]
    assert r[0]["ms"] == r[1]["ms"] == 2.0                   # slowest rank's time on every rank
    from workloads import CONFIGS
    wl = CONFIGS["llava_ov_7b"]
    T = wl.budget + wl.chunk_tokens
    expect = 2 * wl.n_streams * wl.n_layers * T / 2.0e-3     # both replicas' tokens over the slowest time
    assert r[0]["value"] == pytest.approx(expect) and r[1]["value"] == pytest.approx(expect)
    assert r[0]["env"][0] == 0 and r[1]["env"][0] == 1 and r[0]["env"][2] == 2


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.dist_env() == (int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)),
                                int(os.environ.get("WORLD_SIZE", 1)))


def test_reference_arm_under_torchrun_prints_once():
    """`bench.py --impl reference` launched as 2 ranks: rank 0 times the oracle sample and prints ONE JSON
    line, the other rank exits 0 without work."""
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
