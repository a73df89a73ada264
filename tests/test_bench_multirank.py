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


# ---- the real run_ours() path on 2 ranks, with the library and the device stubbed at their boundaries ----------
class _FakeEvent:
    def record(self):
        import time
        self.t = time.perf_counter()

    def elapsed_time(self, other):
        return (other.t - self.t) * 1e3

    def synchronize(self):
        pass


class _CpuBackend:
    """Stand-in for bench.CudaBackend: CPU tensors, wall-clock events, gloo."""
    dist_backend = "gloo"

    def __init__(self):
        self.dev = torch.device("cpu")

    def init_process_group(self, d):
        d.init_process_group("gloo")

    def event(self):
        return _FakeEvent()

    def synchronize(self):
        pass

    def stream_synchronize(self):
        pass

    def pin(self, t):
        return t


class _FakeHermes:
    """Stand-in for the ctypes binding: tracks only what bench.py reads back (len, launch count, profile, cache)."""
    HERMES_REINDEX_LAZY, HERMES_SCORE_TCGEN05 = 1, 2

    def __init__(self):
        self.calls = 0

    def config_for_workload(self, wl, device=0, **over):
        return dict(wl=wl, device=device, **over)

    def hermes_create(self, cfg):
        return dict(cfg=cfg, len=0)

    def hermes_append_chunk(self, h, K, V, Q, pos_start=-1):
        assert K.shape[0] == h["cfg"]["wl"].n_streams and K.shape == V.shape
        n = K.shape[2]
        h["len"] = min(h["len"] + n, h["cfg"]["wl"].budget) if Q is not None else h["len"] + n
        self.calls += 1

    def hermes_append_chunk_host(self, h, K, V, Q, kept_out=None):
        self.hermes_append_chunk(h, K, V, Q)

    def hermes_len(self, h):
        return h["len"]

    def hermes_last_launch_count(self, h):
        return 4

    def hermes_last_score_path(self, h):
        return 2

    def hermes_v_pending(self, h):
        return 1

    def hermes_set_profiling(self, h, on):
        pass

    def hermes_get_profile(self, h):
        return {"append": 0.01, "score_stats": 0.2, "select": 0.02, "gather": 0.03}

    def hermes_get_cache(self, h, b, l):
        z = torch.zeros(4)
        return {"k": z, "v": z, "pos": z, "last_kept": z, "last_scores": z}

    def hermes_destroy(self, h):
        pass


def _ours_worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    import argparse
    import bench
    import workloads
    # a tiny stand-in workload under the default name, so that the pools are cheap to generate
    small = workloads.CONFIGS["llava_ov_7b"].scaled(n_layers=2, budget=392, probe_tokens=4)
    workloads.CONFIGS["llava_ov_7b"] = small
    bench.CONFIGS["llava_ov_7b"] = small
    args = argparse.Namespace(gpus=world, steps=3, warmup=3, impl="ours", workload="llava_ov_7b", score_path="auto",
                              reindex="eager", max_position=32768, summary_token=False, no_cpu_baseline=True,
                              no_defer_v=False, no_replay_check=False, budget_weight="", streams=0)
    fake = _FakeHermes()
    out = bench.run_ours(args, backend=_CpuBackend(), hb=fake)
    with open(os.path.join(out_dir, f"o{rank}.json"), "w") as f:
        json.dump({"out": out, "calls": fake.calls}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_run_ours_world2_prints_one_line_with_n_gpus_2(tmp_path):
    port = _free_port()
    mp.spawn(_ours_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r = [json.load(open(tmp_path / f"o{i}.json")) for i in range(2)]
    assert r[1]["out"] is None                              # only rank 0 returns (and prints) the line
    d = r[0]["out"]
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["steps"] == 3 and d["warmup"] == 3
    assert d["config"]["parallelism"].startswith("replicas x2")
    assert d["gpu_launches"] == 4 * 3 and d["replay_check"]["bit_identical"]
    # whole-job value = both ranks' B * L * T over the (max-over-ranks) step time
    wl_T = 392 + 196
    assert d["value"] == pytest.approx(2 * 1 * 2 * wl_T / (d["ms_per_step"] * 1e-3))
    assert r[0]["calls"] == r[1]["calls"] > 0               # both ranks did the same work


def test_bench_gpus_flag_spawns_its_own_ranks():
    """Plain `python bench.py --gpus 2` (no torchrun around it) must launch two ranks itself."""
    env = dict(os.environ, MASTER_PORT=str(_free_port()))
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        env.pop(k, None)
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT, env=env)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2
    # and a WORLD_SIZE that contradicts --gpus is refused
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "3"],
                       capture_output=True, text=True, timeout=60, cwd=ROOT, env=dict(env, WORLD_SIZE="2", RANK="0"))
    assert p.returncode != 0 and "WORLD_SIZE" in p.stderr
