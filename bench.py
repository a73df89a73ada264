#!/usr/bin/env python
"""Benchmark of the HERMES per-chunk KV-cache update (BASELINE.json metric) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one evicting chunk arrival (all rows a0-a7 of SURVEY.md section 8a) on the LLaVA-OV-7B
geometry of BASELINE.json configs[1].  Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import CONFIGS, chunk_kv, probe_q, sweep_point  # noqa: E402

METRIC, UNIT = "kv_tokens_managed_per_s", "tokens/s"
POOL = 16          # distinct pre-generated chunk/probe sets cycled through the timed region
# dram__bytes_read.sum + dram__bytes_write.sum per launch at configs[1], transcribed from the one
# `ncu --set full` capture summarised in profiles/r2_ncu_full_summary.txt (command in profiles/r2_README.md);
# the scoring kernel's figure includes the previous update's V compaction (360 MB) that rides in it
NCU_TRAFFIC_BYTES = {"gather": 181.35e6 + 132.39e6, "score": 561.45e6 + 188.30e6,
                     "select": 1.44e6, "append": 11.25e6}


# ------------------------------------------------------------------------------- shared helpers
def algorithmic_work(wl, n_streams=1):
    """per-update algorithmic flops / bytes of the method (not of our design)."""
    L, T, M, P = wl.n_layers, wl.budget + wl.chunk_tokens, wl.budget, wl.probe_tokens
    n_sh = max(1, (L + 5) // 10)
    Ls = L - n_sh
    es = 2 if wl.dtype == "bf16" else 4
    row = wl.n_kv_heads * wl.head_dim * es
    flops = 2.0 * wl.n_q_heads * P * T * wl.head_dim * Ls * n_streams
    bytes_min = n_streams * (L * (T + 3 * M) * row + Ls * wl.n_q_heads * P * wl.head_dim * es)
    gather_bytes = n_streams * L * 4 * M * row               # kept K,V rows read + written
    return dict(flops=flops, bytes_min=bytes_min, gather_bytes=gather_bytes, T=T, Ls=Ls)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], tensor=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    tensor_burst=d["bf16_tflops"], source="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, tensor=1400.0, tensor_burst=1590.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        rows = [r.split(",") for r in open(self.f.name).read().strip().splitlines() if r.count(",") >= 6]
        os.unlink(self.f.name)
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = [float(r[0]) for r in rows]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].strip().lower().startswith("active") for r in rows)]
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": float(rows[0][1]), "samples": len(rows),
                "power_w_max": max(float(r[2]) for r in rows), "reasons": reasons}


def workload_by_name(name: str):
    """CONFIGS key, or `sweep:<budget>:<probe>` for a point of BASELINE.json configs[3]."""
    if name.startswith("sweep:"):
        _, m, p = name.split(":")
        return sweep_point(int(m), int(p))
    return CONFIGS[name]


def cfg_index(name: str) -> int:
    return 3 if name.startswith("sweep") else {"toy": 0, "llava_ov_7b": 1, "llava_ov_7b_c16": 1, "qwen25_vl_7b": 2, "batched_72b": 4}[name]


def cfg_label(name: str) -> str:
    if name == "llava_ov_7b_c16":
        return "SURVEY.md 8(d) row 2b (BASELINE.json configs[1] geometry, the paper's 16-frame chunk)"
    return f"BASELINE.json configs[{cfg_index(name)}]"


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(ms: float, world: int, device=None) -> float:
    """Slowest rank's time (all_reduce MAX); identity for one process."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(wl, world: int, streams_per_rank: int, ms_per_step: float) -> float:
    """Whole-job KV tokens managed per second: all ranks' B*L*T over the slowest rank's step time."""
    T = wl.budget + wl.chunk_tokens
    return world * streams_per_rank * wl.n_layers * T / (ms_per_step * 1e-3)


def make_pool(wl, rank: int, n_sets: int):
    """Seeded chunk / probe sets [B, L, ...] as fp32 numpy (storage-representable values)."""
    B = wl.n_streams
    sets = []
    for u in range(n_sets):
        per = [chunk_kv(wl, rank * B + b, 1000 + u, (1000 + u) * wl.chunk_tokens, wl.chunk_tokens) for b in range(B)]
        K = np.stack([p[0] for p in per]); V = np.stack([p[1] for p in per])
        Q = np.stack([probe_q(wl, rank * B + b, 1000 + u) for b in range(B)])
        sets.append((K, V, Q))
    return sets


# ------------------------------------------------------------------------------- our arm (CUDA)
class CudaBackend:
    """The device plumbing run_ours needs from torch: memory, events, synchronisation, the process group.
    tests/test_bench_multirank.py substitutes a CPU / gloo stand-in to run the N > 1 path without GPUs."""
    dist_backend = "nccl"

    def __init__(self, local_rank: int):
        import torch
        self.torch = torch
        torch.cuda.set_device(local_rank)
        self.dev = torch.device("cuda", local_rank)

    def init_process_group(self, dist):
        dist.init_process_group(self.dist_backend, device_id=self.dev)

    def event(self):
        return self.torch.cuda.Event(enable_timing=True)

    def synchronize(self):
        self.torch.cuda.synchronize()

    def stream_synchronize(self):
        self.torch.cuda.current_stream().synchronize()

    def pin(self, t):
        return t.pin_memory()


def run_ours(args, backend=None, hb=None):
    import torch
    import torch.distributed as dist
    if hb is None:
        import paper_2601_14724_b200 as hb

    rank, local_rank, world = dist_env()
    be = backend if backend is not None else CudaBackend(local_rank)
    if world > 1 and not dist.is_initialized():
        be.init_process_group(dist)
    dev = be.dev
    wl = workload_by_name(args.workload)
    if args.streams > 0:                                     # independent streams advanced by one call (one handle)
        wl = wl.scaled(n_streams=args.streams)
    B = wl.n_streams
    tdt = torch.bfloat16 if wl.dtype == "bf16" else torch.float32
    over = dict(score_path={"auto": 0, "simt": 1, "tcgen05": 2}[args.score_path])
    if args.reindex == "lazy":                               # the paper's default for streaming
        over.update(reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=args.max_position)
    if args.summary_token:
        over.update(summary_token=1)
    if args.no_defer_v:
        over.update(defer_v=0)
    lb = None
    if args.budget_weight:                                   # layer-dependent budgets (Tab. 5)
        lb = tuple(float(x) for x in args.budget_weight.split(","))
        assert len(lb) == 3, "--budget-weight takes shallow,middle,deep"
        over.update(budget_weight=lb, max_tokens=0)
    cfg = hb.config_for_workload(wl, device=local_rank, **over)
    h = hb.hermes_create(cfg)
    fill_to = max(hb.hermes_layer_budgets(cfg)) if lb else wl.budget   # every layer holds at least its budget before timing

    host_pool = [tuple(be.pin(torch.from_numpy(x).to(tdt)) for x in s) for s in make_pool(wl, rank, POOL)]
    dev_pool = [tuple(x.to(dev) for x in s) for s in host_pool]
    # fill to the budget without a probe (no eviction), then W warm evicting updates
    n_fill, rem = divmod(fill_to, wl.chunk_tokens)

    def fill(hh):
        for i in range(n_fill):
            K, V, _ = dev_pool[i % POOL]
            hb.hermes_append_chunk(hh, K, V, None)
        if rem:                                              # budget not a multiple of the chunk: one partial append
            K, V, _ = dev_pool[n_fill % POOL]
            hb.hermes_append_chunk(hh, K[:, :, :rem].contiguous(), V[:, :, :rem].contiguous(), None)
        assert hb.hermes_len(hh) == fill_to

    fill(h)

    def barrier():
        be.synchronize()
        if world > 1:
            dist.barrier()
        be.synchronize()

    def timed(n, fn):
        e0, e1 = be.event(), be.event()
        barrier()
        e0.record()
        for i in range(n):
            fn(i)
        e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, dev) / n

    replay = []                                              # pool index of every evicting update, in order

    def dev_step(i):
        K, V, Q = dev_pool[i % POOL]
        hb.hermes_append_chunk(h, K, V, Q)
        replay.append(i % POOL)

    for i in range(max(args.warmup, 3)):
        dev_step(i)
    sampler = ClockSampler(local_rank) if rank == 0 and backend is None else None
    ms = timed(args.steps, dev_step)
    clocks = sampler.stop() if sampler else None
    launches = hb.hermes_last_launch_count(h) * args.steps
    score_path = {1: "simt", 2: "tcgen05"}.get(hb.hermes_last_score_path(h), "none")

    # per-kernel durations: CUDA events recorded by the library on the launch stream, same steps
    hb.hermes_set_profiling(h, True)
    n_prof = min(args.steps, 32)
    acc = {}
    for i in range(n_prof):
        dev_step(i)
        for k, v in hb.hermes_get_profile(h).items():
            acc[k] = acc.get(k, 0.0) + v / n_prof
    hb.hermes_set_profiling(h, False)

    # end to end: HOST (pinned) inputs, H2D + update + D2H of the kept index lists inside the timed region
    # two updates in flight: the caller consumes the kept lists of update i - 1 (its own pinned buffer) while update i,
    # whose inputs are crossing PCIe, is enqueued behind it
    kept_host = [be.pin(torch.zeros(B, wl.n_layers, wl.budget, dtype=torch.int32)) for _ in range(2)]
    done = [None, None]

    def host_step(i):
        K, V, Q = host_pool[i % POOL]
        # (with layer-dependent budgets the lists have per-layer lengths and the host entry point does not return them)
        hb.hermes_append_chunk_host(h, K, V, Q, kept_out=None if lb else kept_host[i & 1])
        replay.append(i % POOL)
        done[i & 1] = be.event()
        done[i & 1].record()
        if done[(i & 1) ^ 1] is not None:
            done[(i & 1) ^ 1].synchronize()                  # update i - 1 is complete: its kept lists are on the host

    n_e2e = min(args.steps, 64)
    for i in range(3):
        host_step(i)
    ms_e2e = timed(n_e2e, host_step)
    # bytes the library moves per call: K, V and the probe slices of the scored layers (shallow layers' slices are never read;
    # n_shallow defaults to max(1, round(0.1 L)), include/hermes.h)
    n_shallow = max(1, (wl.n_layers + 5) // 10)
    Kh, Vh, Qh = host_pool[0]
    h2d = (Kh.numel() * Kh.element_size() + Vh.numel() * Vh.element_size()
           + Qh.numel() * Qh.element_size() * (wl.n_layers - n_shallow) // wl.n_layers)
    d2h = 0 if lb else kept_host[0].numel() * 4
    rides = bool(hb.hermes_v_pending(h))

    # outside every timed region: the cache the timed updates left behind must equal, bit for bit, the cache of a
    # handle that never defers a compaction (defer_v = 0; that configuration is the one the lock-step
    # oracle tests check) after the same sequence of updates
    check = None
    if not args.no_replay_check:
        h2 = hb.hermes_create(hb.config_for_workload(wl, device=local_rank, **dict(over, defer_v=0)))
        fill(h2)
        for j in replay:
            K, V, Q = dev_pool[j]
            hb.hermes_append_chunk(h2, K, V, Q)
        be.synchronize()
        bad = 0
        for b in range(B):
            for l in range(wl.n_layers):
                va, vb = hb.hermes_get_cache(h, b, l), hb.hermes_get_cache(h2, b, l)
                bad += sum(0 if torch.equal(va[k], vb[k]) else 1 for k in ("k", "v", "pos", "last_kept", "last_scores"))
        check = {"updates_replayed": len(replay), "against": "defer_v=0 handle, same inputs",
                 "tensors_compared": 5 * B * wl.n_layers, "mismatching_tensors": bad, "bit_identical": bad == 0}
        hb.hermes_destroy(h2)
        if bad:
            raise SystemExit(f"bench.py: the timed handle's cache differs from the non-deferring replay in {bad} tensors")

    if rank != 0:
        hb.hermes_destroy(h)
        return None
    work = algorithmic_work(wl, B)
    row_b = wl.n_kv_heads * wl.head_dim * (2 if wl.dtype == "bf16" else 4)
    ws_mb = B * wl.n_layers * 2 * work["T"] * row_b / 1e6          # K and V slabs read (scoring + gather)
    wr_mb = B * wl.n_layers * 2 * wl.budget * row_b / 1e6            # compacted K and V written
    pk = peaks()
    sm = clocks.get("sm_mhz") if clocks else None
    kern = {k: v for k, v in acc.items() if v > 0}
    if score_path == "tcgen05" and "score_stats" in kern:      # one persistent kernel runs both scoring passes
        kern["score"] = kern.pop("score_stats")
    dom = max(kern, key=kern.get)
    t_dom = kern[dom] * 1e-3
    traffic = NCU_TRAFFIC_BYTES.get(dom) if args.workload == "llava_ov_7b" else None
    if dom == "gather" or dom == "append":
        ach = work["gather_bytes"] / 2 / t_dom / 1e9          # K-only launch (V is moved inside the scoring kernel)
        roof = dict(kernel=dom, bound="hbm", achieved=ach, peak=pk["hbm"], unit="GB/s", frac=ach / pk["hbm"], traffic=traffic)
    elif dom == "score":
        # a1's contraction is the tensor-core work of the path: algorithmic 2 H_q P T d L_s flops per
        # launch against the sustained bf16 peak.  The launch also evaluates exp2 on the XU pipe (16 results / clk / SM):
        # the method needs H_q P T L_s of them, the two-pass design evaluates twice that -- both reported beside it.
        n_exp_method = work["flops"] / (2.0 * wl.head_dim)
        sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
        xu_peak = 16 * 148 * sm_max * 1e6 / 1e9
        ach = work["flops"] / t_dom / 1e12
        roof = dict(kernel=dom, bound="tensor", achieved=ach, peak=pk["tensor"], unit="TFLOP/s", frac=ach / pk["tensor"], traffic=traffic,
                    exp2={"peak_gexp2_s": xu_peak, "method_gexp2_s": n_exp_method / t_dom / 1e9, "method_frac": n_exp_method / t_dom / 1e9 / xu_peak,
                          "design_gexp2_s": 2 * n_exp_method / t_dom / 1e9, "design_frac": 2 * n_exp_method / t_dom / 1e9 / xu_peak,
                          "note": "XU pipe, 16 exp2/clk/SM x 148 SMs x clocks.max.sm; the design evaluates 2 exp2 per (probe row, token)"},
                    rides="the previous update's V compaction is moved inside this launch" if rides else None)
    elif dom in ("score_stats", "score_colsum"):
        ach = work["flops"] / t_dom / 1e12
        roof = dict(kernel=dom, bound="tensor", achieved=ach, peak=pk["tensor"], unit="TFLOP/s", frac=ach / pk["tensor"], traffic=traffic)
    else:
        ach = wl.n_layers * B * work["T"] * 4 * 3 / t_dom / 1e9
        roof = dict(kernel=dom, bound="hbm", achieved=ach, peak=pk["hbm"], unit="GB/s", frac=ach / pk["hbm"], traffic=traffic)
    roof["peak_source"] = pk["source"]
    t_roof = max(work["bytes_min"] / (pk["hbm"] * 1e9), work["flops"] / (pk["tensor"] * 1e12))
    # third floor, not part of north_star's roofline but the binding one on the tcgen05 path: the two-pass softmax column
    # sum needs 2 exp2 per (probe row, token) at 16 / clk / SM
    exp2_floor = (2.0 * work["flops"] / (2.0 * wl.head_dim)) / (16 * 148 * ((clocks or {}).get("sm_max_mhz") or 1965.0) * 1e6)
    step_roof = dict(bound="hbm" if work["bytes_min"] / (pk["hbm"] * 1e9) >= work["flops"] / (pk["tensor"] * 1e12) else "tensor",
                     roofline_us=t_roof * 1e6, measured_us=ms * 1e3, frac=t_roof / (ms * 1e-3),
                     bytes_min=work["bytes_min"], flops=work["flops"],
                     exp2_floor_us=exp2_floor * 1e6 if score_path == "tcgen05" else None)
    out = {
        "metric": METRIC, "value": job_value(wl, world, B, ms), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "chunk_update_latency_us": ms * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": wl.dtype, "data": "synthetic",
        "config": {"workload": f"{cfg_label(wl.name)} {wl.name}: L{wl.n_layers} Hq{wl.n_q_heads}/Hkv{wl.n_kv_heads} "
                               f"d{wl.head_dim} {wl.dtype}, budget {wl.budget}, chunk {wl.chunk_tokens}, probe {wl.probe_tokens}, "
                               f"T {work['T']}", "streams_per_gpu": B, "parallelism": f"replicas x{world} (independent streams, no collective)",
                   "l2": (f"cache slabs touched per step: {ws_mb:.0f} MB read + {wr_mb:.0f} MB written "
                          + ("(exceeds the 126 MB L2)" if ws_mb + wr_mb > 252 else "(comparable to the 126 MB L2: no flush, L2-assisted)")
                          + f"; inputs cycle through {POOL} chunk/probe sets"),
                   "score_path": score_path, "reindex": args.reindex, "summary_token": bool(args.summary_token),
                   **({"budget_weight": list(lb), "layer_budgets_min_max": [min(hb.hermes_layer_budgets(cfg)), max(hb.hermes_layer_budgets(cfg))]} if lb else {})},
        "e2e": {"value": job_value(wl, world, B, ms_e2e), "unit": UNIT, "ms_per_step": ms_e2e,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": n_e2e},
        "gpu_launches": launches,
        "kernel_ms": kern,
        "roofline": roof,
        "roofline_step": step_roof,
        "replay_check": check,
        "clocks": clocks,
    }
    hb.hermes_destroy(h)
    return out


# ------------------------------------------------------------------------------- oracle timing (CPU)
def oracle_sample(wl, steps: int, n_layers_sample: int, warmup: int = 0):
    """Times oracle_step, as it stands, on a bounded sample: the full-geometry cache (budget, chunk, probe,
    heads, head_dim) with `n_layers_sample` layers, in steady state.  Returns (seconds per step, threads)."""
    from oracle import hermes_oracle as ho
    swl = wl.scaled(n_layers=n_layers_sample, n_streams=1)
    cfg = ho.OracleConfig(n_layers=swl.n_layers, n_q_heads=swl.n_q_heads, n_kv_heads=swl.n_kv_heads,
                          head_dim=swl.head_dim, budget=swl.budget, forget_rate=swl.k_forget, dtype=swl.dtype,
                          rope_mode=swl.rope_mode, rope_theta=swl.rope_theta, mrope_section=swl.mrope_section,
                          mrope_compact_axes=swl.mrope_compact_axes, pos_offset=swl.pos_offset, capacity=swl.cap)
    st = ho.OracleStream(cfg)
    K, V, _ = chunk_kv(swl, 0, 0, 0, swl.budget)
    ho.oracle_step(st, K, V, None)
    times = []
    for u in range(warmup + steps):
        K, V, _ = chunk_kv(swl, 0, 1 + u, swl.budget + u * swl.chunk_tokens, swl.chunk_tokens)
        Q = probe_q(swl, 0, 1 + u)
        t0 = time.perf_counter()
        ho.oracle_step(st, K, V, Q)
        times.append(time.perf_counter() - t0)
    times = times[warmup:]
    try:
        from threadpoolctl import threadpool_info
        threads = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        threads = len(os.sched_getaffinity(0))
    return sum(times) / len(times), threads, swl


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return None
    wl = workload_by_name(args.workload)
    Ls = 4                                                   # 1 shallow + 2 middle + 1 deep (10/60/30 % rule at L = 4)
    sec, threads, swl = oracle_sample(wl, args.steps, Ls, warmup=min(args.warmup, 2))
    T = wl.budget + wl.chunk_tokens
    val = Ls * T / sec
    sample = (f"oracle_step on {Ls} of {wl.n_layers} layers (1 shallow, 2 middle, 1 deep) of the full-geometry cache "
              f"(T {T}, budget {wl.budget}, probe {wl.probe_tokens}), steady state, per step")
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": min(args.warmup, 2), "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[1] {wl.name} (bounded sample: {Ls} layers)"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=256)   # BASELINE.json configs[1]: 256 timed chunk arrivals
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="llava_ov_7b", help="one of %s, or sweep:<budget>:<probe>" % sorted(CONFIGS))
    ap.add_argument("--score-path", default="auto", choices=["auto", "simt", "tcgen05"])
    ap.add_argument("--reindex", default="eager", choices=["eager", "lazy"])
    ap.add_argument("--max-position", type=int, default=32768, help="lazy re-indexing: the model's position limit")
    ap.add_argument("--streams", type=int, default=0, help="streams per GPU advanced by one call (0: the workload's own count)")
    ap.add_argument("--summary-token", action="store_true")
    ap.add_argument("--budget-weight", default="", help="layer-dependent budgets: shallow,middle,deep weights (PAPER.md Tab. 5), e.g. 1.3,1.0,0.7")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-defer-v", action="store_true", help="compact V in the gather kernel instead of inside the next scoring launch")
    ap.add_argument("--no-replay-check", action="store_true", help="skip the post-timing bit-equality check against a non-deferring handle")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: launch the N ranks ourselves (one process per GPU), same as the driver's torchrun line
        if args.impl == "ours":
            import torch
            n_dev = torch.cuda.device_count()
            if n_dev < args.gpus:
                raise SystemExit(f"bench.py --gpus {args.gpus}: only {n_dev} CUDA device(s) visible")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", os.environ.get("MASTER_PORT", "29531"), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if "WORLD_SIZE" in os.environ and int(os.environ["WORLD_SIZE"]) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ['WORLD_SIZE']}")
    if args.impl == "reference":
        out = run_reference(args)
    else:
        out = run_ours(args)
        rank, _, world = dist_env()
        if out is not None and world == 1 and not args.no_cpu_baseline:
            wl = workload_by_name(args.workload)
            sec, threads, swl = oracle_sample(wl, 2, wl.n_layers)       # two full-size oracle updates
            T = wl.budget + wl.chunk_tokens
            out["cpu_baseline"] = {"value": wl.n_layers * T / sec, "unit": UNIT, "cores": threads, "kind": "oracle",
                                   "ms_per_step": sec * 1e3,
                                   "sample": f"2 full-size oracle_step updates of one stream ({wl.n_layers} layers, T {T}) in steady state"}
    if out is not None:
        print(json.dumps(out))


if __name__ == "__main__":
    main()
