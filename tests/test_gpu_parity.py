"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, lock-step, on the seeded
workloads of BASELINE.json (`configs[0..4]`, full size where the oracle finishes in seconds)."""
import numpy as np
import pytest
import torch

import paper_2601_14724_b200 as hb
from gpu_harness import LockStep, to_dev
from workloads import CONFIGS, rope_at_arrival, sweep_point

pytestmark = pytest.mark.gpu


def _run(wl, n_checked, n_warm=0, cfg_over=None, oracle_over=None, streams=None):
    ls = LockStep(wl, cfg_over, oracle_over, streams)
    try:
        ls.fill()
        for _ in range(n_warm):
            ls.step(check=False)
        reps = []
        for _ in range(n_checked):
            reps += ls.step(check=True)
        assert hb.hermes_device_status(ls.h) == 0
        return ls, reps
    except Exception:
        ls.close()
        raise


def test_toy_config_all_ten_updates():
    """configs[0]: preload 128, ten scored arrivals (T = 160 then 128), every one checked."""
    wl = CONFIGS["toy"]
    ls, reps = _run(wl, 10)
    assert [r["T"] for r in reps] == [160] + [128] * 9
    assert hb.hermes_last_score_path(ls.h) == hb.HERMES_SCORE_SIMT        # fp32 cache -> CUDA-core path
    # end to end on the GPU state: every retained key == RoPE(k0[id], offset + slot) (rotation composition)
    fd = ls.feeders[0]
    for l in range(wl.n_layers):
        v = hb.hermes_get_cache(ls.h, 0, l)
        k0 = np.stack([fd.k0_by_id[int(t)][l] for t in ls.ids[0][l]])[None]
        ref = rope_at_arrival(k0, np.arange(wl.budget)[None, :], wl)[0]
        np.testing.assert_allclose(v["k"].float().cpu().numpy(), ref, atol=2e-5)
        assert v["pos"].cpu().numpy()[0].tolist() == list(range(wl.budget))
    ls.close()


def test_llava_geometry_reduced_multi_tile_ragged():
    """LLaVA-OV-7B geometry, fewer layers / smaller budget: T = 1764 spans 13.8 token tiles."""
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=10, budget=1568, probe_tokens=24)
    ls, reps = _run(wl, 3, n_warm=1)
    assert all(r["max_score_rel"] < 1e-3 for r in reps)
    ls.close()


def test_llava_ov_7b_full_size():
    """configs[1] at full size, 2 lock-step updates.  Every checked update starts from a flushed cache
    (hermes_get_cache runs a pending compaction), so the scoring launch here carries no movers; the launch
    bench.py times is checked by test_timed_launch_configuration_full_size."""
    wl = CONFIGS["llava_ov_7b"]
    ls, reps = _run(wl, 2, n_warm=2)
    assert all(r["T"] == 6468 for r in reps)
    ls.close()


def _raw_steps_vs_lockstep(wl, n_steps, over=None, oover=None):
    """The launch configuration bench.py times: `n_steps` consecutive evicting updates through hermes_append_chunk
    with NO hermes_get_cache in between, so that the previous update's V compaction rides in every scoring
    launch (tc_v_mover warp, 32 KB staging ring, 2-stage K ring).  The final cache must equal, bit for bit, the cache
    of a handle that never defers (defer_v = 0) and is compared with the oracle, lock-step, at every step on the same
    inputs."""
    over, oover = dict(over or {}), dict(oover or {})
    a = LockStep(wl, cfg_over=over, oracle_over=oover)
    a.fill()
    pend = []
    for _ in range(n_steps):
        a.raw_step()
        pend.append(hb.hermes_v_pending(a.h))
    torch.cuda.synchronize()
    assert hb.hermes_last_score_path(a.h) == hb.HERMES_SCORE_TCGEN05
    got = [[{k: t.clone() for k, t in hb.hermes_get_cache(a.h, b, l).items() if torch.is_tensor(t)}
            for l in range(wl.n_layers)] for b in range(wl.n_streams)]
    assert hb.hermes_v_pending(a.h) == 0 and hb.hermes_device_status(a.h) == 0
    a.close()
    ref = LockStep(wl, cfg_over=dict(over, defer_v=0), oracle_over=oover)
    ref.fill()
    for _ in range(n_steps):
        ref.step(check=True)
    for b in range(wl.n_streams):
        for l in range(wl.n_layers):
            v = hb.hermes_get_cache(ref.h, b, l)
            for key in ("k", "v", "pos", "last_kept", "last_scores"):
                assert torch.equal(v[key], got[b][l][key]), (b, l, key)
    ref.close()
    return pend


def test_timed_launch_configuration_full_size():
    """configs[1] at full size exactly as bench.py runs it: 5 back-to-back evicting updates, the V mover riding
    (~1190 rows = 37 batches per CTA, ~34 K tiles per CTA through the 2-stage ring)."""
    pend = _raw_steps_vs_lockstep(CONFIGS["llava_ov_7b"], 5)
    assert all(v == 1 for v in pend)                       # V always rides in the next scoring launch


def test_timed_launch_configuration_reduced_variants():
    """Same protocol on reduced geometries: M-RoPE (three delta axes), the summary token slot, lazy re-indexing
    (pure copies), a chunk that is not a multiple of anything, and B > 1 streams."""
    _raw_steps_vs_lockstep(CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=784, probe_tokens=64), 4)
    _raw_steps_vs_lockstep(CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=784, probe_tokens=64), 3,
                           over=dict(summary_token=1), oover=dict(summary_token=True))
    _raw_steps_vs_lockstep(CONFIGS["qwen25_vl_7b"].scaled(n_layers=6, budget=1024, probe_tokens=64, pos_offset=5), 3)
    _raw_steps_vs_lockstep(CONFIGS["batched_72b"].scaled(n_layers=5, n_streams=3, budget=1177, probe_tokens=48), 3)
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=6, budget=784, probe_tokens=64)
    mp = 784 + 196 * 4                                      # the 3rd update re-indexes, the others copy
    _raw_steps_vs_lockstep(wl, 5, over=dict(reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=mp),
                           oover=dict(reindex_mode="lazy", max_position=mp, max_chunk_span=wl.chunk_tokens))


def test_llava_ov_7b_16_frame_chunk_full_size():
    """the paper's 16-frame chunk (3136 tokens) at configs[1] geometry --
    every update evicts a third of the cache; T = 9408 = 73.5 token tiles."""
    wl = CONFIGS["llava_ov_7b_c16"]
    ls, reps = _run(wl, 2, n_warm=1)
    assert all(r["T"] == 9408 for r in reps)
    assert hb.hermes_last_score_path(ls.h) == hb.HERMES_SCORE_TCGEN05
    ls.close()


def test_qwen25_vl_mrope_reduced_and_all_axes():
    wl = CONFIGS["qwen25_vl_7b"].scaled(n_layers=6, budget=1024, probe_tokens=32, pos_offset=5)
    ls, reps = _run(wl, 3, n_warm=1)
    ls.close()
    wl_all = wl.scaled(mrope_compact_axes=0b111)
    ls, reps = _run(wl_all, 2)
    ls.close()


def test_qwen25_vl_7b_full_size():
    """configs[2] at full size: M-RoPE, budget 8192, chunk 128, 128 probe tokens; 1 lock-step update."""
    ls, reps = _run(CONFIGS["qwen25_vl_7b"], 1, n_warm=1)
    assert reps[0]["T"] == 8320
    ls.close()


def test_sweep_corners_reduced_layers():
    """configs[3] corners (budget 2K / P 16 and budget 4K / P 256) on 6 layers."""
    for budget, probe in ((2048, 16), (4096, 256)):
        wl = sweep_point(budget, probe).scaled(n_layers=6)
        ls, _ = _run(wl, 1, n_warm=1)
        ls.close()


def test_sweep_32k_budget_point_full_layers():
    """configs[3], the largest budget (32 768 tokens per layer, T = 32 964) at all 28 layers with 64 probe rows:
    k_select with 129 KB of dynamic shared memory and 2 flag chunks per thread, 258 token tiles per group."""
    wl = sweep_point(32768, 64)
    ls, reps = _run(wl, 1)
    assert reps[0]["T"] == 32768 + 196 and hb.hermes_last_score_path(ls.h) == hb.HERMES_SCORE_TCGEN05
    ls.close()


def test_batched_72b_full_size_schedule():
    """configs[4] at full size (80 layers x 16 streams, 64 q / 8 kv heads, budget 4096): SURVEY.md 8(d)'s parity
    schedule -- streams {0, 7, 15} compared with the oracle on 2 evicting updates (the second one with the first
    one's V compaction pending until the lock-step download flushes it)."""
    wl = CONFIGS["batched_72b"]
    ls, reps = _run(wl, 2, streams=[0, 7, 15])
    assert len(reps) == 6 and all(r["T"] == 4096 + 196 for r in reps)
    assert hb.hermes_last_score_path(ls.h) == hb.HERMES_SCORE_TCGEN05
    ls.close()


def test_batched_72b_geometry_reduced_equals_single_streams():
    """configs[4] geometry (64 q / 8 kv heads), 3 streams x 8 layers: oracle parity per stream, and the
    batched call equals B single-stream calls bit for bit."""
    wl = CONFIGS["batched_72b"].scaled(n_layers=8, n_streams=3, budget=784)
    ls, reps = _run(wl, 2, n_warm=1)
    batched = [[{k: t.clone() for k, t in hb.hermes_get_cache(ls.h, b, l).items() if torch.is_tensor(t)}
                for l in range(wl.n_layers)] for b in range(3)]
    ls.close()
    for b in (0, 2):
        single = wl.scaled(n_streams=1)
        one = LockStep(single)
        one.feeders[0].stream = b                                     # same seeded inputs as stream b
        one.fill(); one.step(check=False); one.step(check=False); one.step(check=False)
        torch.cuda.synchronize()
        for l in range(wl.n_layers):
            v = hb.hermes_get_cache(one.h, 0, l)
            for key in ("k", "v", "pos", "last_kept", "last_scores"):
                assert torch.equal(v[key], batched[b][l][key]), (b, l, key)
        one.close()


def test_edge_cases_small():
    wl = CONFIGS["toy"].scaled(preload_tokens=0, capacity=0, chunk_tokens=32)
    # (a) below budget and without a probe nothing is evicted; (b) evicting exactly one token; (c) one probe row
    ls = LockStep(wl)
    ls.step(check=True, n_new=32)                 # T = 32 <= 96: append only, even with a probe
    ls.step(check=True, n_new=32)
    ls.step(check=True, n_new=32)                 # T = 96 == budget: still no eviction
    assert hb.hermes_len(ls.h) == 96
    r = ls.step(check=True, n_new=1, n_probe=1)   # T = 97: evict exactly one token, single probe row
    assert r[0]["evicted"] and hb.hermes_len(ls.h) == 96
    r = ls.step(check=True, n_new=32, n_probe=3)
    # capacity: len 96 + 33 > 128
    K = torch.zeros(1, wl.n_layers, 33, wl.n_kv_heads, wl.head_dim, device="cuda")
    with pytest.raises(hb.HermesError) as e:
        hb.hermes_append_chunk(ls.h, K, K, None)
    assert e.value.code == hb.HERMES_ECAPACITY and hb.hermes_len(ls.h) == 96
    # explicit pos_start jump: deltas leave the rotary table -> fp64 slow path, still within tolerance
    r = ls.step(check=True, n_new=32, pos_start=5000)
    assert hb.hermes_device_status(ls.h) & 2
    with pytest.raises(hb.HermesError):           # positions must stay above the cache
        ls.step(check=False, n_new=8, pos_start=3)
    ls.close()


@pytest.mark.parametrize("over,oover", [
    (dict(norm_mode=hb.HERMES_NORM_SUM), dict(norm_mode="sum")),
    (dict(lambda_shallow=0.0, lambda_middle=0.0, lambda_deep=0.0), dict(lambda_shallow=0.0, lambda_middle=0.0, lambda_deep=0.0)),
    (dict(n_shallow=4, n_deep=0, lambda_shallow=0.0), dict(n_shallow=4, n_deep=0, lambda_shallow=0.0)),   # FIFO
    (dict(pos_offset=13), dict(pos_offset=13)),
    (dict(softmax_scale=0.05, omega0=0.5, gamma=0.2, forget_rate=0.3), dict(softmax_scale=0.05, omega0=0.5, gamma=0.2, forget_rate=0.3)),
])
def test_hyperparameter_variants(over, oover):
    wl = CONFIGS["toy"]
    if "pos_offset" in over:
        wl, over, oover = wl.scaled(pos_offset=13), {}, {}
    ls, reps = _run(wl, 3, cfg_over=over, oracle_over=oover)
    if over.get("n_shallow") == 4:                 # pure recency everywhere: sliding window of PAPER.md:49
        newest = np.arange(ls.feeders[0].tokens_fed - wl.budget, ls.feeders[0].tokens_fed)
        assert (ls.ids[0] == newest[None, :]).all()
    ls.close()


def test_determinism_and_host_api():
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=5, budget=784, probe_tokens=8)

    def run(host: bool):
        ls = LockStep(wl)
        ls.fill()
        kept = torch.zeros(1, wl.n_layers, wl.budget, dtype=torch.int32).pin_memory()
        for _ in range(3):
            K, V, Q, ids = ls._gen(wl.chunk_tokens, True)
            if host:
                args = [torch.from_numpy(x).to(torch.bfloat16).pin_memory() for x in (K, V, Q)]
                hb.hermes_append_chunk_host(ls.h, *args, kept_out=kept)
            else:
                hb.hermes_append_chunk(ls.h, to_dev(K, "bf16"), to_dev(V, "bf16"), to_dev(Q, "bf16"))
            torch.cuda.synchronize()
        out = [{k: t.clone() for k, t in hb.hermes_get_cache(ls.h, 0, l).items() if torch.is_tensor(t)}
               for l in range(wl.n_layers)]
        ls.close()
        return out, kept.clone()

    a, _ = run(False)
    b, _ = run(False)
    c, kept = run(True)
    for l in range(wl.n_layers):
        for key in ("k", "v", "pos", "last_kept", "last_scores"):
            assert torch.equal(a[l][key], b[l][key])          # same inputs -> same bits
            assert torch.equal(a[l][key], c[l][key])          # host-buffer entry point == device entry point
        assert torch.equal(kept[0, l].cuda(), a[l]["last_kept"])


def test_host_entry_point_fill_and_batched_streams():
    """Host-buffer entry point on the paths the test above does not reach: appends without a probe (no eviction:
    the V rows arrive through the late, V-only append) and B > 1 streams; caches must equal the device entry point's."""
    wl = CONFIGS["batched_72b"].scaled(n_layers=4, n_streams=2, budget=392, probe_tokens=8)
    from workloads import chunk_kv, probe_q
    pool = []
    for u in range(4):                                   # two fills, then two evicting updates
        per = [chunk_kv(wl, b, u, u * wl.chunk_tokens, wl.chunk_tokens) for b in range(wl.n_streams)]
        K = np.stack([p[0] for p in per]); V = np.stack([p[1] for p in per])
        Q = np.stack([probe_q(wl, b, u) for b in range(wl.n_streams)]) if u >= 2 else None
        pool.append((K, V, Q))

    def run(host: bool):
        h = hb.hermes_create(hb.config_for_workload(wl))
        for K, V, Q in pool:
            if host:
                args = [None if x is None else torch.from_numpy(x).to(torch.bfloat16).pin_memory() for x in (K, V, Q)]
                hb.hermes_append_chunk_host(h, *args)
            else:
                hb.hermes_append_chunk(h, to_dev(K, "bf16"), to_dev(V, "bf16"), None if Q is None else to_dev(Q, "bf16"))
            torch.cuda.synchronize()
        out = [[{k: t.clone() for k, t in hb.hermes_get_cache(h, b, l).items() if torch.is_tensor(t)}
                for l in range(wl.n_layers)] for b in range(wl.n_streams)]
        n = hb.hermes_len(h)
        hb.hermes_destroy(h)
        return out, n

    a, na = run(False)
    b, nb = run(True)
    assert na == nb == wl.budget
    for s in range(wl.n_streams):
        for l in range(wl.n_layers):
            for key in ("k", "v", "pos", "last_kept"):
                assert torch.equal(a[s][l][key], b[s][l][key]), (s, l, key)


def test_lazy_reindexing_toy_and_bf16():
    """DESIGN f2: lazy mode copies kept keys bit for bit and keeps their original indices;
    the step after which the next chunk would cross max_position re-indexes exactly like the eager path."""
    wl = CONFIGS["toy"]
    ls, reps = _run(wl, 10, cfg_over=dict(reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=300),
                    oracle_over=dict(reindex_mode="lazy", max_position=300, max_chunk_span=wl.chunk_tokens))
    fd = ls.feeders[0]
    for l in range(wl.n_layers):                    # every key == RoPE(k0[id], its current position)
        v = hb.hermes_get_cache(ls.h, 0, l)
        pos = v["pos"].cpu().numpy().astype(np.int64)
        k0 = np.stack([fd.k0_by_id[int(t)][l] for t in ls.ids[0][l]])[None]
        ref = rope_at_arrival(k0, pos, wl)[0]
        np.testing.assert_allclose(v["k"].float().cpu().numpy(), ref, atol=3e-5)
        assert (np.diff(pos[0]) > 0).all() and pos.max() < 300
    ls.close()
    # bf16, multi-tile, tcgen05 scoring; max_position chosen so that the 4th checked update re-indexes
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=6, budget=784, probe_tokens=16)
    mp = 784 + 196 * 5
    ls, reps = _run(wl, 6, cfg_over=dict(reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=mp),
                    oracle_over=dict(reindex_mode="lazy", max_position=mp, max_chunk_span=wl.chunk_tokens))
    v = hb.hermes_get_cache(ls.h, 0, 0)
    assert int(v["pos"].max()) < mp
    assert sum(r["k_mismatch_bits"] for r in reps) == 0
    ls.close()


def test_summary_token_toy_and_bf16():
    """DESIGN f1 (Alg. 1): deep layers keep |M| - 1 tokens and append the summary of the evicted ones."""
    wl = CONFIGS["toy"]
    ls, reps = _run(wl, 6, cfg_over=dict(summary_token=1), oracle_over=dict(summary_token=True))
    assert all(r.get("summary_layers") == 1 for r in reps)                     # 4 layers: one deep
    assert (ls.ids[0][3] == -1).sum() >= 1 and (ls.ids[0][:3] >= 0).all()
    ls.close()
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=784, probe_tokens=16)    # 1 shallow, 4 middle, 2 deep
    ls, reps = _run(wl, 3, n_warm=1, cfg_over=dict(summary_token=1), oracle_over=dict(summary_token=True))
    assert all(r.get("summary_layers") == 2 for r in reps)
    ls.close()


def test_summary_token_under_lazy_reindexing():
    """The paper's streaming configuration of the management path: lazy re-indexing with the
    deep-layer summary token at every compression step.  Kept keys are copied, the summary token is
    aligned to the position after the newest token; the re-index step in the middle re-rotates everything."""
    wl = CONFIGS["toy"]
    ls, reps = _run(wl, 8, cfg_over=dict(summary_token=1, reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=300),
                    oracle_over=dict(summary_token=True, reindex_mode="lazy", max_position=300, max_chunk_span=wl.chunk_tokens))
    assert all(r.get("summary_layers") == 1 for r in reps)
    pos = hb.hermes_get_cache(ls.h, 0, 3)["pos"].cpu().numpy()[0]
    assert (np.diff(pos) > 0).all() and pos.max() < 300
    ls.close()
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=784, probe_tokens=64)    # bf16, tcgen05, V mover riding
    mp = 784 + 197 * 4
    _raw_steps_vs_lockstep(wl, 6, over=dict(summary_token=1, reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=mp),
                           oover=dict(summary_token=True, reindex_mode="lazy", max_position=mp, max_chunk_span=wl.chunk_tokens))


def test_summary_token_with_16_frame_chunk():
    """Alg. 1 with the paper's 16-frame chunk: 3137 tokens are pruned per deep layer and step, more than the summary
    kernel's evicted list could hold in the default 48 KB of shared memory (the opt-in is made at create time)."""
    wl = CONFIGS["llava_ov_7b_c16"].scaled(n_layers=4, budget=3136, probe_tokens=16)      # T = 6272, evicts 3136 (+1)
    ls, reps = _run(wl, 2, cfg_over=dict(summary_token=1), oracle_over=dict(summary_token=True))
    assert all(r.get("summary_layers") == 1 for r in reps)
    ls.close()


def test_probe_count_changes_between_updates_on_tcgen05():
    """n_probe is a per-call argument: crossing G * P = 512 changes the number of row super-chunks (and of groups) of the
    tcgen05 scoring kernel from one update to the next; its progress counters are reset every update."""
    wl = CONFIGS["qwen25_vl_7b"].scaled(n_layers=5, budget=1024, probe_tokens=128)
    ls = LockStep(wl)
    ls.fill()
    for n_probe in (64, 128, 16, 128, 73, 74):                                # 448 / 896 / 112 / 896 / 511 / 518 probe rows per KV head
        ls.step(check=True, n_probe=n_probe)
        assert hb.hermes_last_score_path(ls.h) == hb.HERMES_SCORE_TCGEN05
    for n_probe in (128, 64, 128):                                            # and with the compaction riding (no get_cache)
        ls.raw_step(n_probe=n_probe)
    ls.step(check=True, n_probe=128)
    assert hb.hermes_device_status(ls.h) == 0
    ls.close()


def test_probe_row_ranges_simt_and_tcgen05():
    """DESIGN f3 (App. B): deep layers score with the global-prompt rows [probe_deep_begin, P) only."""
    ls, _ = _run(CONFIGS["toy"], 3, cfg_over=dict(probe_deep_begin=3), oracle_over=dict(probe_deep_begin=3))
    assert hb.hermes_last_score_path(ls.h) == hb.HERMES_SCORE_SIMT
    ls.close()
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=784, probe_tokens=24)
    ls, _ = _run(wl, 2, n_warm=1, cfg_over=dict(probe_deep_begin=8), oracle_over=dict(probe_deep_begin=8))
    assert hb.hermes_last_score_path(ls.h) == hb.HERMES_SCORE_TCGEN05
    ls.close()


def test_deferred_v_compaction_equals_immediate():
    """defer_v: V rows moved by the next update's scoring kernel (tc_v_mover) or by a flush must give the same cache,
    bit for bit, as compacting V at once; the summary-token slot and a SIMT-path update in between are covered."""
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=784, probe_tokens=64)   # long enough scoring for the move to ride

    def run(defer, summary):
        ls = LockStep(wl, cfg_over=dict(defer_v=defer, summary_token=summary), oracle_over=dict(summary_token=bool(summary)))
        ls.fill()

        def raw_step(n_probe=None):          # no hermes_get_cache in between (it would flush the pending move)
            K, V, Q, _ = ls._gen(wl.chunk_tokens, True, n_probe)
            hb.hermes_append_chunk(ls.h, to_dev(K, wl.dtype), to_dev(V, wl.dtype), to_dev(Q, wl.dtype))

        for i in range(5):
            raw_step()                                           # deferred moves ride in the next scoring kernel
            assert hb.hermes_v_pending(ls.h) == defer
        raw_step(n_probe=2)                                      # G*P = 14 < 32: CUDA-core path -> flush before append
        assert hb.hermes_v_pending(ls.h) == 0
        raw_step()
        torch.cuda.synchronize()
        out = [{k: t.clone() for k, t in hb.hermes_get_cache(ls.h, 0, l).items() if torch.is_tensor(t)}
               for l in range(wl.n_layers)]                      # get_cache flushes the last pending move
        assert hb.hermes_v_pending(ls.h) == 0 and hb.hermes_device_status(ls.h) == 0
        ls.close()
        return out

    for summary in (0, 1):
        a, b = run(1, summary), run(0, summary)
        for l in range(wl.n_layers):
            for key in ("k", "v", "pos", "last_kept", "last_scores"):
                assert torch.equal(a[l][key], b[l][key]), (summary, l, key)
    # and the lock-step oracle comparison still holds when every checked update starts from a flushed cache
    ls, reps = _run(wl, 3, n_warm=2, cfg_over=dict(defer_v=1))
    ls.close()


def test_steady_state_updates_replay_from_a_cuda_graph():
    """An evicting update on the device entry point enqueues kernels only (no copy, no allocation, no host
    synchronisation; cooperative + programmatic-dependent launches included), so it can be stream-captured.  In steady
    state (eager re-indexing, len == budget, default pos_start) two consecutive updates form a period -- the double buffer
    flips twice, every kernel argument repeats -- and a graph of two updates replayed n times equals 2 n eager updates on
    the same input buffers, bit for bit (the V move rides inside the captured scoring launches as well)."""
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=6, budget=784, probe_tokens=64)
    gen = torch.Generator(device="cuda").manual_seed(11)
    L, C = wl.n_layers, wl.chunk_tokens
    K, V = (torch.randn(1, L, C, wl.n_kv_heads, wl.head_dim, generator=gen, device="cuda").to(torch.bfloat16) for _ in range(2))
    Q = torch.randn(1, L, wl.n_q_heads, wl.probe_tokens, wl.head_dim, generator=gen, device="cuda").to(torch.bfloat16)
    K2, V2, Q2 = K.clone(), V.clone(), Q.clone()              # the eager handle reads its own copies

    def warm(k, v, q):
        h = hb.hermes_create(hb.config_for_workload(wl))
        for _ in range(wl.budget // C):
            hb.hermes_append_chunk(h, k, v, None)
        for _ in range(2):
            hb.hermes_append_chunk(h, k, v, q)
        return h

    a, b = warm(K, V, Q), warm(K2, V2, Q2)
    torch.cuda.synchronize()
    graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.graph(graph, stream=side):                # the binding launches on torch's current stream: the capturing one
        hb.hermes_append_chunk(a, K, V, Q)
        hb.hermes_append_chunk(a, K, V, Q)
    for i in range(4):
        fresh = torch.randn(K.shape, generator=gen, device="cuda").to(torch.bfloat16)
        K.copy_(fresh); K2.copy_(fresh)                       # new data in the same buffers, as a serving loop would do
        graph.replay()
        hb.hermes_append_chunk(b, K2, V2, Q2)
        hb.hermes_append_chunk(b, K2, V2, Q2)
        torch.cuda.synchronize()
    assert hb.hermes_last_score_path(a) == hb.HERMES_SCORE_TCGEN05 and hb.hermes_len(a) == hb.hermes_len(b) == wl.budget
    for l in range(L):
        va, vb = hb.hermes_get_cache(a, 0, l), hb.hermes_get_cache(b, 0, l)
        torch.cuda.synchronize()
        for k in ("k", "v", "pos", "last_kept", "last_scores"):
            assert torch.equal(va[k], vb[k]), f"layer {l}: {k} differs between graph replay and eager updates"
    hb.hermes_destroy(a); hb.hermes_destroy(b)
