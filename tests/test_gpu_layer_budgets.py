"""GPU parity for layer-dependent budgets (Tab. 5; DESIGN f4): the CUDA path through the C ABI
against oracle_step_layer_budgets, lock-step, at the three non-uniform weightings of Tab. 5."""
import numpy as np
import pytest
import torch

import paper_2601_14724_b200 as hb
from gpu_harness import BAND_RTOL, K_RTOL, SCORE_RTOL, to_dev
from helpers import Feeder, bf16_ulp, oracle_config
from oracle import hermes_oracle as ho
from workloads import CONFIGS

pytestmark = pytest.mark.gpu
TAB5 = [(1.3, 1.0, 0.7), (0.7, 1.6, 0.7), (0.7, 1.0, 1.3)]


def _gpu_state(h, ocfg, wl):
    """Oracle stream holding the GPU's current cache (per-layer lengths)."""
    torch.cuda.synchronize()
    st = ho.OracleStream(ocfg)
    L = wl.n_layers
    st.lens = np.array([hb.hermes_layer_len(h, l) for l in range(L)], np.int64)
    st.len = int(st.lens.max())
    st._ensure(max(st.len, 1))
    for l in range(L):
        v = hb.hermes_get_cache(h, 0, l)
        n = int(st.lens[l])
        assert v["len"] == n
        st.K[l, :n] = v["k"].float().cpu().numpy(); st.V[l, :n] = v["v"].float().cpu().numpy()
        st.pos[l, :, :n] = v["pos"].cpu().numpy()
    return st


def _run(wl, w, n_updates, oover=None, **over):
    ocfg = oracle_config(wl, budget_weights=w, capacity=0, **(oover or {}))
    m = ho.layer_budgets(ocfg)
    # slots per layer: the largest layer plus a chunk, and at least the workload's own capacity (the toy preload)
    cfg = hb.config_for_workload(wl, budget_weight=w, max_tokens=int(max(wl.cap, m.max() + wl.chunk_tokens)), **over)
    h = hb.hermes_create(cfg)
    assert [hb.hermes_layer_budget(h, l) for l in range(wl.n_layers)] == m.tolist()
    fd = Feeder(wl, 0)
    half = wl.head_dim // 2
    n_cmp = n_untouched = 0
    paths = set()
    n_summ = 0
    sizes = [wl.preload_tokens] if wl.preload_tokens else []
    next_pos = -1                                           # lazy mode: the running position counter, mirrored from the oracle
    for u, n in enumerate(sizes + [wl.chunk_tokens] * n_updates):
        st = _gpu_state(h, ocfg, wl)
        st.next_pos = next_pos
        ap = ho.arrival_positions(ocfg, st, n, -1)
        K, V, Q, _ = fd.next(n, ap, with_probe=u >= len(sizes))
        hb.hermes_append_chunk(h, to_dev(K[None], wl.dtype), to_dev(V[None], wl.dtype), None if Q is None else to_dev(Q[None], wl.dtype))
        torch.cuda.synchronize()
        out = ho.oracle_step_layer_budgets(st, K, V, Q)
        next_pos = st.next_pos
        if out["evicted"]:
            paths.add(hb.hermes_last_score_path(h))
        assert hb.hermes_len(h) == int(st.lens.max())
        for l in range(wl.n_layers):
            v = hb.hermes_get_cache(h, 0, l)
            n_l = int(st.lens[l])
            assert v["len"] == n_l == hb.hermes_layer_len(h, l)
            k_gpu = v["k"].float().cpu().numpy(); v_gpu = v["v"].float().cpu().numpy(); p_gpu = v["pos"].cpu().numpy()
            if not out["evicted"] or not out["evicted_layers"][l]:          # appended to, otherwise untouched: bit-exact
                assert np.array_equal(k_gpu, st.K[l, :n_l]) and np.array_equal(v_gpu, st.V[l, :n_l])
                assert np.array_equal(p_gpu, st.pos[l, :, :n_l])
                n_untouched += bool(out["evicted"])
                continue
            assert v["last_T"] == out["T"][l]
            s_gpu = v["last_scores"].cpu().numpy().astype(np.float64)
            s_or = out["S_tilde"][l]
            rel = np.abs(s_gpu - s_or) / np.maximum(np.abs(s_or), 1e-30)
            assert (rel <= SCORE_RTOL).all(), f"layer {l}: score rel err {rel.max():.3e}"
            kept_gpu = v["last_kept"].cpu().numpy().astype(np.int64)
            kept_or = np.asarray(out["kept"][l])
            assert len(kept_gpu) == m[l]
            if kept_or[-1] < 0:
                # summary token (DESIGN f1 x f4) in the layer's last slot: computed values, so K AND V get the K tolerance
                assert kept_gpu[-1] == -1 and p_gpu[0, -1] == st.pos[l, 0, n_l - 1]
                for g_, o_ in ((k_gpu[-1], st.K[l, n_l - 1]), (v_gpu[-1], st.V[l, n_l - 1])):
                    tol = np.maximum(K_RTOL * np.abs(o_), 2 * bf16_ulp(o_) if wl.dtype == "bf16" else 0.0) + 1e-30
                    assert (np.abs(g_.astype(np.float64) - o_) <= tol).all(), f"layer {l}: summary token off"
                n_summ += 1
                kept_gpu, kept_or = kept_gpu[:-1], kept_or[:-1]
                k_gpu, v_gpu, p_gpu, n_l = k_gpu[:-1], v_gpu[:-1], p_gpu[:, :-1], n_l - 1
            assert (np.diff(kept_gpu) > 0).all() and kept_gpu[0] >= 0
            if not np.array_equal(kept_gpu, kept_or):
                tau = s_or[kept_or].min()
                diff = np.setxor1d(kept_gpu, kept_or)
                assert (np.abs(s_or[diff] - tau) <= BAND_RTOL * abs(tau)).all(), f"layer {l}: kept sets differ outside the band"
                continue
            assert np.array_equal(p_gpu, st.pos[l, :, :n_l])
            assert np.array_equal(v_gpu.view(np.uint32), st.V[l, :n_l].view(np.uint32))
            ko = st.K[l, :n_l]
            nrm = np.hypot(ko[..., :half].astype(np.float64), ko[..., half:].astype(np.float64))
            tol = K_RTOL * np.concatenate([nrm, nrm], -1)
            if wl.dtype == "bf16":
                tol = np.maximum(tol, 2 * bf16_ulp(ko))
            assert (np.abs(k_gpu.astype(np.float64) - ko) <= tol + 1e-30).all(), f"layer {l}: K beyond tolerance"
            n_cmp += 1
    assert hb.hermes_device_status(h) == 0 and hb.hermes_v_pending(h) == 0
    lens = [hb.hermes_layer_len(h, l) for l in range(wl.n_layers)]
    hb.hermes_destroy(h)
    _run.n_summ = n_summ
    return m, lens, n_cmp, n_untouched, paths


@pytest.mark.parametrize("w", TAB5)
def test_toy_config_at_tab5_weightings(w):
    wl = CONFIGS["toy"]                                       # fp32, 4 layers (1 / 2 / 1), preload 128, chunks of 32
    m, lens, n_cmp, n_untouched, paths = _run(wl, w, 8)
    assert lens == m.tolist() and n_cmp >= 20 and paths == {hb.HERMES_SCORE_SIMT}
    if m.max() > 160:
        assert n_untouched > 0                                # a big layer was still under its budget while others compressed


def test_bf16_geometry_at_tab5_weighting():
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=588, probe_tokens=8)     # 1 / 4 / 2 layers, bf16, d 128
    m, lens, n_cmp, _, paths = _run(wl, (0.7, 1.0, 1.3), 6, score_path=hb.HERMES_SCORE_SIMT)
    assert lens == np.minimum(m, 196 * 6).tolist() and n_cmp >= 14 and paths == {hb.HERMES_SCORE_SIMT}


@pytest.mark.parametrize("w", TAB5)
def test_bf16_geometry_on_tcgen05_at_tab5_weightings(w):
    """Per-layer candidate counts on the tensor-core scoring path (k_tc_score<true>): the tile grid is the largest scored
    layer's, every other layer's tail -- whole tiles and whole pass-1 segments of it at these weightings -- is masked."""
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=896, probe_tokens=24)    # 1 / 4 / 2 layers; T_l from ~820 to ~1450
    m, lens, n_cmp, _, paths = _run(wl, w, 10, score_path=hb.HERMES_SCORE_TCGEN05)
    assert lens == np.minimum(m, 196 * 10).tolist() and n_cmp >= 20 and paths == {hb.HERMES_SCORE_TCGEN05}


def test_equal_weights_are_the_uniform_path():
    wl = CONFIGS["toy"]
    m, lens, n_cmp, n_untouched, _ = _run(wl, (2.0, 2.0, 2.0), 3)
    assert lens == [wl.budget] * wl.n_layers and n_untouched == 0


def test_deferred_v_move_with_layer_budgets_full_size():
    """configs[1] geometry at a Tab. 5 weighting, the launch bench.py --budget-weight times: consecutive evicting updates with
    no hermes_get_cache in between, so the previous update's V compaction (per-layer row counts) rides in the scoring
    launch.  The final cache must equal, bit for bit, that of a handle that never defers (the configuration the lock-step
    tests above compare with the oracle)."""
    wl = CONFIGS["llava_ov_7b"]
    w = (1.3, 1.0, 0.7)
    gen = torch.Generator(device="cuda").manual_seed(4242)
    L, Hkv, Hq, d, C, P = wl.n_layers, wl.n_kv_heads, wl.n_q_heads, wl.head_dim, wl.chunk_tokens, wl.probe_tokens
    chunks = [tuple(torch.randn(1, L, C, Hkv, d, generator=gen, device="cuda").to(torch.bfloat16) for _ in range(2)) +
              (torch.randn(1, L, Hq, P, d, generator=gen, device="cuda").to(torch.bfloat16),) for _ in range(6)]
    caches = []
    for defer in (1, 0):
        cfg = hb.config_for_workload(wl, budget_weight=w, max_tokens=0, defer_v=defer)
        h = hb.hermes_create(cfg)
        m_max = max(hb.hermes_layer_budgets(cfg))
        n = 0
        while hb.hermes_len(h) < m_max:                       # fill without a probe: nothing is evicted
            K, V, _ = chunks[n % 6]
            take = min(C, m_max - hb.hermes_len(h))
            hb.hermes_append_chunk(h, K[:, :, :take].contiguous(), V[:, :, :take].contiguous(), None)
            n += 1
        pend = []
        for i in range(5):
            K, V, Q = chunks[i % 6]
            hb.hermes_append_chunk(h, K, V, Q)
            pend.append(hb.hermes_v_pending(h))
        assert hb.hermes_last_score_path(h) == hb.HERMES_SCORE_TCGEN05
        assert pend == [defer] * 5, pend                      # the move rides (and is pending again) at every update
        torch.cuda.synchronize()
        out = []
        for l in range(L):
            v = hb.hermes_get_cache(h, 0, l)
            assert v["len"] == hb.hermes_layer_budget(h, l)
            out.append({k: v[k].clone() for k in ("k", "v", "pos", "last_kept", "last_scores")})
        torch.cuda.synchronize()
        assert hb.hermes_device_status(h) == 0
        hb.hermes_destroy(h)
        caches.append(out)
    for l in range(L):
        for k in caches[0][l]:
            assert torch.equal(caches[0][l][k], caches[1][l][k]), f"layer {l}: {k} differs between deferred and immediate V compaction"


@pytest.mark.parametrize("lazy", [False, True])
@pytest.mark.parametrize("w", TAB5)
def test_summary_token_with_layer_budgets_toy(w, lazy):
    """DESIGN f1 x f4: a deep layer that compresses keeps m_l - 1 tokens and one summary token of what it evicted; eager and
    lazy re-indexing (lazy: the running position advances by one more at such a step)."""
    wl = CONFIGS["toy"]
    over, oover = dict(summary_token=1), dict(summary_token=True)
    if lazy:
        over.update(reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=420)       # re-index steps inside the run
        oover.update(reindex_mode="lazy", max_position=420, max_chunk_span=wl.chunk_tokens)
    m, lens, n_cmp, _, paths = _run(wl, w, 8, oover=oover, **over)
    assert lens == m.tolist() and n_cmp >= 18 and _run.n_summ >= 5


def test_summary_token_with_layer_budgets_on_tcgen05():
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=896, probe_tokens=24)    # 1 / 4 / 2 layers: two deep layers
    m, lens, n_cmp, _, paths = _run(wl, (1.3, 1.0, 0.7), 9, oover=dict(summary_token=True), summary_token=1,
                                    score_path=hb.HERMES_SCORE_TCGEN05)
    assert lens == np.minimum(m, 196 * 9).tolist() and paths == {hb.HERMES_SCORE_TCGEN05} and _run.n_summ >= 8


@pytest.mark.parametrize("seed", range(6))
def test_random_geometry_with_layer_budgets(seed):
    """Seeded random geometries and weightings (ragged sizes, 1-4 KV heads, probe counts across the 512-row super-chunk
    boundary) through the same lock-step comparison; even seeds force the tcgen05 path and its per-layer tile schedule."""
    r = np.random.default_rng(500 + seed)
    tc = seed % 2 == 0
    hkv, grp = int(r.choice([1, 2, 3, 4])), int(r.choice([2, 4, 7]))
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=int(r.integers(4, 9)), n_kv_heads=hkv, n_q_heads=hkv * grp,
                                       budget=int(r.integers(600, 1100)), chunk_tokens=int(r.integers(40, 230)),
                                       probe_tokens=int(r.integers(max(1, -(-32 // grp)), 100)), seed=8100 + seed)
    w = tuple(float(x) for x in np.round(r.uniform(0.6, 1.7, 3), 2))
    summ = bool(r.integers(0, 2))
    over = dict(score_path=hb.HERMES_SCORE_TCGEN05 if tc else hb.HERMES_SCORE_SIMT)
    oover = {}
    if summ:
        over.update(summary_token=1); oover.update(summary_token=True)
    n_up = int(np.ceil(max(ho.layer_budgets(oracle_config(wl, budget_weights=w, capacity=0)).max() / wl.chunk_tokens, 1))) + 4
    m, lens, n_cmp, _, paths = _run(wl, w, n_up, oover=oover, **over)
    assert lens == m.tolist() and n_cmp >= wl.n_layers, (wl, w, summ)
    assert paths == {hb.HERMES_SCORE_TCGEN05 if tc else hb.HERMES_SCORE_SIMT}


def test_two_streams_with_layer_budgets_equal_two_single_stream_handles():
    """The per-layer schedule tables of k_tc_score<true> are per (stream, scored layer): a 2-stream handle must leave, for
    each stream, exactly the cache a single-stream handle leaves for the same inputs (bit for bit), V move riding or not."""
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=7, budget=896, probe_tokens=40)
    w = (0.7, 1.6, 0.7)
    gen = torch.Generator(device="cuda").manual_seed(77)
    L, Hkv, Hq, d, C, P = wl.n_layers, wl.n_kv_heads, wl.n_q_heads, wl.head_dim, wl.chunk_tokens, wl.probe_tokens
    steps = [(torch.randn(2, L, C, Hkv, d, generator=gen, device="cuda").to(torch.bfloat16),
              torch.randn(2, L, C, Hkv, d, generator=gen, device="cuda").to(torch.bfloat16),
              torch.randn(2, L, Hq, P, d, generator=gen, device="cuda").to(torch.bfloat16)) for _ in range(12)]

    def run(n_streams, pick):
        cfg = hb.config_for_workload(wl.scaled(n_streams=n_streams), budget_weight=w, max_tokens=0,
                                     score_path=hb.HERMES_SCORE_TCGEN05)
        h = hb.hermes_create(cfg)
        for i, (K, V, Q) in enumerate(steps):
            K, V, Q = (x[pick].contiguous() for x in (K, V, Q))
            hb.hermes_append_chunk(h, K, V, Q if i >= 3 else None)
        torch.cuda.synchronize()
        out = []
        for b in range(n_streams):
            for l in range(L):
                v = hb.hermes_get_cache(h, b, l)
                out.append({k: v[k].clone() for k in ("k", "v", "pos", "last_kept", "last_scores")})
        torch.cuda.synchronize()
        assert hb.hermes_device_status(h) == 0 and hb.hermes_last_score_path(h) == hb.HERMES_SCORE_TCGEN05
        hb.hermes_destroy(h)
        return out

    both = run(2, slice(0, 2))
    singles = run(1, slice(0, 1)) + run(1, slice(1, 2))
    for i, (a, b) in enumerate(zip(both, singles)):
        for k in a:
            assert torch.equal(a[k], b[k]), f"stream {i // L} layer {i % L}: {k} differs"
