"""Pins for lazy re-indexing (DESIGN f2) in the oracle, on BASELINE.json configs[0].

Lazy mode keeps the original position indices of the retained tokens (keys are copied, not re-rotated) and
re-indexes, exactly as the eager path does, only at the compression step after which the next chunk would no
longer fit below `max_position`."""
import numpy as np

from helpers import run_oracle_schedule
from oracle import hermes_oracle as ho
from workloads import CONFIGS, rope_at_arrival

LAZY = dict(reindex_mode="lazy", max_position=300, max_chunk_span=32)


def test_trigger_rule_closed_form():
    cfg = ho.OracleConfig(n_layers=2, n_q_heads=2, n_kv_heads=1, head_dim=4, budget=8, forget_rate=0.1,
                          reindex_mode="lazy", max_position=100, max_chunk_span=10)
    assert not ho.lazy_reindex_due(cfg, 90)          # 90 + 10 == 100: the next chunk still fits [90, 100)
    assert ho.lazy_reindex_due(cfg, 91)


def test_lazy_keeps_original_indices_until_the_limit():
    wl = CONFIGS["toy"]
    cfg, st, fd, ids, hist = run_oracle_schedule(wl, 10, cfg_over=LAZY)
    # arrival p_end = 160 + 32 u until the first trigger; 288 + 32 > 300 -> update 4 re-indexes, then 96 + 32 (u - 4)
    assert [h["out"]["reindexed"] for h in hist] == [False] * 4 + [True] + [False] * 5
    for u, h in enumerate(hist):
        out = h["out"]
        if not out["reindexed"]:
            # positions are the ORIGINAL ones of the kept tokens: strictly increasing, not contiguous in general
            assert (np.diff(out["pos_new"][:, 0], axis=1) > 0).all()
            assert out["pos_new"].max() == (160 + 32 * u - 1 if u < 4 else 96 + 32 * (u - 4) - 1)
        else:
            np.testing.assert_array_equal(out["pos_new"][:, 0], np.broadcast_to(np.arange(96), (4, 96)))
    # every key still equals RoPE(k0[id], its position), whatever mix of copies and re-rotations it went through
    for l in range(wl.n_layers):
        k0 = np.stack([fd.k0_by_id[int(t)][l] for t in ids[l]])[None]
        ref = rope_at_arrival(k0, st.pos[l][:, :wl.budget], wl)[0]
        np.testing.assert_allclose(st.K[l, :wl.budget], ref, atol=3e-5)


def test_lazy_copy_is_bit_exact_without_trigger():
    wl = CONFIGS["toy"]
    over = dict(reindex_mode="lazy", max_position=10 ** 6, max_chunk_span=32)
    _, st, _, _, hist = run_oracle_schedule(wl, 3, cfg_over=over)
    assert not any(x["out"]["reindexed"] for x in hist)
    # the schedule is deterministic: the state after 2 updates is the state before the third
    _, st2, _, _, _ = run_oracle_schedule(wl, 2, cfg_over=over)
    h = hist[-1]
    K_cand = np.concatenate([st2.K[:, :wl.budget], h["K_new"]], axis=1)
    for l in range(wl.n_layers):                     # K' rows are the candidate rows bit for bit: no rotation at all
        assert st.K[l, :wl.budget].tobytes() == np.ascontiguousarray(K_cand[l, h["out"]["kept"][l]]).tobytes()


def test_lazy_with_tiny_limit_equals_eager():
    wl = CONFIGS["toy"]
    _, st_e, _, ids_e, _ = run_oracle_schedule(wl, 6)
    _, st_l, _, ids_l, hist = run_oracle_schedule(wl, 6, cfg_over=dict(reindex_mode="lazy", max_position=1, max_chunk_span=32))
    assert all(h["out"]["reindexed"] for h in hist)
    assert np.array_equal(ids_e, ids_l)
    assert st_e.K.tobytes() == st_l.K.tobytes() and st_e.V.tobytes() == st_l.V.tobytes()
    assert np.array_equal(st_e.pos, st_l.pos)
