"""Pins for the summary token (Alg. 1 at :640-672; DESIGN f1) in the oracle."""
import numpy as np

from helpers import run_oracle_schedule
from oracle import hermes_oracle as ho
from workloads import CONFIGS, rope_at_arrival


def _cfg(d=8, dtype="f32", theta=100.0):
    return ho.OracleConfig(n_layers=2, n_q_heads=2, n_kv_heads=2, head_dim=d, budget=4, forget_rate=0.1,
                           dtype=dtype, rope_theta=theta)


class _WL:                      # the fields rope_at_arrival reads
    rope_mode, head_dim, rope_theta = "1d", 8, 100.0


def test_single_pruned_token_is_that_token_moved_to_t():
    cfg = _cfg()
    g = np.random.default_rng(1)
    k = g.standard_normal((1, 2, 8)).astype(np.float32)
    v = g.standard_normal((1, 2, 8)).astype(np.float32)
    k_sum, v_sum = ho.summary_token(cfg, k, v, np.array([[17]]), 5)
    moved = ho.rotary_delta(cfg, k, np.array([[5 - 17]]))
    assert np.array_equal(k_sum, moved[0]) and np.array_equal(v_sum, v[0])


def test_phase_alignment_same_content_at_different_positions():
    """Pruned keys that are ONE un-rotated key k0 seen at different positions align to RoPE(k0, t): the mean of
    the aligned keys is RoPE(k0, t), while the plain mean of the un-aligned keys is not."""
    cfg = _cfg()
    g = np.random.default_rng(2)
    k0 = g.standard_normal((1, 1, 2, 8)).astype(np.float32)
    pos = np.array([[3, 11, 40, 41, 97]])
    K_p = rope_at_arrival(np.repeat(k0, 5, axis=1), pos, _WL)[0]            # [5, 2, 8]
    V_p = g.standard_normal((5, 2, 8)).astype(np.float32)
    k_sum, v_sum = ho.summary_token(cfg, K_p, V_p, pos, 7)
    ref = rope_at_arrival(k0, np.array([[7]]), _WL)[0, 0]
    np.testing.assert_allclose(k_sum, ref, atol=2e-6)
    assert np.abs(K_p.mean(axis=0) - ref).max() > 0.05
    np.testing.assert_allclose(v_sum, V_p.astype(np.float64).mean(axis=0), atol=1e-7)   # Step 1: simple mean


def test_mean_closed_form_and_linearity():
    cfg = _cfg()
    pos = np.array([[9, 9]])                                                # same position as t: delta 0
    a = np.full((1, 2, 8), 2.0, np.float32); b = np.full((1, 2, 8), 4.0, np.float32)
    k_sum, v_sum = ho.summary_token(cfg, np.concatenate([a, b]), np.concatenate([b, b]), pos, 9)
    assert (k_sum == 3.0).all() and (v_sum == 4.0).all()


def test_stream_with_summary_tokens_keeps_the_budget_and_contiguous_positions():
    wl = CONFIGS["toy"]                                                     # 4 layers: 1 shallow, 2 middle, 1 deep
    cfg, st, fd, ids, hist = run_oracle_schedule(wl, 6, cfg_over=dict(summary_token=True))
    for h in hist:
        out = h["out"]
        assert (out["kept"][:3] >= 0).all()                                 # only the deep layer aggregates
        assert out["kept"][3, -1] == -1 and (np.diff(out["kept"][3, :-1]) > 0).all()
        np.testing.assert_array_equal(out["pos_new"][:, 0], np.broadcast_to(np.arange(96), (4, 96)))
    assert st.len == wl.budget
    # retained real tokens still obey the rotation-composition pin; exactly one summary slot per deep layer
    assert (ids[3] == -1).sum() >= 1 and (ids[:3] >= 0).all()
    for l in range(wl.n_layers):
        real = np.nonzero(ids[l] >= 0)[0]
        k0 = np.stack([fd.k0_by_id[int(t)][l] for t in ids[l][real]])[None]
        ref = rope_at_arrival(k0, real[None, :], wl)[0]
        np.testing.assert_allclose(st.K[l, real], ref, atol=3e-5)


def test_summary_equals_alg1_on_the_evicted_set_and_folds_an_evicted_summary_token():
    """Every step's summary token is Alg. 1 recomputed, outside oracle_step, from that step's evicted candidates at
    their positions; and a summary token that is itself evicted later is an ordinary member of the next pruned set
    (DESIGN f1 (iv)) -- the schedule below contains such a step."""
    wl = CONFIGS["toy"]
    M = wl.budget
    folded = 0
    for u in range(1, 7):
        cfg, st_prev, _, ids_prev, _ = run_oracle_schedule(wl, u - 1, cfg_over=dict(summary_token=True))
        _, st, _, _, hist = run_oracle_schedule(wl, u, cfg_over=dict(summary_token=True))
        h = hist[-1]
        n_prev = st_prev.len
        K_cand = np.concatenate([st_prev.K[3, :n_prev], h["K_new"][3]], axis=0)
        V_cand = np.concatenate([st_prev.V[3, :n_prev], h["V_new"][3]], axis=0)
        n_new = h["K_new"].shape[1]
        P_cand = np.concatenate([st_prev.pos[3][:, :n_prev], (cfg.pos_offset + n_prev + np.arange(n_new))[None, :]], axis=1)
        T = K_cand.shape[0]
        ev = np.setdiff1d(np.arange(T), h["out"]["kept"][3, :-1])
        assert len(ev) == T - (M - 1)
        k_sum, v_sum = ho.summary_token(cfg, K_cand[ev], V_cand[ev], P_cand[:, ev], cfg.pos_offset + M - 1)
        assert np.array_equal(st.K[3, M - 1], k_sum) and np.array_equal(st.V[3, M - 1], v_sum)
        if u > 1 and (M - 1) in ev:                      # slot M-1 of the previous cache is the previous summary token
            assert ids_prev[3, M - 1] == -1
            folded += 1
    assert folded >= 1


def test_summary_token_off_is_the_default_path():
    wl = CONFIGS["toy"]
    _, st_a, _, ids_a, _ = run_oracle_schedule(wl, 3)
    _, st_b, _, ids_b, _ = run_oracle_schedule(wl, 3, cfg_over=dict(summary_token=False))
    assert st_a.K.tobytes() == st_b.K.tobytes() and np.array_equal(ids_a, ids_b)


# ---- summary tokens under lazy re-indexing: the paper's streaming default (PAPER.md:314 with :318) -------------
LAZY_SUM = dict(summary_token=True, reindex_mode="lazy", max_position=300, max_chunk_span=32)


def test_lazy_summary_token_sits_after_the_newest_token():
    """Between re-index steps the kept tokens keep their original indices and the summary token,
    concatenated after them (Alg. 1 step 3), takes the position after the newest token; the next chunk starts one
    position later, and the re-index trigger counts that position."""
    wl = CONFIGS["toy"]
    cfg, st, fd, ids, hist = run_oracle_schedule(wl, 8, cfg_over=LAZY_SUM)
    # without summary tokens p_end = 160 + 32 u and update 4 re-indexes (tests/test_oracle_lazy.py); every summary
    # token costs one position: p_end = 160 + 33 u, and 160 + 33*4 + 1 + 32 = 325 > 300, but already
    # 160 + 33*3 + 1 + 32 = 292 <= 300 and update 4 is the first over the limit
    assert [h["out"]["reindexed"] for h in hist] == [False] * 4 + [True] + [False] * 3
    p_end = 160
    for u, h in enumerate(hist):
        out = h["out"]
        pos3 = out["pos_new"][3, 0]
        assert out["kept"][3, -1] == -1 and (np.diff(pos3) > 0).all()        # strictly increasing, summary last
        if not out["reindexed"]:
            assert pos3[-1] == p_end                                         # the position after the newest token
            assert out["pos_new"][:3, 0].max() == p_end - 1                  # other layers: the newest token itself
            p_end += 33
        else:
            np.testing.assert_array_equal(out["pos_new"][:, 0], np.broadcast_to(np.arange(96), (4, 96)))
            p_end = 96 + 32                                                  # after re-indexing everything is below offset + |M|
    assert st.next_pos == p_end - 32


def test_lazy_summary_keys_obey_rotation_composition_and_alg1():
    wl = CONFIGS["toy"]
    cfg, st, fd, ids, hist = run_oracle_schedule(wl, 6, cfg_over=LAZY_SUM)
    for l in range(wl.n_layers):                                             # real tokens: RoPE(k0[id], current position)
        real = np.nonzero(ids[l] >= 0)[0]
        k0 = np.stack([fd.k0_by_id[int(t)][l] for t in ids[l][real]])[None]
        ref = rope_at_arrival(k0, st.pos[l][:, real], wl)[0]
        np.testing.assert_allclose(st.K[l, real], ref, atol=3e-5)
    # the summary token of a lazy (copy) step is Alg. 1 on exactly the evicted candidates, aligned to p_end
    _, st_prev, _, _, hist_prev = run_oracle_schedule(wl, 3, cfg_over=LAZY_SUM)
    h = hist[3]
    assert not h["out"]["reindexed"]
    K_cand = np.concatenate([st_prev.K[3, :wl.budget], h["K_new"][3]], axis=0)
    V_cand = np.concatenate([st_prev.V[3, :wl.budget], h["V_new"][3]], axis=0)
    T = K_cand.shape[0]
    P_cand = np.concatenate([st_prev.pos[3][:, :wl.budget], h["out"]["pos_new"][:3, :, -1:].max() - 31 + np.arange(32)[None, :]], axis=1)
    ev = np.setdiff1d(np.arange(T), h["out"]["kept"][3, :-1])
    t = int(h["out"]["pos_new"][3, 0, -1])
    k_sum, v_sum = ho.summary_token(cfg, K_cand[ev], V_cand[ev], P_cand[:, ev], t)
    _, st4, _, _, _ = run_oracle_schedule(wl, 4, cfg_over=LAZY_SUM)
    assert np.array_equal(st4.K[3, wl.budget - 1], k_sum) and np.array_equal(st4.V[3, wl.budget - 1], v_sum)


def test_lazy_summary_with_tiny_limit_equals_eager_summary():
    wl = CONFIGS["toy"]
    _, st_e, _, ids_e, _ = run_oracle_schedule(wl, 5, cfg_over=dict(summary_token=True))
    _, st_l, _, ids_l, hist = run_oracle_schedule(wl, 5, cfg_over=dict(summary_token=True, reindex_mode="lazy", max_position=1, max_chunk_span=32))
    assert all(h["out"]["reindexed"] for h in hist) and np.array_equal(ids_e, ids_l)
    assert st_e.K.tobytes() == st_l.K.tobytes() and st_e.V.tobytes() == st_l.V.tobytes() and np.array_equal(st_e.pos, st_l.pos)
