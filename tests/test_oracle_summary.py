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
    # the last step's summary equals Alg. 1 recomputed from that step's evicted set
    h = hist[-1]
    assert h["out"]["kept"][3, -1] == -1


def test_summary_token_off_is_the_default_path():
    wl = CONFIGS["toy"]
    _, st_a, _, ids_a, _ = run_oracle_schedule(wl, 3)
    _, st_b, _, ids_b, _ = run_oracle_schedule(wl, 3, cfg_over=dict(summary_token=False))
    assert st_a.K.tobytes() == st_b.K.tobytes() and np.array_equal(ids_a, ids_b)
