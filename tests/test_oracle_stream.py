"""End-to-end pins of `oracle_step` over multi-update schedules (config 1 = BASELINE.json configs[0])."""
import numpy as np
import pytest

from helpers import Feeder, fill_chunks, oracle_config, run_oracle_schedule
from oracle import hermes_oracle as ho
from workloads import CONFIGS, rope_at_arrival


def test_toy_schedule_invariants():
    wl = CONFIGS["toy"]
    cfg, st, fd, ids, hist = run_oracle_schedule(wl, 10)
    assert [h["out"]["T"] for h in hist] == [160] + [128] * 9          # DESIGN c16
    for h in hist:
        out = h["out"]
        assert out["kept"].shape == (wl.n_layers, wl.budget)              # retained count == |M| exactly
        assert (np.diff(out["kept"], axis=1) > 0).all()                   # ascending = temporal order
        np.testing.assert_array_equal(out["pos_new"][:, 0], np.broadcast_to(np.arange(96), (4, 96)))
        np.testing.assert_allclose(out["W"][1:].sum(axis=1), 1.0, rtol=1e-12)
        assert (out["W"][0] == 0).all()                                   # shallow layer is not scored
    assert st.len == wl.budget
    assert (np.diff(ids, axis=1) > 0).all()                               # order-preserving
    # V rows are the source rows, bit for bit, across 10 updates (identity via token id)
    # and every retained key equals RoPE(k0[id], offset + slot): rotation composition end to end
    slot_pos = np.arange(wl.budget)[None, :]
    for l in range(wl.n_layers):
        k0 = np.stack([fd.k0_by_id[int(t)][l] for t in ids[l]])[None]     # [1, n, H, d]
        ref = rope_at_arrival(k0, slot_pos, wl)[0]
        np.testing.assert_allclose(st.K[l, :wl.budget], ref, atol=2e-5)
    # anchors (slot 0 of each frame, key x3) survive preferentially in the deep layer
    deep_anchor = (ids[-1] % wl.tokens_per_frame == 0).mean()
    assert deep_anchor > 1.5 / wl.tokens_per_frame


def test_gather_is_bit_exact_single_step():
    wl = CONFIGS["toy"]
    _, st, _, _, hist = run_oracle_schedule(wl, 2)
    h = hist[-1]
    V_all = np.concatenate([h["V_pre"], h["V_new"]], axis=1)
    for l in range(wl.n_layers):
        assert st.V[l, :wl.budget].tobytes() == np.ascontiguousarray(V_all[l, h["out"]["kept"][l]]).tobytes()


def test_fifo_degenerate_is_sliding_window():
    wl = CONFIGS["toy"]
    over = dict(n_shallow=4, n_deep=0, lambda_shallow=0.0)               # every layer pure recency, no smoothing
    _, st, fd, ids, _ = run_oracle_schedule(wl, 5, cfg_over=over)
    newest = np.arange(fd.tokens_fed - wl.budget, fd.tokens_fed)
    assert (ids == newest[None, :]).all()                                 # FIFO baseline of PAPER.md:49


def test_no_eviction_below_budget_and_without_probe():
    wl = CONFIGS["toy"]
    cfg = oracle_config(wl)
    st = ho.OracleStream(cfg)
    fd = Feeder(wl)
    K, V, Q, _ = fd.next(64, ho.arrival_positions(cfg, st, 64, -1), True)
    out = ho.oracle_step(st, K, V, Q)                                     # T = 64 <= 96
    assert not out["evicted"] and st.len == 64
    K, V, _, _ = fd.next(64, ho.arrival_positions(cfg, st, 64, -1), False)
    out = ho.oracle_step(st, K, V, None)                                  # over budget but no probe
    assert not out["evicted"] and st.len == 128
    assert st.pos[0, 0, :128].tolist() == list(range(128))


def test_determinism_and_stream_independence():
    wl = CONFIGS["toy"]
    a = run_oracle_schedule(wl, 3, stream=0)[1]
    b = run_oracle_schedule(wl, 3, stream=0)[1]
    c = run_oracle_schedule(wl, 3, stream=1)[1]
    assert a.K.tobytes() == b.K.tobytes() and a.V.tobytes() == b.V.tobytes()
    assert a.K.tobytes() != c.K.tobytes()


def test_mrope_stream_small():
    wl = CONFIGS["qwen25_vl_7b"].scaled(n_layers=4, n_q_heads=4, n_kv_heads=2, budget=512,
                                        chunk_tokens=128, probe_tokens=8, pos_offset=3)
    cfg, st, fd, ids, hist = run_oracle_schedule(wl, 4)
    assert len(fill_chunks(wl)) == 4
    for h in hist:
        pn = h["out"]["pos_new"]                                          # [L, 3, |M|]
        for l in range(wl.n_layers):
            t = pn[l, 0]
            assert (np.diff(t) >= 0).all() and t[0] == wl.pos_offset
            assert set(np.unique(t)) == set(range(wl.pos_offset, wl.pos_offset + len(np.unique(t))))
    # h/w ids are preserved: they still equal the grid coordinates of each token's slot in its t-step
    tok_in_step = ids % 64
    np.testing.assert_array_equal(st.pos[:, 1, :wl.budget], wl.pos_offset + tok_in_step // 8)
    np.testing.assert_array_equal(st.pos[:, 2, :wl.budget], wl.pos_offset + tok_in_step % 8)
    # arrival t of the next chunk is above every compacted t in every layer
    nxt = ho.arrival_positions(cfg, st, 128, -1)
    assert nxt[0].min() > st.pos[:, 0, :wl.budget].max()


def test_llava_geometry_small_step_has_structure():
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=10, budget=784, probe_tokens=16)
    _, st, _, ids, hist = run_oracle_schedule(wl, 2)
    out = hist[-1]["out"]
    assert out["kept"].shape == (10, 784)
    ev0 = np.setdiff1d(np.arange(out["T"]), out["kept"][0])
    assert ev0.max() < 400                                                # shallow layer evicts old tokens
    anchor_frac_deep = (ids[-1] % 196 == 98).mean()
    assert anchor_frac_deep >= 1.0 / 196                                  # anchors are never the evicted ones
    is_anchor = (np.arange(out["T"]) % 196 == 98)
    assert out["S_tilde"][-1][is_anchor].mean() > 3 * out["S_tilde"][-1][~is_anchor].mean()
