"""Pins for layer-dependent budgets (Tab. 5; DESIGN f4) in the oracle."""
import numpy as np
import pytest

from helpers import Feeder, oracle_config, run_oracle_schedule, take_ids
from oracle import hermes_oracle as ho
from workloads import CONFIGS, rope_at_arrival

TAB5 = [(1.0, 1.0, 1.0), (1.3, 1.0, 0.7), (0.7, 1.6, 0.7), (0.7, 1.0, 1.3)]


def _cfg(L, budget, w, **kw):
    return ho.OracleConfig(n_layers=L, n_q_heads=2, n_kv_heads=1, head_dim=4, budget=budget, forget_rate=0.1,
                           budget_weights=w, **kw)


@pytest.mark.parametrize("w", TAB5)
@pytest.mark.parametrize("L,budget", [(4, 96), (28, 6000), (28, 6272), (80, 4096), (7, 785)])
def test_budgets_sum_to_the_fixed_total(L, budget, w):
    m = ho.layer_budgets(_cfg(L, budget, w))
    assert m.sum() == budget * L and (m > 0).all()                # "the total token budget remains fixed"
    ns, nm, nd = ho.stage_split(L)
    # one weight per stage: equal budgets inside a stage (the residue sits on the last layer only)
    assert len(set(m[:ns])) == 1 and len(set(m[ns:ns + nm])) == 1 and len(set(m[ns + nm:L - 1])) <= 1
    if w == (1.0, 1.0, 1.0):
        assert (m == budget).all()
    # floor of the proportional share, residue 0 <= r < L on the last layer
    share = np.array([w[0]] * ns + [w[1]] * nm + [w[2]] * nd) / (w[0] * ns + w[1] * nm + w[2] * nd) * budget * L
    assert (np.abs(m[:-1] - np.floor(share[:-1])) <= 1).all()     # <= 1: fp32 weights vs the decimal ones typed here
    assert 0 <= m[-1] - np.floor(share[-1]) <= L


def test_hand_example():
    # L = 4 -> 1 shallow / 2 middle / 1 deep; weights 1.3 / 1.0 / 0.7 sum to 4.0; |M| = 4 * 96 = 384:
    # 384 * 1.3 / 4 = 124.8 -> 124, 96, 96, 384 * 0.7 / 4 = 67.2 -> 67; residue 384 - 383 = 1 -> last layer 68
    assert ho.layer_budgets(_cfg(4, 96, (1.3, 1.0, 0.7))).tolist() == [124, 96, 96, 68]


def test_aligned_smoothing_reduces_to_eq5_and_pairs_equal_distances():
    cfg = _cfg(3, 8, (1, 1, 1), n_shallow=1, n_deep=1)
    g = np.random.default_rng(0)
    S = g.random((3, 6))
    same = ho.smooth_scores_aligned(cfg, [S[0], S[1], S[2]])
    np.testing.assert_array_equal(np.stack(same), ho.smooth_scores(cfg, S))
    # T = 4 over T = 2: the two newest candidates of layer 0 meet layer 1's two; the two oldest keep their raw score
    S0, S1 = np.array([0.1, 0.2, 0.3, 0.4]), np.array([1.0, 2.0])
    out = ho.smooth_scores_aligned(cfg, [S0, S1, np.array([5.0])])
    lam = cfg.lambda_shallow
    np.testing.assert_allclose(out[0], [0.1, 0.2, (1 - lam) * 0.3 + lam * 1.0, (1 - lam) * 0.4 + lam * 2.0])
    # T = 2 over T = 1 (layer 1 over layer 2), and a SHORTER layer over a longer one: newest-to-newest both ways
    np.testing.assert_allclose(out[1], [1.0, (1 - cfg.lambda_middle) * 2.0 + cfg.lambda_middle * 5.0])
    out = ho.smooth_scores_aligned(cfg, [S1, S0, S0])
    np.testing.assert_allclose(out[0], [(1 - lam) * 1.0 + lam * 0.3, (1 - lam) * 2.0 + lam * 0.4])


def _run_lb(wl, n_updates, w, **over):
    cfg = oracle_config(wl, budget_weights=w, **dict(dict(capacity=0), **over))
    st = ho.OracleStream(cfg)
    fd = Feeder(wl, 0)
    L = wl.n_layers
    ids = [np.zeros(0, np.int64) for _ in range(L)]
    hist = []
    sizes = [wl.preload_tokens] if wl.preload_tokens else []
    for u, n in enumerate(sizes + [wl.chunk_tokens] * n_updates):
        if st.lens is None:
            st.lens = np.zeros(L, np.int64)
        ap = ho.arrival_positions(cfg, st, n, -1)
        K, V, Q, new_ids = fd.next(n, ap, with_probe=u >= len(sizes))
        pre = {"lens": st.lens.copy(), "K": st.K.copy() if st.K is not None else None,
               "V": st.V.copy() if st.V is not None else None, "pos": st.pos.copy() if st.pos is not None else None}
        out = ho.oracle_step_layer_budgets(st, K, V, Q)
        for l in range(L):
            ids[l] = np.concatenate([ids[l], new_ids])
            if out["evicted"]:
                ids[l] = take_ids(ids[l][None, :], np.asarray(out["kept"][l])[None, :])[0]   # -1: a summary token
        hist.append(dict(out=out, pre=pre, K_new=K, V_new=V, p_arr=ap))
    return cfg, st, fd, ids, hist


def test_equal_weights_reproduce_the_uniform_path_bit_for_bit():
    wl = CONFIGS["toy"]
    _, st_u, _, ids_u, hist_u = run_oracle_schedule(wl, 6)
    cfg, st, fd, ids, hist = _run_lb(wl, 6, (1.0, 1.0, 1.0), capacity=wl.cap)
    assert (st.lens == wl.budget).all()
    M = wl.budget
    assert st.K[:, :M].tobytes() == st_u.K[:, :M].tobytes() and st.V[:, :M].tobytes() == st_u.V[:, :M].tobytes()
    assert np.array_equal(st.pos[:, :, :M], st_u.pos[:, :, :M]) and np.array_equal(np.stack(ids), ids_u)
    for a, b in zip(hist[1:], hist_u):
        assert np.array_equal(np.stack(a["out"]["kept"]), b["out"]["kept"])
        np.testing.assert_array_equal(np.stack(a["out"]["S_tilde"]), b["out"]["S_tilde"])


@pytest.mark.parametrize("w", TAB5[1:])
def test_stream_invariants_with_tab5_weights(w):
    wl = CONFIGS["toy"]                                         # preload 128, then 32-token chunks; budgets around 96
    cfg, st, fd, ids, hist = _run_lb(wl, 8, w)
    m = ho.layer_budgets(cfg)
    assert (st.lens == np.minimum(m, 128 + 8 * 32)).all() and (st.lens == m).all()
    untouched = 0
    for h in hist[1:]:
        out, pre = h["out"], h["pre"]
        T = pre["lens"] + wl.chunk_tokens
        assert out["evicted"] == bool((T > m).any())
        for l in range(wl.n_layers):
            if out["evicted"] and not out["evicted_layers"][l]:  # under its budget: appended to, nothing else
                untouched += 1
                assert np.array_equal(out["kept"][l], np.arange(T[l]))
                assert st.K is not None and np.array_equal(out["pos_new"][l][0, :pre["lens"][l]], pre["pos"][l, 0, :pre["lens"][l]])
            elif out["evicted"]:
                assert len(out["kept"][l]) == m[l] and (np.diff(out["kept"][l]) > 0).all()
                np.testing.assert_array_equal(out["pos_new"][l][0], cfg.pos_offset + np.arange(m[l]))   # Eq. 8 per layer
    # every retained key is RoPE(k0[id], its position) and every V row is its source row, layer by layer
    for l in range(wl.n_layers):
        n = int(st.lens[l])
        k0 = np.stack([fd.k0_by_id[int(t)][l] for t in ids[l]])[None]
        ref = rope_at_arrival(k0, st.pos[l][:, :n], wl)[0]
        np.testing.assert_allclose(st.K[l, :n], ref, atol=3e-5)
        assert len(ids[l]) == n and (np.diff(ids[l]) > 0).all()
    # the weightings differ in which layers are over budget first: with a 128-token preload and budgets of 68..154
    # at least one (layer, step) pair must have been left untouched for the non-uniform weightings with m_l > 160
    if m.max() > 160:
        assert untouched > 0


def test_pure_recency_layers_keep_their_newest_m_l_tokens():
    wl = CONFIGS["toy"]
    cfg, st, fd, ids, hist = _run_lb(wl, 5, (1.3, 1.0, 0.7), n_shallow=4, n_deep=0, lambda_shallow=0.0)
    m = ho.layer_budgets(cfg)
    for l in range(wl.n_layers):                                # sliding window of PAPER.md:49, one width per layer
        assert ids[l].tolist() == list(range(fd.tokens_fed - m[l], fd.tokens_fed))


# ---- summary tokens under layer-dependent budgets (DESIGN f1 x f4) ---------------------------------------------
def test_equal_weights_with_summary_token_reproduce_the_uniform_path_bit_for_bit():
    wl = CONFIGS["toy"]
    _, st_u, _, ids_u, hist_u = run_oracle_schedule(wl, 6, cfg_over=dict(summary_token=True))
    cfg, st, fd, ids, hist = _run_lb(wl, 6, (1.0, 1.0, 1.0), capacity=wl.cap, summary_token=True)
    M = wl.budget
    assert (st.lens == M).all() and st.next_pos == st_u.next_pos
    assert st.K[:, :M].tobytes() == st_u.K[:, :M].tobytes() and st.V[:, :M].tobytes() == st_u.V[:, :M].tobytes()
    assert np.array_equal(st.pos[:, :, :M], st_u.pos[:, :, :M]) and np.array_equal(np.stack(ids), ids_u)


@pytest.mark.parametrize("lazy", [False, True])
@pytest.mark.parametrize("w", TAB5[1:])
def test_summary_token_of_a_deep_layer_is_alg1_of_what_that_layer_evicted(w, lazy):
    """Toy: 4 layers, layer 3 deep.  At every step at which layer 3 compresses, its last slot (m_3 - 1) is Alg. 1 recomputed
    here from the candidates it evicted (previous cache + chunk, at their positions); the other layers never hold one; a
    step at which layer 3 is still under its budget makes none.  Lazy mode: target = the position after the newest token,
    and the next chunk starts one position later."""
    wl = CONFIGS["toy"]
    over = dict(summary_token=True)
    if lazy:
        over.update(reindex_mode="lazy", max_position=100000, max_chunk_span=wl.chunk_tokens)
    cfg, st, fd, ids, hist = _run_lb(wl, 8, w, **over)
    m = ho.layer_budgets(cfg)
    made = 0
    for h in hist[1:]:
        out, pre = h["out"], h["pre"]
        n3, n_new = int(pre["lens"][3]), h["K_new"].shape[1]
        T3 = n3 + n_new
        if not out["evicted"] or T3 <= m[3]:
            if out["evicted"]:
                assert np.array_equal(out["kept"][3], np.arange(T3))        # untouched: no summary token
            continue
        kept3 = np.asarray(out["kept"][3])
        assert len(kept3) == m[3] and kept3[-1] == -1 and (np.diff(kept3[:-1]) > 0).all()
        for l in range(3):
            assert (np.asarray(out["kept"][l]) >= 0).all()
        K_cand = np.concatenate([pre["K"][3, :n3], h["K_new"][3]], axis=0)
        V_cand = np.concatenate([pre["V"][3, :n3], h["V_new"][3]], axis=0)
        P_cand = np.concatenate([pre["pos"][3][:, :n3], h["p_arr"]], axis=1)
        ev = np.setdiff1d(np.arange(T3), kept3[:-1])
        assert len(ev) == T3 - (m[3] - 1)
        p_end = int(h["p_arr"][0, -1]) + 1
        t = cfg.pos_offset + m[3] - 1 if out["reindexed"] else p_end
        k_sum, v_sum = ho.summary_token(cfg, K_cand[ev], V_cand[ev], P_cand[:, ev], t)
        assert out["pos_new"][3][0, -1] == t and (np.diff(out["pos_new"][3][0]) > 0).all()
        made += 1
        h["expect"] = (k_sum, v_sum)
    assert made >= 5
    # the last step's summary token is still in the cache as computed
    k_sum, v_sum = hist[-1]["expect"]
    assert np.array_equal(st.K[3, m[3] - 1], k_sum) and np.array_equal(st.V[3, m[3] - 1], v_sum)
    assert ids[3][-1] == -1 and all((i >= 0).all() for i in ids[:3])
    if lazy:                                                                # one position per step went to a summary token
        assert st.next_pos == cfg.pos_offset + fd.tokens_fed + made
