"""Pins for the scoring half of the oracle (Eq. 1-7): closed forms, hand fixtures, a library
softmax, invariants.  Each test names the mistake it would catch."""
import numpy as np
import pytest
import torch

from helpers import oracle_config, read_fixture
from oracle import hermes_oracle as ho
from workloads import CONFIGS


def _cfg(L=2, **kw):
    base = dict(n_layers=L, n_q_heads=4, n_kv_heads=2, head_dim=8, budget=2, forget_rate=0.5, dtype="f32")
    base.update(kw)
    return ho.OracleConfig(**base)


# ---- hand-worked example (tests/golden/hand_example.txt) -------------------------------------
def test_hand_example_scores_and_selection():
    fx = read_fixture("hand_example.txt")
    cfg = _cfg(L=2, pos_offset=5)
    T = 4
    W = np.zeros((2, T))
    W[1] = fx["W1"]
    np.testing.assert_allclose(ho.normalise_attention(W[1], "max"), fx["A1"], atol=1e-12)
    np.testing.assert_allclose(ho.recency_scores(T, 0.5, "max"), fx["R"], atol=5e-7)
    S = ho.raw_scores(cfg, W, T)
    St = ho.smooth_scores(cfg, S)
    np.testing.assert_allclose(St[0], fx["S_tilde0"], atol=1e-6)   # catches swapped lambda / (1-lambda)
    np.testing.assert_allclose(St[1], fx["S_tilde1"], atol=1e-12)  # last layer untouched
    assert ho.select_topk(St[0], 2).tolist() == fx["kept0_m2"].astype(int).tolist()
    assert ho.select_topk(St[1], 2).tolist() == fx["kept1_m2"].astype(int).tolist()
    assert ho.select_topk(St[1], 3).tolist() == fx["kept1_m3"].astype(int).tolist()  # tie -> larger index
    pos = np.array([[5, 6, 7, 8]])
    for l, key in ((0, "delta0_m2"), (1, "delta1_m2")):
        I = ho.select_topk(St[l], 2)
        p_new = ho.compact_positions(cfg, pos[:, I])
        assert p_new[0].tolist() == fx["pos_new_m2"].astype(int).tolist()
        assert (p_new - pos[:, I])[0].tolist() == fx[key].astype(int).tolist()


def test_omega_lambda_split_tables():
    fx = read_fixture("omega_table.txt")
    cfg = _cfg(L=28, n_q_heads=28, n_kv_heads=4)
    for l, w in fx["rows"]:
        assert ho.omega_of_layer(cfg, int(l)) == pytest.approx(w, abs=1e-12)
    for L in (28, 80, 4, 2):
        assert list(ho.stage_split(L)) == fx[f"split_{L}"].astype(int).tolist()
    lam = [ho.lambda_of_layer(cfg, l) for l in (0, 3, 19, 20)]
    assert lam == pytest.approx(fx["lambda_28"].tolist())


def test_omega_degenerate_single_middle_layer():
    cfg = _cfg(L=3, n_shallow=1, n_deep=1)           # one middle layer: l_long == l_short
    assert ho.omega_of_layer(cfg, 1) == 0.75


# ---- Eq. 1 -----------------------------------------------------------------------------------
def test_recency_closed_forms():
    T, k = 37, 0.21
    R = ho.recency_scores(T, k, "max")
    assert R[-1] == 1.0 and np.all(np.diff(R) > 0)                 # newest token scores highest
    np.testing.assert_allclose(R[0], np.exp(-k * (T - 1)), rtol=1e-14)
    np.testing.assert_allclose(R[1:] / R[:-1], np.exp(k), rtol=1e-12)   # geometric in i
    Rs = ho.recency_scores(T, k, "sum")
    np.testing.assert_allclose(Rs.sum(), 1.0, rtol=1e-14)
    np.testing.assert_allclose(Rs[-1], (1 - np.exp(-k)) / (1 - np.exp(-k * T)), rtol=1e-13)


# ---- Eq. 2 -----------------------------------------------------------------------------------
def _qk(T=53, Hq=6, Hkv=3, P=5, d=16, seed=1):
    g = np.random.default_rng(seed)
    return (g.standard_normal((Hq, P, d)).astype(np.float32),
            g.standard_normal((T, Hkv, d)).astype(np.float32))


def test_attention_matches_library_softmax():
    Q, K = _qk()
    G, scale = 2, 0.25
    W = ho.attention_weights(Q, K, G, scale)
    Qt, Kt = torch.from_numpy(Q).double(), torch.from_numpy(K).double()
    Kh = Kt.permute(1, 0, 2).repeat_interleave(G, dim=0)           # [Hq, T, d]
    P = torch.softmax(scale * torch.einsum("hpd,htd->hpt", Qt, Kh), dim=-1)
    np.testing.assert_allclose(W, P.mean(dim=(0, 1)).numpy(), rtol=1e-12)


def test_attention_invariants():
    Q, K = _qk()
    W = ho.attention_weights(Q, K, 2, 0.25)
    assert W.sum() == pytest.approx(1.0, abs=1e-13)
    T = K.shape[0]
    np.testing.assert_allclose(ho.attention_weights(np.zeros_like(Q), K, 2, 0.25), 1.0 / T, rtol=1e-14)
    perm = np.random.default_rng(3).permutation(T)                 # permuting tokens permutes W
    np.testing.assert_allclose(ho.attention_weights(Q, K[perm], 2, 0.25), W[perm], rtol=1e-12)
    K_mha = np.repeat(K, 2, axis=1)                                # GQA == MHA with replicated heads
    np.testing.assert_allclose(ho.attention_weights(Q, K_mha, 1, 0.25), W, rtol=1e-12)
    # wrong head->group map (h % Hkv instead of h // G) would change W:
    K_roll = K[:, [1, 2, 0], :]
    assert not np.allclose(ho.attention_weights(Q, K_roll, 2, 0.25), W)


def test_attention_large_logits_are_stable():
    Q, K = _qk()
    W = ho.attention_weights(Q * 60, K * 60, 2, 1.0)               # logits ~ 1e4: needs the max shift
    assert np.isfinite(W).all() and W.sum() == pytest.approx(1.0, abs=1e-12)


# ---- Eq. 4 / Eq. 5 ---------------------------------------------------------------------------
def test_layer_weighting_reduces_to_eq1_eq2():
    cfg = _cfg(L=10, n_q_heads=4, n_kv_heads=2)                    # 1 shallow / 6 middle / 3 deep
    T = 20
    W = np.random.default_rng(0).random((10, T)) + 0.01
    S = ho.raw_scores(cfg, W, T)
    R = ho.recency_scores(T, cfg.forget_rate)
    np.testing.assert_array_equal(S[0], R)                          # shallow = Eq. 1
    np.testing.assert_allclose(S[9], W[9] / W[9].max(), rtol=1e-15)  # deep = Eq. 2
    w = ho.omega_of_layer(cfg, 3)
    np.testing.assert_allclose(S[3], (1 - w) * W[3] / W[3].max() + w * R, rtol=1e-15)
    assert 0.15 - 1e-12 <= ho.omega_of_layer(cfg, 6) <= ho.omega_of_layer(cfg, 1) <= 0.75 + 1e-12


def test_smoothing_limits():
    S = np.random.default_rng(2).random((5, 9))
    c0 = _cfg(L=5, lambda_shallow=0, lambda_middle=0, lambda_deep=0)
    np.testing.assert_array_equal(ho.smooth_scores(c0, S), S)       # lambda = 0: unchanged (Tab. 6 row 0/0/0)
    c1 = _cfg(L=5, lambda_shallow=1, lambda_middle=1, lambda_deep=1)
    St = ho.smooth_scores(c1, S)
    np.testing.assert_array_equal(St[:-1], S[1:])                   # lambda = 1: layer l+1's RAW score
    np.testing.assert_array_equal(St[-1], S[-1])
    c = _cfg(L=5)
    St = ho.smooth_scores(c, S)                                     # non-recursive: uses raw S[l+1]
    lam = ho.lambda_of_layer(c, 1)
    np.testing.assert_allclose(St[1], (1 - lam) * S[1] + lam * S[2], rtol=1e-15)
    St2 = ho.smooth_scores(c, 2 * S + 0)                            # linear in S
    np.testing.assert_allclose(St2, 2 * St, rtol=1e-15)


# ---- Eq. 6 -----------------------------------------------------------------------------------
def test_topk_bruteforce_and_pairwise():
    from itertools import combinations
    g = np.random.default_rng(5)
    for T in range(2, 13):
        for m in range(1, T):
            s = np.round(g.random(T), 1)                            # coarse values -> many ties
            I = ho.select_topk(s, m)
            assert len(I) == m and np.all(np.diff(I) > 0)           # exactly |M|, ascending
            best = max(sum(s[list(c)]) for c in combinations(range(T), m))
            assert s[I].sum() == pytest.approx(best, abs=1e-12)     # maximises the kept score mass
            ev = np.setdiff1d(np.arange(T), I)
            for i in I:
                for j in ev:
                    assert s[i] > s[j] or (s[i] == s[j] and i > j)  # tie -> more recent index kept


def test_pure_recency_layer_is_fifo():
    R = ho.recency_scores(50, 0.1)
    assert ho.select_topk(R, 30).tolist() == list(range(20, 50))    # sliding window of PAPER.md:49
    flat = np.ones(50)                                              # total underflow -> still FIFO by tie rule
    assert ho.select_topk(flat, 30).tolist() == list(range(20, 50))


def test_workload_to_oracle_config_defaults():
    cfg = oracle_config(CONFIGS["llava_ov_7b"])
    assert ho.stage_split(cfg.n_layers) == (3, 17, 8)
    assert cfg.forget_rate == pytest.approx(4.0 / 6272)
