"""Pins for per-stage probe row ranges (hybrid guidance, App. B; DESIGN f3) in the oracle."""
import numpy as np
import torch

from helpers import Feeder, fill_chunks, oracle_config
from oracle import hermes_oracle as ho
from workloads import CONFIGS


def _one_step(over, q_edit=None):
    wl = CONFIGS["toy"]
    cfg = oracle_config(wl, **over)
    st = ho.OracleStream(cfg)
    fd = Feeder(wl)
    for n in fill_chunks(wl):
        K, V, _, _ = fd.next(n, ho.arrival_positions(cfg, st, n, -1), False)
        ho.oracle_step(st, K, V, None)
    K, V, Q, _ = fd.next(wl.chunk_tokens, ho.arrival_positions(cfg, st, wl.chunk_tokens, -1), True)
    if q_edit is not None:
        Q = q_edit(Q.copy())
    K_all = np.concatenate([st.K[:, :st.len], K], axis=1)
    return wl, cfg, ho.oracle_step(st, K, V, Q), Q, K_all


def test_default_uses_all_rows_everywhere():
    _, _, a, _, _ = _one_step({})
    _, _, b, _, _ = _one_step(dict(probe_deep_begin=0))
    assert np.array_equal(a["W"], b["W"]) and np.array_equal(a["kept"], b["kept"])


def test_deep_layers_see_only_the_global_rows():
    wl, cfg, out, Q, K_all = _one_step(dict(probe_deep_begin=3))
    G = wl.n_q_heads // wl.n_kv_heads
    scale = 1.0 / np.sqrt(wl.head_dim)
    for l, rows in ((1, slice(0, None)), (2, slice(0, None)), (3, slice(3, None))):      # toy: layers 1, 2 middle, 3 deep
        q = torch.from_numpy(Q[l][:, rows]).double()                                      # [H_q, P', d]
        k = torch.from_numpy(K_all[l]).double()[:, np.arange(wl.n_q_heads) // G, :]       # [T, H_q, d]
        p = torch.softmax(torch.einsum("hpd,thd->hpt", q, k) * scale, dim=-1)
        np.testing.assert_allclose(out["W"][l], p.mean(dim=(0, 1)).numpy(), rtol=1e-12)


def test_local_rows_do_not_influence_deep_layers():
    def edit(Q):
        Q[:, :, :3] *= -2.5                       # scramble the local-prompt rows only
        return Q
    _, _, a, _, _ = _one_step(dict(probe_deep_begin=3))
    _, _, b, _, _ = _one_step(dict(probe_deep_begin=3), edit)
    assert np.array_equal(a["W"][3], b["W"][3])                       # deep layer unchanged
    assert not np.allclose(a["W"][1], b["W"][1])                      # middle layers do use them
