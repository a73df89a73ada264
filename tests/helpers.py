"""Test-side glue: workload -> oracle config, schedule driver, fixture reader, comparisons."""
from __future__ import annotations

import os

import numpy as np

from oracle import hermes_oracle as ho
from workloads import Workload, chunk_kv, probe_q

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_fixture(name: str) -> dict:
    """`key: v v v` lines -> {key: np.array}; bare `a b` lines are collected under 'rows'."""
    out, rows = {}, []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            if ":" in line:
                k, v = line.split(":", 1)
                out[k.strip()] = np.array([float(x) for x in v.split()])
            else:
                rows.append([float(x) for x in line.split()])
    if rows:
        out["rows"] = np.array(rows)
    return out


def oracle_config(wl: Workload, **over) -> ho.OracleConfig:
    kw = dict(n_layers=wl.n_layers, n_q_heads=wl.n_q_heads, n_kv_heads=wl.n_kv_heads,
              head_dim=wl.head_dim, budget=wl.budget, forget_rate=wl.k_forget, dtype=wl.dtype,
              rope_mode=wl.rope_mode, rope_theta=wl.rope_theta, mrope_section=wl.mrope_section,
              mrope_compact_axes=wl.mrope_compact_axes, mrope_grid_h=wl.mrope_grid_h,
              mrope_grid_w=wl.mrope_grid_w, pos_offset=wl.pos_offset, capacity=wl.cap)
    kw.update(over)
    return ho.OracleConfig(**kw)


class Feeder:
    """Generates the chunk / probe sequence of one stream of a workload (same for both sides)."""

    def __init__(self, wl: Workload, stream: int = 0):
        self.wl, self.stream = wl, stream
        self.tokens_fed = 0
        self.update = 0
        self.k0_by_id = {}           # config 1: un-rotated key of every token id, [L, H_kv, d]

    def next(self, n_new: int, arrival_pos: np.ndarray | None, with_probe: bool, n_probe=None):
        wl = self.wl
        K, V, k0 = chunk_kv(wl, self.stream, self.update, self.tokens_fed, n_new, arrival_pos)
        if k0 is not None:
            for j in range(n_new):
                self.k0_by_id[self.tokens_fed + j] = k0[:, j]
        Q = probe_q(wl, self.stream, self.update, n_probe) if with_probe else None
        ids = np.arange(self.tokens_fed, self.tokens_fed + n_new)
        self.tokens_fed += n_new
        self.update += 1
        return K, V, Q, ids


def take_ids(ids: np.ndarray, kept: np.ndarray) -> np.ndarray:
    """Token ids of the kept slots; kept == -1 (a summary token, DESIGN f1) gets id -1."""
    out = np.take_along_axis(ids, np.maximum(kept, 0), axis=1)
    out[kept < 0] = -1
    return out


def fill_chunks(wl: Workload):
    """Chunk sizes of the un-probed fill phase: preload (config 1) or chunks up to the budget."""
    if wl.preload_tokens:
        return [wl.preload_tokens]
    n_full = wl.budget // wl.chunk_tokens
    sizes = [wl.chunk_tokens] * n_full
    if wl.budget - n_full * wl.chunk_tokens:
        sizes.append(wl.budget - n_full * wl.chunk_tokens)
    return sizes


def run_oracle_schedule(wl: Workload, n_updates: int, cfg_over=None, stream: int = 0):
    """Fill, then `n_updates` scored arrivals through the oracle alone.  Tracks token ids."""
    cfg = oracle_config(wl, **(cfg_over or {}))
    st = ho.OracleStream(cfg)
    fd = Feeder(wl, stream)
    ids = np.zeros((wl.n_layers, 0), np.int64)
    history = []
    for n in fill_chunks(wl):
        ap = ho.arrival_positions(cfg, st, n, -1)
        K, V, _, new_ids = fd.next(n, ap, with_probe=False)
        ho.oracle_step(st, K, V, None)
        ids = np.concatenate([ids, np.broadcast_to(new_ids, (wl.n_layers, n))], axis=1)
    for _ in range(n_updates):
        n = wl.chunk_tokens
        ap = ho.arrival_positions(cfg, st, n, -1)
        K, V, Q, new_ids = fd.next(n, ap, with_probe=True)
        pre_len = st.len
        V_pre = st.V[:, :pre_len].copy()
        out = ho.oracle_step(st, K, V, Q)
        ids = np.concatenate([ids, np.broadcast_to(new_ids, (wl.n_layers, n))], axis=1)
        if out["evicted"]:
            ids = take_ids(ids, out["kept"])
        history.append(dict(out=out, ids=ids.copy(), V_pre=V_pre, V_new=V, K_new=K, Q=Q, pre_len=pre_len))
    return cfg, st, fd, ids, history


def bf16_ulp(x: np.ndarray) -> np.ndarray:
    """Spacing of bf16 numbers at |x| (8 significand bits incl. the hidden one)."""
    ax = np.maximum(np.abs(x).astype(np.float64), 2.0 ** -126)
    return 2.0 ** (np.floor(np.log2(ax)) - 7)
