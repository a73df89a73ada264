"""Seeded, synthetic K / V / probe-Q tensors shaped like the paper's workloads.

They stand in for what LLaVA-OV-7B / Qwen2.5-VL-7B would produce on the paper's videos
(28 layers, 196 tokens per frame; one high-attention "anchor"
token per frame, exactly N_f apart; recency bias).  None of the paper's
benchmark data or model weights is used or needed.  Geometry per BASELINE.json `configs`.

Nothing here is the method's arithmetic.  `rope_at_arrival` is the MLLM's own rotary
embedding of a fresh key at its arrival position (input preparation for config 1, so
that the rotation-composition pin can be checked end to end); the method's rotary DELTA
correction lives only in `oracle/` and in the CUDA kernels.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

_MASK64 = (1 << 64) - 1


def _mix(*ints: int) -> int:
    """splitmix64-style fold of a tuple of ints into one 64-bit key."""
    x = 0x9E3779B97F4A7C15
    for v in ints:
        x = (x ^ (int(v) & _MASK64)) & _MASK64
        x = (x + 0x9E3779B97F4A7C15) & _MASK64
        x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
        x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _MASK64
        x = x ^ (x >> 31)
    return x


_TAGS = {"K": 1, "V": 2, "Q": 3, "U": 4, "misc": 5}


def stream_rng(seed: int, stream: int, tag: str, *idx: int) -> np.random.Generator:
    """Counter-based generator keyed by (seed, stream, tensor tag, indices)."""
    return np.random.Generator(np.random.Philox(key=[_mix(seed, stream), _mix(_TAGS[tag], *idx)]))


def round_storage(x: np.ndarray, dtype: str) -> np.ndarray:
    """fp32 array -> fp32 array whose values are representable in `dtype` (RNE)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    if dtype == "f32":
        return x
    u = x.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32)


def storage_bits(x: np.ndarray, dtype: str) -> np.ndarray:
    """Bit pattern of storage-representable fp32 values (uint32 for f32, uint16 for bf16)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    return u if dtype == "f32" else (u >> 16).astype(np.uint16)


@dataclass(frozen=True)
class Workload:
    name: str
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    dtype: str                 # "f32" | "bf16"
    tokens_per_frame: int      # N_f (per temporal step for M-RoPE)
    budget: int                # |M|
    chunk_tokens: int          # C
    probe_tokens: int          # P
    rope_theta: float
    seed: int
    n_streams: int = 1
    rope_mode: str = "1d"
    mrope_section: tuple = (16, 24, 24)
    mrope_compact_axes: int = 0b001
    mrope_grid_h: int = 8
    mrope_grid_w: int = 8
    pos_offset: int = 0
    preload_tokens: int = 0    # tokens appended without a probe before the first scored arrival
    capacity: int = 0          # 0 -> budget + chunk_tokens
    anchor_slot: int = -1      # -1 -> N_f / 2
    anchor_gain: float = 3.0
    drift_beta: float = 0.125  # 0 -> no recency drift
    apply_rope: bool = False   # config 1: generate un-rotated k0 and rotate at arrival
    forget_rate: float = 0.0   # 0 -> 4 / budget (DESIGN c1)
    timed_updates: int = 256

    @property
    def k_forget(self) -> float:
        return self.forget_rate if self.forget_rate > 0 else 4.0 / self.budget

    @property
    def cap(self) -> int:
        return self.capacity if self.capacity > 0 else self.budget + self.chunk_tokens

    @property
    def n_axes(self) -> int:
        return 3 if self.rope_mode == "m3d" else 1

    @property
    def anchor(self) -> int:
        return self.anchor_slot if self.anchor_slot >= 0 else self.tokens_per_frame // 2

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


def _llava(name, budget=6272, probe=64, seed=2000, **kw):
    return Workload(name=name, n_layers=28, n_q_heads=28, n_kv_heads=4, head_dim=128, dtype="bf16",
                    tokens_per_frame=196, budget=budget, chunk_tokens=196, probe_tokens=probe,
                    rope_theta=1.0e6, seed=seed, **kw)


CONFIGS = {
    # BASELINE.json configs[0]: 8 frames x 16 tokens cached + 2 x 16 incoming, budget 96, 10 arrivals
    "toy": Workload(name="toy", n_layers=4, n_q_heads=4, n_kv_heads=2, head_dim=64, dtype="f32",
                    tokens_per_frame=16, budget=96, chunk_tokens=32, probe_tokens=8,
                    rope_theta=1.0e4, seed=0, preload_tokens=128, capacity=160, anchor_slot=0,
                    drift_beta=0.0, apply_rope=True, timed_updates=10),
    # configs[1]: LLaVA-OV-7B geometry (Qwen2-7B backbone), the benchmark workload
    "llava_ov_7b": _llava("llava_ov_7b"),
    # the same geometry with the paper's 16-frame chunk (16 frames x 196 tokens)
    "llava_ov_7b_c16": _llava("llava_ov_7b_c16", seed=2016).scaled(chunk_tokens=3136, timed_updates=64),
    # configs[2]: Qwen2.5-VL-7B geometry, M-RoPE, 64 tokens per temporal step, t-only compaction
    "qwen25_vl_7b": Workload(name="qwen25_vl_7b", n_layers=28, n_q_heads=28, n_kv_heads=4,
                             head_dim=128, dtype="bf16", tokens_per_frame=64, budget=8192,
                             chunk_tokens=128, probe_tokens=128, rope_theta=1.0e6, seed=3000,
                             rope_mode="m3d"),
    # configs[4]: 72B-class geometry, 16 independent streams in one batch
    "batched_72b": Workload(name="batched_72b", n_layers=80, n_q_heads=64, n_kv_heads=8,
                            head_dim=128, dtype="bf16", tokens_per_frame=196, budget=4096,
                            chunk_tokens=196, probe_tokens=64, rope_theta=1.0e6, seed=5000,
                            n_streams=16, timed_updates=32),
}


def sweep_point(budget: int, probe: int) -> Workload:
    """configs[3]: LLaVA-OV-7B geometry, budget in {2K..32K}, probe in {16, 64, 256}."""
    return _llava(f"sweep_m{budget}_p{probe}", budget=budget, probe=probe, seed=4000)


def _drift_dirs(wl: Workload) -> np.ndarray:
    """u in {+1,-1}^d fixed per (layer, KV head): [L, H_kv, d]."""
    g = stream_rng(wl.seed, 0, "U")
    return np.where(g.random((wl.n_layers, wl.n_kv_heads, wl.head_dim)) < 0.5, -1.0, 1.0).astype(np.float32)


def rope_at_arrival(k0: np.ndarray, pos: np.ndarray, wl: Workload) -> np.ndarray:
    """The MLLM's rotary embedding of fresh keys: k0 [L, n, H_kv, d], pos [A, n] -> rotated fp32,
    computed with fp64 complex numbers on half-split pairs (j, j + d/2), theta_j = base^(-2j/d)."""
    d = wl.head_dim
    half = d // 2
    theta = float(wl.rope_theta) ** (-2.0 * np.arange(half, dtype=np.float64) / d)
    if wl.rope_mode == "1d":
        p = np.broadcast_to(pos[0][:, None], (pos.shape[1], half))
    else:
        s_t, s_h, s_w = wl.mrope_section
        ax = np.array([0] * s_t + [1] * s_h + [2] * s_w)
        p = pos[ax, :].T
    phase = np.exp(1j * p.astype(np.float64) * theta[None, :])             # [n, half]
    z = k0[..., :half].astype(np.float64) + 1j * k0[..., half:].astype(np.float64)
    z = z * phase[None, :, None, :]
    return np.concatenate([z.real, z.imag], axis=-1).astype(np.float32)


def chunk_kv(wl: Workload, stream: int, update: int, first_token: int, n_new: int,
             arrival_pos: np.ndarray | None = None):
    """K_new, V_new [L, n_new, H_kv, d] (fp32 holding storage values) of one arriving chunk,
    plus the un-rotated k0 (config 1 only, else None).

    `first_token` is the global number of the chunk's first token in its stream (frame =
    token // N_f, slot = token % N_f); `update` keys the random draw."""
    shape = (wl.n_layers, n_new, wl.n_kv_heads, wl.head_dim)
    K = stream_rng(wl.seed, stream, "K", update).standard_normal(shape, dtype=np.float32)
    V = stream_rng(wl.seed, stream, "V", update).standard_normal(shape, dtype=np.float32)
    tok = first_token + np.arange(n_new)
    frame, slot = tok // wl.tokens_per_frame, tok % wl.tokens_per_frame
    K[:, slot == wl.anchor] *= np.float32(wl.anchor_gain)                  # frame-level anchor token
    if wl.drift_beta > 0:
        r = ((frame % 512) / 32.0).astype(np.float32)                       # mild recency drift
        K += np.float32(wl.drift_beta) * r[None, :, None, None] * _drift_dirs(wl)[:, None, :, :]
    k0 = None
    if wl.apply_rope:
        assert arrival_pos is not None
        k0 = round_storage(K, wl.dtype)
        K = rope_at_arrival(k0, arrival_pos, wl)
    return round_storage(K, wl.dtype), round_storage(V, wl.dtype), k0


def probe_q(wl: Workload, stream: int, update: int, n_probe: int | None = None) -> np.ndarray:
    """Query states of the guidance prompt: [L, H_q, P, d], N(0,1) + u_{l, h//G} / sqrt(d)."""
    P = wl.probe_tokens if n_probe is None else n_probe
    shape = (wl.n_layers, wl.n_q_heads, P, wl.head_dim)
    Q = stream_rng(wl.seed, stream, "Q", update).standard_normal(shape, dtype=np.float32)
    if wl.drift_beta > 0:
        G = wl.n_q_heads // wl.n_kv_heads
        u = np.repeat(_drift_dirs(wl), G, axis=1)                            # [L, H_q, d]
        Q += u[:, :, None, :] / np.float32(np.sqrt(wl.head_dim))
    return round_storage(Q, wl.dtype)
