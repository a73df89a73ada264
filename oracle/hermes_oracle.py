"""CPU oracle for the HERMES per-chunk hierarchical KV-cache update (arXiv 2601.14724).

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and the
`cpu_baseline` / `--impl reference` legs of `bench.py` may import this module.
It shares no code with the CUDA path (`paper_2601_14724_b200/`), imports
nothing from it, and is never a fallback for it.

The method is a heuristic pipeline, so the oracle is the algorithm written out
step by step, in the paper's order and notation, with numpy: fp64 for every
score, fp32 for the rotary correction (then round-to-nearest-even to the
storage dtype).  Library primitives used as steps: `@` (matmul), `np.exp`,
`np.lexsort`, `np.unique`, `np.cos`, `np.sin`.  No blocking, fusion or
re-ordering beyond what the equations state.

Citations are `PAPER.md:<line>` (the text under /root/reference at build time)
plus the equation; "DESIGN c<N>" points at the numbered reading in DESIGN.md
where the paper is silent, ambiguous or garbled.

Parity status: every function below is pinned by
`tests/test_oracle_*.py` against closed forms, hand-worked fixtures in
`tests/golden/`, a torch-fp64 library softmax, brute force and invariants.
PARITY UNPINNED (the paper prints no number that depends on them): the choice
of normalisation factor alpha (DESIGN c2), the value of the forgetting rate k
(c1), the mean over heads / probe rows (c3) and the softmax domain (c4).
Also unpinned against the authors' code: where the summary token sits, its target
position and the budget accounting (DESIGN f1), and the exact lazy re-index trigger
(DESIGN f2); the arithmetic of both IS pinned (tests/test_oracle_summary.py,
tests/test_oracle_lazy.py).

Storage convention: K and V are held as float32 arrays whose values are exactly
representable in the storage dtype ("f32" or "bf16"); positions are int64.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

__all__ = [
    "OracleConfig", "OracleStream", "stage_split", "layer_stage", "omega_of_layer",
    "lambda_of_layer", "attention_weights", "recency_scores", "normalise_attention",
    "raw_scores", "smooth_scores", "select_topk", "compact_positions",
    "rope_frequencies", "pair_axis", "rotary_delta", "round_to_storage", "oracle_step",
    "summary_token", "lazy_reindex_due", "layer_budgets", "smooth_scores_aligned", "oracle_step_layer_budgets",
]


# --------------------------------------------------------------------------- config
@dataclass
class OracleConfig:
    """Problem statement of the update path."""
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    budget: int                       # |M| tokens per layer
    forget_rate: float                # k of Eq. 1, PAPER.md:82 (paper gives no value: DESIGN c1)
    dtype: str = "bf16"               # storage dtype of K/V: "f32" | "bf16"
    n_shallow: int = -1               # -1 -> 10 % / 30 % rule, PAPER.md:144 (DESIGN c7)
    n_deep: int = -1
    l_short: int = -1                 # -1 -> first / last middle layer (DESIGN c8)
    l_long: int = -1
    omega0: float = 0.75
    gamma: float = 0.6
    norm_mode: str = "max"            # alpha of Eq. 1/2: "max" | "sum" (DESIGN c2)
    lambda_shallow: float = 0.1       # PAPER.md:508 (Eq. 7)
    lambda_middle: float = 0.3
    lambda_deep: float = 0.4
    softmax_scale: float = 0.0        # 0 -> 1/sqrt(head_dim) (DESIGN c4)
    rope_mode: str = "1d"             # "1d" (App. E.1) | "m3d" (App. E.2)
    rope_theta: float = 10000.0
    mrope_section: tuple = (16, 24, 24)   # rotary pairs per (t, h, w) axis, sum = head_dim/2
    mrope_compact_axes: int = 0b001   # bit0 t, bit1 h, bit2 w (DESIGN c13)
    mrope_grid_h: int = 8
    mrope_grid_w: int = 8
    pos_offset: int = 0               # length of the fixed system prefix
    reindex_mode: str = "eager"       # "eager" | "lazy" (DESIGN f2)
    max_position: int = 0             # lazy: the model's position limit that triggers a re-index
    max_chunk_span: int = 0           # lazy: largest position span of one arriving chunk (tokens; M-RoPE: t steps)
    probe_deep_begin: int = 0         # deep layers use probe rows [begin, P): the global prompt only (DESIGN f3)
    summary_token: bool = False       # deep layers: evicted tokens -> one summary token (Alg. 1; DESIGN f1)
    capacity: int = 0                 # slots per layer; 0 -> budget + largest chunk seen
    budget_weights: tuple = (1.0, 1.0, 1.0)   # layer-dependent budgets: weight of a shallow / middle / deep layer
                                      # (Tab. 5; DESIGN f4); equal weights = `budget` everywhere

    @property
    def n_axes(self) -> int:
        return 3 if self.rope_mode == "m3d" else 1

    @property
    def group(self) -> int:           # G query heads per KV head
        return self.n_q_heads // self.n_kv_heads


def stage_split(n_layers: int, n_shallow: int = -1, n_deep: int = -1):
    """10 % shallow / 60 % middle / 30 % deep; rounding is DESIGN c7:
    n_shallow = max(1, round-half-up(0.1 L)), n_deep = max(1, round-half-up(0.3 L))."""
    if n_shallow < 0:
        n_shallow = max(1, (n_layers + 5) // 10)
    if n_deep < 0:
        n_deep = max(1, (3 * n_layers + 5) // 10)
    n_middle = n_layers - n_shallow - n_deep
    if n_middle < 0:
        raise ValueError("n_shallow + n_deep exceeds n_layers")
    return n_shallow, n_middle, n_deep


def layer_stage(cfg: OracleConfig, l: int) -> str:
    n_s, n_m, _ = stage_split(cfg.n_layers, cfg.n_shallow, cfg.n_deep)
    if l < n_s:
        return "shallow"
    if l < n_s + n_m:
        return "middle"
    return "deep"


def omega_of_layer(cfg: OracleConfig, l: int) -> float:
    """Weight of the recency term at layer l.

    shallow: 1 (Eq. 1 alone); deep: 0 (Eq. 2 alone);
    middle: Eq. 3: w = w0 - gamma (l - l_short)/(l_long - l_short),
    with l_short / l_long = first / last middle layer (DESIGN c8)."""
    stage = layer_stage(cfg, l)
    if stage == "shallow":
        return 1.0
    if stage == "deep":
        return 0.0
    n_s, n_m, _ = stage_split(cfg.n_layers, cfg.n_shallow, cfg.n_deep)
    l_short = cfg.l_short if cfg.l_short >= 0 else n_s
    l_long = cfg.l_long if cfg.l_long >= 0 else n_s + n_m - 1
    if l_long == l_short:
        return float(cfg.omega0)
    return float(cfg.omega0) - float(cfg.gamma) * (l - l_short) / (l_long - l_short)


def lambda_of_layer(cfg: OracleConfig, l: int) -> float:
    """Eq. 7: 0.1 / 0.3 / 0.4 by the stage of layer l."""
    return {"shallow": cfg.lambda_shallow, "middle": cfg.lambda_middle,
            "deep": cfg.lambda_deep}[layer_stage(cfg, l)]


# --------------------------------------------------------------------------- scores
def attention_weights(Q: np.ndarray, K: np.ndarray, group: int, scale: float) -> np.ndarray:
    """W_i of Eq. 2 for one layer.

    Q: [H_q, P, d] pseudo-query states (guidance prompt), K: [T, H_kv, d]
    cached keys.  For every query head h and probe row r, a softmax over the T
    video tokens (DESIGN c4) of scale * q . k with k from KV head h // group;
    W_i = arithmetic mean over all heads and probe rows (DESIGN c3; "average
    attention weights")."""
    H_q, P, _ = Q.shape
    T = K.shape[0]
    Q64 = Q.astype(np.float64)
    K64 = K.astype(np.float64)
    W = np.zeros(T, dtype=np.float64)
    for h in range(H_q):
        s = scale * (Q64[h] @ K64[:, h // group, :].T)        # [P, T]
        m = s.max(axis=1, keepdims=True)
        e = np.exp(s - m)
        Z = e.sum(axis=1, keepdims=True)
        W += (e / Z).sum(axis=0)
    return W / float(H_q * P)


def recency_scores(T: int, k: float, norm_mode: str = "max") -> np.ndarray:
    """Eq. 1: alpha * exp(-k * dt_i), dt_i = T - 1 - i (i = cache index).

    alpha (DESIGN c2): "max" -> 1 / max_i = 1 (the newest token has dt = 0);
    "sum" -> 1 / sum_i exp(-k dt_i) = (1 - e^-k) / (1 - e^-kT)."""
    dt = (T - 1 - np.arange(T)).astype(np.float64)
    R = np.exp(-float(k) * dt)
    if norm_mode == "max":
        return R / R.max()
    if norm_mode == "sum":
        return R / R.sum()
    raise ValueError(norm_mode)


def normalise_attention(W: np.ndarray, norm_mode: str = "max") -> np.ndarray:
    """A_i = alpha * W_i of Eq. 2; alpha per layer, DESIGN c2."""
    if norm_mode == "max":
        return W / W.max()
    if norm_mode == "sum":
        return W / W.sum()
    raise ValueError(norm_mode)


def raw_scores(cfg: OracleConfig, W: np.ndarray, T: int) -> np.ndarray:
    """S^l_i for every layer: Eq. 1 (shallow), Eq. 2 (deep), Eq. 4 (middle),
    PAPER.md:80-101.  W: [L, T] (rows of shallow layers are ignored)."""
    R = recency_scores(T, cfg.forget_rate, cfg.norm_mode)
    S = np.zeros((cfg.n_layers, T), dtype=np.float64)
    for l in range(cfg.n_layers):
        w = omega_of_layer(cfg, l)
        if layer_stage(cfg, l) == "shallow":
            S[l] = R
        else:
            A = normalise_attention(W[l], cfg.norm_mode)
            S[l] = (1.0 - w) * A + w * R                      # Eq. 4
    return S


def smooth_scores(cfg: OracleConfig, S: np.ndarray) -> np.ndarray:
    """Eq. 5: S~^l = (1 - lam_l) S^l + lam_l S^{l+1}, on the same cache
    index i (DESIGN c10), with the RAW S^{l+1} (DESIGN c9); the last layer has no
    l+1 and keeps S^{L-1}."""
    L = S.shape[0]
    out = np.array(S, dtype=np.float64, copy=True)
    for l in range(L - 1):
        lam = lambda_of_layer(cfg, l)
        out[l] = (1.0 - lam) * S[l] + lam * S[l + 1]
    return out


def select_topk(s_tilde: np.ndarray, budget: int) -> np.ndarray:
    """I_l = TopK(S~_l, |M|), Eq. 6.  Ties keep the larger (more recent)
    index; the result is in ascending cache index, i.e. temporal order (DESIGN c6)."""
    T = s_tilde.shape[0]
    idx = np.arange(T)
    order = np.lexsort((-idx, -s_tilde))       # primary: score descending; then index descending
    return np.sort(order[:budget])


# --------------------------------------------------------------------------- positions
def compact_positions(cfg: OracleConfig, pos_kept: np.ndarray) -> np.ndarray:
    """Left-compaction of the retained positions.

    1D (Eq. 8): p_new = offset + rank_P(p_old), P = sorted retained positions.
    M-RoPE (Eq. 11): the same per axis, rank within the sorted SET of
    retained coordinates of that axis; axes not in
    `mrope_compact_axes` keep their coordinate (DESIGN c13).
    pos_kept: [A, n] -> [A, n]."""
    A, _ = pos_kept.shape
    out = np.array(pos_kept, dtype=np.int64, copy=True)
    for a in range(A):
        if A == 3 and not (cfg.mrope_compact_axes >> a) & 1:
            continue
        distinct = np.unique(pos_kept[a])                     # sorted set P^(d)
        out[a] = cfg.pos_offset + np.searchsorted(distinct, pos_kept[a])
    return out


def rope_frequencies(head_dim: int, theta: float) -> np.ndarray:
    """theta_j = base^(-2j/d), j = 0..d/2-1, in fp64 (DESIGN c11)."""
    j = np.arange(head_dim // 2, dtype=np.float64)
    return np.power(float(theta), -2.0 * j / float(head_dim))


def pair_axis(cfg: OracleConfig) -> np.ndarray:
    """Axis that owns rotary pair j: 1D -> 0; M-RoPE -> t for j < s_t, h for the next
    s_h pairs, w for the rest (DESIGN c12)."""
    half = cfg.head_dim // 2
    if cfg.rope_mode == "1d":
        return np.zeros(half, dtype=np.int64)
    s_t, s_h, s_w = cfg.mrope_section
    assert s_t + s_h + s_w == half
    return np.concatenate([np.full(s_t, 0), np.full(s_h, 1), np.full(s_w, 2)]).astype(np.int64)


def round_to_storage(x: np.ndarray, dtype: str) -> np.ndarray:
    """Round an fp32 array to the storage dtype, round-to-nearest-even (DESIGN c14)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    if dtype == "f32":
        return x
    if dtype == "bf16":
        u = x.view(np.uint32)
        bias = np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))
        return ((u + bias) & np.uint32(0xFFFF0000)).view(np.float32)
    raise ValueError(dtype)


def rotary_delta(cfg: OracleConfig, k_old: np.ndarray, delta: np.ndarray) -> np.ndarray:
    """k_new = k_old (.) e^{i (p_new - p_old) theta}, Eq. 9-10 and, per
    channel section, Eq. 12-13.

    k_old: [n, H_kv, d] fp32 holding storage-dtype values; delta: [A, n] = p_new - p_old.
    Pairs are (j, j + d/2) with z = x_j + i x_{j+d/2} (DESIGN c11).  Angle in fp64,
    cos/sin rounded to fp32, rotation in fp32 without fused multiply-add, result
    rounded to the storage dtype; a pair whose delta is 0 is copied bit for bit
    (DESIGN c14)."""
    n, _, d = k_old.shape
    half = d // 2
    theta = rope_frequencies(d, cfg.rope_theta)                     # [half] fp64
    axis = pair_axis(cfg)                                           # [half]
    dl = delta[axis, :].T.astype(np.float64)                        # [n, half]
    ang = dl * theta[None, :]
    c = np.cos(ang).astype(np.float32)[:, None, :]                  # [n, 1, half]
    s = np.sin(ang).astype(np.float32)[:, None, :]
    x = k_old[:, :, :half].astype(np.float32)
    y = k_old[:, :, half:].astype(np.float32)
    xc = x * c
    ys = y * s
    xs = x * s
    yc = y * c
    x_new = (xc - ys).astype(np.float32)
    y_new = (xs + yc).astype(np.float32)
    out = np.concatenate([x_new, y_new], axis=2)
    out = round_to_storage(out, cfg.dtype)
    zero = (dl == 0.0)[:, None, :]                                  # bit-exact copy when delta = 0
    zero2 = np.concatenate([zero, zero], axis=2)
    return np.where(zero2, k_old, out).astype(np.float32)


def summary_token(cfg: OracleConfig, K_p: np.ndarray, V_p: np.ndarray, P_p: np.ndarray, t: int):
    """Algorithm 1: one (k_sum, v_sum) from the pruned tokens of a layer.

    K_p, V_p: [n, H_kv, d] pruned keys / values (storage values); P_p: [1, n] their position indices;
    t: target position of the summary token.  Step 1: v_sum = Mean(V_p).  Step 2: every pruned key is
    phase-aligned to t by the rotary delta t - p (Eq. 9-10, fp64 angle, fp32 cos / sin and rotation as in
    `rotary_delta`, NOT rounded to storage), then k_sum = Mean(K_aligned).  Means are taken in fp64 and
    rounded once to the storage dtype (DESIGN f1).  1D RoPE only."""
    n, _, d = K_p.shape
    half = d // 2
    theta = rope_frequencies(d, cfg.rope_theta)
    ang = (float(t) - P_p[0].astype(np.float64))[:, None] * theta[None, :]     # [n, half]
    c = np.cos(ang).astype(np.float32)[:, None, :]
    s_ = np.sin(ang).astype(np.float32)[:, None, :]
    x = K_p[:, :, :half].astype(np.float32)
    y = K_p[:, :, half:].astype(np.float32)
    xa = ((x * c).astype(np.float32) - (y * s_).astype(np.float32)).astype(np.float32)
    ya = ((x * s_).astype(np.float32) + (y * c).astype(np.float32)).astype(np.float32)
    K_aligned = np.concatenate([xa, ya], axis=2).astype(np.float64)
    k_sum = round_to_storage(K_aligned.mean(axis=0).astype(np.float32), cfg.dtype)
    v_sum = round_to_storage(V_p.astype(np.float64).mean(axis=0).astype(np.float32), cfg.dtype)
    return k_sum, v_sum


# --------------------------------------------------------------------------- layer-dependent budgets (f4)
def layer_budgets(cfg: OracleConfig) -> np.ndarray:
    """Per-layer budgets m_i: with the total budget |M| = budget * L fixed,
    m_i = floor(w_i / sum_j w_j * |M|), and the rounding residue |M| - sum_i m_i goes to the last layer.
    w_i is the weight of layer i's stage (Tab. 5 gives one weight per stage).  The weights cross the C ABI
    as single-precision numbers, so they are rounded to fp32 first; the quotient is taken in fp64."""
    L = cfg.n_layers
    w3 = [float(np.float32(x)) for x in cfg.budget_weights]
    if min(w3) <= 0.0:
        raise ValueError("budget weights must be positive")
    stage_w = {"shallow": w3[0], "middle": w3[1], "deep": w3[2]}
    w = np.array([stage_w[layer_stage(cfg, l)] for l in range(L)], np.float64)
    total = cfg.budget * L
    wsum = 0.0
    for x in w:                                           # plain left-to-right fp64 sum (the host code does the same)
        wsum += float(x)
    m = np.array([int(np.floor(float(x) / wsum * float(total))) for x in w], np.int64)
    m[L - 1] += total - int(m.sum())
    return m


def smooth_scores_aligned(cfg: OracleConfig, S: list) -> list:
    """Eq. 5 when layers hold different numbers of candidates (DESIGN f4): the caches are aligned at
    their NEWEST token -- candidate i of layer l (T_l candidates) meets candidate i - T_l + T_{l+1} of layer l+1, the
    one at the same distance from the newest token, which both layers received together.  A candidate of layer l that
    is older than everything layer l+1 holds has no counterpart and keeps its raw score.  With equal T this is
    `smooth_scores`."""
    L = len(S)
    out = [np.array(x, dtype=np.float64, copy=True) for x in S]
    for l in range(L - 1):
        lam = lambda_of_layer(cfg, l)
        T0, T1 = len(S[l]), len(S[l + 1])
        i = np.arange(T0)
        j = i - T0 + T1
        has = j >= 0
        out[l][has] = (1.0 - lam) * S[l][has] + lam * S[l + 1][j[has]]
    return out


# --------------------------------------------------------------------------- state + step
@dataclass
class OracleStream:
    """One stream's cache: K, V [L, cap, H_kv, d] (fp32 holding storage values),
    pos [L, A, cap] int64, `len` valid tokens per layer (identical across layers)."""
    cfg: OracleConfig
    K: Optional[np.ndarray] = None
    V: Optional[np.ndarray] = None
    pos: Optional[np.ndarray] = None
    len: int = 0
    lens: Optional[np.ndarray] = None # layer-dependent budgets (DESIGN f4): valid tokens per layer; `len` is then their max
    t_steps_seen: int = 0             # M-RoPE: temporal steps appended so far
    next_pos: int = -1                # lazy mode: position (1D) / temporal index (M-RoPE) after the newest token
    last: dict = field(default_factory=dict)

    def _ensure(self, need: int):
        c = self.cfg
        cap = max(need, c.capacity)
        if self.K is None:
            shape = (c.n_layers, cap, c.n_kv_heads, c.head_dim)
            self.K = np.zeros(shape, np.float32)
            self.V = np.zeros(shape, np.float32)
            self.pos = np.zeros((c.n_layers, c.n_axes, cap), np.int64)
        elif self.K.shape[1] < cap:
            grow = cap - self.K.shape[1]
            self.K = np.pad(self.K, ((0, 0), (0, grow), (0, 0), (0, 0)))
            self.V = np.pad(self.V, ((0, 0), (0, grow), (0, 0), (0, 0)))
            self.pos = np.pad(self.pos, ((0, 0), (0, 0), (0, grow)))


def arrival_positions(cfg: OracleConfig, st: OracleStream, n_new: int, pos_start: int) -> np.ndarray:
    """Positions the arriving chunk was rotated at, identical for all layers -> [A, n_new].

    1D: pos_start + j, default pos_start = offset + len (the slot after the compacted
    cache).  M-RoPE: token j of the chunk sits at temporal step
    j // (gh*gw) of the chunk and at (row, col) of the gh x gw merged patch grid;
    default first step = offset + min(steps seen, |M|), which is host-computable and
    above every compacted t of every layer (DESIGN c13/c16)."""
    j = np.arange(n_new, dtype=np.int64)
    lazy = cfg.reindex_mode == "lazy"
    nxt = st.next_pos if st.next_pos >= 0 else cfg.pos_offset       # lazy: positions keep growing
    if cfg.rope_mode == "1d":
        p0 = pos_start if pos_start >= 0 else (nxt if lazy else cfg.pos_offset + st.len)
        return (p0 + j)[None, :]
    tpt = cfg.mrope_grid_h * cfg.mrope_grid_w
    t0 = pos_start if pos_start >= 0 else (nxt if lazy else cfg.pos_offset + min(st.t_steps_seen, cfg.budget))
    t = t0 + j // tpt
    h = cfg.pos_offset + (j % tpt) // cfg.mrope_grid_w
    w = cfg.pos_offset + j % cfg.mrope_grid_w
    return np.stack([t, h, w])


def lazy_reindex_due(cfg: OracleConfig, p_end: int) -> bool:
    """Lazy re-indexing: re-index "only when positional indices approach the model limit".
    Reading (DESIGN f2): the compression step re-indexes when the NEXT chunk (at most `max_chunk_span`
    positions) would no longer fit below `max_position`, p_end being the position after the newest token."""
    return p_end + cfg.max_chunk_span > cfg.max_position


def oracle_step(st: OracleStream, K_new: np.ndarray, V_new: np.ndarray,
                Q_probe: Optional[np.ndarray], pos_start: int = -1) -> dict:
    """One chunk arrival (Fig. 3 at :61).

    K_new, V_new: [L, n_new, H_kv, d] post-RoPE keys / values of the chunk;
    Q_probe: [L, H_q, P, d] query states of the guidance prompt, or None.
    Steps: append -> (if T > |M| and a probe is given) W (Eq. 2) -> S (Eq. 1-4) ->
    S~ (Eq. 5) -> TopK + gather (Eq. 6) -> positions (Eq. 8/11) -> rotary correction
    (Eq. 9-10 / 12-13).  Returns the intermediate quantities for parity checks."""
    cfg = st.cfg
    L, n_new = K_new.shape[0], K_new.shape[1]
    T = st.len + n_new
    st._ensure(T)

    # 1. append: the chunk is prefilled first, compression sees all T tokens (DESIGN c5)
    p_arr = arrival_positions(cfg, st, n_new, pos_start)
    st.K[:, st.len:T] = K_new
    st.V[:, st.len:T] = V_new
    st.pos[:, :, st.len:T] = p_arr[None, :, :]
    span = n_new
    if cfg.rope_mode == "m3d":
        tpt = cfg.mrope_grid_h * cfg.mrope_grid_w
        span = (n_new + tpt - 1) // tpt
        st.t_steps_seen += span
    p_end = int(p_arr[0, 0]) + span                    # position after the newest token (t axis for M-RoPE)
    st.next_pos = p_end
    if Q_probe is None or T <= cfg.budget:        # "triggered once the budget is exceeded"
        st.len = T
        st.last = {"T": T, "evicted": False}
        return st.last

    # 2. attention weights of the pseudo-query (Eq. 2); shallow layers need none
    scale = cfg.softmax_scale if cfg.softmax_scale > 0 else 1.0 / np.sqrt(float(cfg.head_dim))
    W = np.zeros((L, T), np.float64)
    for l in range(L):
        if layer_stage(cfg, l) != "shallow":
            # hybrid guidance (App. B): the probe rows are [local prompt | global prompt]; middle
            # layers use all of them, deep layers only the global part (DESIGN f3)
            pb = cfg.probe_deep_begin if layer_stage(cfg, l) == "deep" else 0
            W[l] = attention_weights(Q_probe[l][:, pb:], st.K[l, :T], cfg.group, scale)

    # 3-4. normalise, recency, layer weighting (Eq. 1-4); 5. smoothing (Eq. 5)
    S = raw_scores(cfg, W, T)
    S_tilde = smooth_scores(cfg, S)

    # 6. per-layer Top-K (Eq. 6); 7. positions (Eq. 8 / 11); 8. gather + rotary correction
    kept = np.zeros((L, cfg.budget), np.int64)
    pos_new = np.zeros((L, cfg.n_axes, cfg.budget), np.int64)
    K_out = np.zeros((L, cfg.budget) + st.K.shape[2:], np.float32)
    V_out = np.zeros_like(K_out)
    if cfg.summary_token and cfg.rope_mode != "1d":
        raise ValueError("summary tokens are defined here for 1D RoPE only: Alg. 1 takes ONE target index t (DESIGN f1)")
    # a summary token takes a position of its own: under lazy re-indexing the position after the newest token
    # (DESIGN f1/f2), so the running position counter -- and with it the re-index trigger -- advances by one more
    summ_pos = 1 if (cfg.summary_token and stage_split(cfg.n_layers, cfg.n_shallow, cfg.n_deep)[2] > 0) else 0
    reindex = cfg.reindex_mode == "eager" or lazy_reindex_due(cfg, p_end + summ_pos)
    for l in range(L):
        if cfg.summary_token and layer_stage(cfg, l) == "deep":
            # deep layers keep |M| - 1 tokens by Top-K and append ONE summary token of everything evicted, so the
            # layer still holds exactly |M| tokens; it sits after the kept tokens
            # (Alg. 1 step 3) and is an ordinary, evictable token from then on (DESIGN f1).  kept[l][-1] = -1 marks
            # it.  Its position t: at a re-index step the next contiguous one, offset + |M| - 1; between re-index
            # steps of the lazy mode the kept tokens keep their original indices and t is the position after the
            # newest token, p_end (PAPER.md:126-128 with Alg. 1 step 3: positions stay strictly increasing).
            I = select_topk(S_tilde[l], cfg.budget - 1)
            ev = np.setdiff1d(np.arange(T), I)
            p_old = st.pos[l][:, I]
            p_new = compact_positions(cfg, p_old) if reindex else p_old
            t = cfg.pos_offset + cfg.budget - 1 if reindex else p_end
            k_sum, v_sum = summary_token(cfg, st.K[l, ev], st.V[l, ev], st.pos[l][:, ev], t)
            kept[l, :-1], kept[l, -1] = I, -1
            pos_new[l][:, :-1], pos_new[l][:, -1] = p_new, t
            V_out[l, :-1], V_out[l, -1] = st.V[l, I], v_sum
            K_out[l, :-1], K_out[l, -1] = rotary_delta(cfg, st.K[l, I], p_new - p_old), k_sum
            continue
        I = select_topk(S_tilde[l], cfg.budget)
        p_old = st.pos[l][:, I]
        p_new = compact_positions(cfg, p_old) if reindex else p_old   # lazy: keep the original indices
        kept[l], pos_new[l] = I, p_new
        V_out[l] = st.V[l, I]                                  # V_l[I_l], bit for bit
        K_out[l] = rotary_delta(cfg, st.K[l, I], p_new - p_old)
    st.K[:, :cfg.budget] = K_out
    st.V[:, :cfg.budget] = V_out
    st.pos[:, :, :cfg.budget] = pos_new
    st.len = cfg.budget                                        # 9.
    if reindex:                       # every position is now below offset + |M| (M-RoPE: + min(steps seen, |M|))
        st.next_pos = cfg.pos_offset + (cfg.budget if cfg.rope_mode == "1d" else min(st.t_steps_seen, cfg.budget))
    else:
        st.next_pos = p_end + summ_pos
    st.last = {"T": T, "evicted": True, "reindexed": reindex, "W": W, "S": S, "S_tilde": S_tilde,
               "kept": kept, "pos_new": pos_new}
    return st.last


def oracle_step_layer_budgets(st: OracleStream, K_new: np.ndarray, V_new: np.ndarray,
                              Q_probe: Optional[np.ndarray], pos_start: int = -1) -> dict:
    """One chunk arrival with layer-dependent budgets (Tab. 5; DESIGN f4).

    Every layer l has its own budget m_l (`layer_budgets`) and its own length len_l; it compresses -- Eq. 1-6, 8-10 as
    in `oracle_step` -- only at an arrival that takes IT over its budget, and is left untouched (appended
    to, not re-indexed) otherwise.  Arrival positions are shared by all layers and lie above every cached position:
    1D default offset + max_l len_l.  Scores of layer l are taken over its own T_l = len_l + n_new candidates, the
    recency term counts the distance from ITS newest token, and Eq. 5 pairs candidates at equal distance from the
    newest token (`smooth_scores_aligned`).  1D RoPE.  With equal weights this is `oracle_step`.

    Summary tokens (Alg. 1; DESIGN f1 x f4): a DEEP layer that compresses at this arrival keeps m_l - 1 tokens by Top-K and
    appends one summary token of everything it evicts in slot m_l - 1, exactly as in `oracle_step` with m_l for |M|: target
    position offset + m_l - 1 at a step that re-indexes, the position after the newest token otherwise (the running
    position counter then advances by one more -- once, whatever the number of deep layers that made one).  A deep layer
    still under its budget makes none."""
    cfg = st.cfg
    if cfg.rope_mode != "1d":
        raise ValueError("layer-dependent budgets are defined here for 1D RoPE (DESIGN f4)")
    L, n_new = K_new.shape[0], K_new.shape[1]
    m = layer_budgets(cfg)
    if st.lens is None:
        st.lens = np.zeros(L, np.int64)
    lens = st.lens
    T = lens + n_new
    st.len = int(lens.max())
    st._ensure(int(T.max()))
    p_arr = arrival_positions(cfg, st, n_new, pos_start)
    for l in range(L):
        st.K[l, lens[l]:T[l]] = K_new[l]
        st.V[l, lens[l]:T[l]] = V_new[l]
        st.pos[l, :, lens[l]:T[l]] = p_arr
    p_end = int(p_arr[0, 0]) + n_new
    st.next_pos = p_end
    over = T > m
    if Q_probe is None or not over.any():
        st.lens = T
        st.len = int(T.max())
        st.last = {"T": T.copy(), "evicted": False}
        return st.last
    scale = cfg.softmax_scale if cfg.softmax_scale > 0 else 1.0 / np.sqrt(float(cfg.head_dim))
    S = []
    for l in range(L):
        R = recency_scores(int(T[l]), cfg.forget_rate, cfg.norm_mode)
        if layer_stage(cfg, l) == "shallow":
            S.append(R)
            continue
        pb = cfg.probe_deep_begin if layer_stage(cfg, l) == "deep" else 0
        W = attention_weights(Q_probe[l][:, pb:], st.K[l, :T[l]], cfg.group, scale)
        w = omega_of_layer(cfg, l)
        S.append((1.0 - w) * normalise_attention(W, cfg.norm_mode) + w * R)
    S_tilde = smooth_scores_aligned(cfg, S)
    summ = [bool(cfg.summary_token and layer_stage(cfg, l) == "deep" and over[l]) for l in range(L)]
    summ_pos = 1 if any(summ) else 0
    reindex = cfg.reindex_mode == "eager" or lazy_reindex_due(cfg, p_end + summ_pos)
    kept, pos_new = [], []
    new_lens = T.copy()
    for l in range(L):
        if not over[l]:                                   # under its budget: nothing happens to this layer
            kept.append(np.arange(T[l])); pos_new.append(st.pos[l][:, :T[l]].copy())
            continue
        if summ[l]:
            n_keep = int(m[l]) - 1
            I = select_topk(S_tilde[l], n_keep)
            ev = np.setdiff1d(np.arange(T[l]), I)
            p_old = st.pos[l][:, I]
            p_new = compact_positions(cfg, p_old) if reindex else p_old
            t = cfg.pos_offset + n_keep if reindex else p_end
            k_sum, v_sum = summary_token(cfg, st.K[l, ev], st.V[l, ev], st.pos[l][:, ev], t)
            V_kept = st.V[l, I].copy()
            K_kept = rotary_delta(cfg, st.K[l, I], p_new - p_old)
            st.V[l, :n_keep], st.V[l, n_keep] = V_kept, v_sum
            st.K[l, :n_keep], st.K[l, n_keep] = K_kept, k_sum
            st.pos[l, :, :n_keep], st.pos[l, :, n_keep] = p_new, t
            kept.append(np.concatenate([I, [-1]])); pos_new.append(st.pos[l][:, :m[l]].copy())
            new_lens[l] = m[l]
            continue
        I = select_topk(S_tilde[l], int(m[l]))
        p_old = st.pos[l][:, I]
        p_new = compact_positions(cfg, p_old) if reindex else p_old
        st.V[l, :m[l]] = st.V[l, I]
        st.K[l, :m[l]] = rotary_delta(cfg, st.K[l, I], p_new - p_old)
        st.pos[l, :, :m[l]] = p_new
        kept.append(I); pos_new.append(p_new)
        new_lens[l] = m[l]
    st.lens = new_lens
    st.len = int(new_lens.max())
    if reindex:                                           # positions of the layers that compressed are below offset + m_l
        st.next_pos = max(cfg.pos_offset + int(new_lens.max()), p_end if (~over).any() else 0)
    else:
        st.next_pos = p_end + summ_pos
    st.last = {"T": T.copy(), "evicted": True, "evicted_layers": over.copy(), "reindexed": reindex, "S": S,
               "S_tilde": S_tilde, "kept": kept, "pos_new": pos_new, "budgets": m}
    return st.last
