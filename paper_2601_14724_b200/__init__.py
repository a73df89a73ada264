"""B200-native HERMES per-chunk hierarchical KV-cache update (arXiv 2601.14724).

C-ABI library (include/hermes.h, csrc/) + this thin binding.  sm_100a only, no CPU fallback."""
from .binding import *  # noqa: F401,F403
from .binding import (HERMES_BF16, HERMES_F32, HERMES_ROPE_1D, HERMES_ROPE_M3D, hermes_default_config)


def config_for_workload(wl, device: int = 0, **over):
    """hermes_config for a workload description (any object with the fields of workloads.Workload)."""
    kw = dict(n_layers=wl.n_layers, n_q_heads=wl.n_q_heads, n_kv_heads=wl.n_kv_heads, head_dim=wl.head_dim,
              dtype=HERMES_BF16 if wl.dtype == "bf16" else HERMES_F32, n_streams=wl.n_streams,
              tokens_per_frame=wl.tokens_per_frame, budget=wl.budget, max_chunk_tokens=wl.chunk_tokens,
              max_tokens=wl.cap, max_probe_tokens=wl.probe_tokens, forget_rate=wl.k_forget,
              rope_mode=HERMES_ROPE_M3D if wl.rope_mode == "m3d" else HERMES_ROPE_1D,
              rope_theta=wl.rope_theta, mrope_section=tuple(wl.mrope_section),
              mrope_compact_axes=wl.mrope_compact_axes, mrope_grid_h=wl.mrope_grid_h,
              mrope_grid_w=wl.mrope_grid_w, pos_offset=wl.pos_offset, device=device)
    kw.update(over)
    return hermes_default_config(**kw)
