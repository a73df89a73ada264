"""Thin ctypes binding over libhermes_b200.so (include/hermes.h).  Argument marshalling only:
every step of the update runs in the CUDA kernels behind the C ABI.  PyTorch supplies device
memory (the workspace, the caller's tensors) and the CUDA stream.  There is no CPU fallback: a
missing library or a missing GPU raises."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, fields

import torch

from . import build as _build

HERMES_OK, HERMES_EINVAL, HERMES_ECAPACITY, HERMES_ESTATE, HERMES_ECUDA, HERMES_ENOMEM = 0, -1, -2, -3, -4, -5
HERMES_F32, HERMES_BF16 = 0, 1
HERMES_ROPE_1D, HERMES_ROPE_M3D = 0, 1
HERMES_REINDEX_EAGER, HERMES_REINDEX_LAZY = 0, 1
HERMES_NORM_MAX, HERMES_NORM_SUM = 0, 1
HERMES_SCORE_AUTO, HERMES_SCORE_SIMT, HERMES_SCORE_TCGEN05 = 0, 1, 2
HERMES_K_NAMES = ("append", "score_stats", "score_combine", "score_colsum", "select", "gather", "summary")

EXPORTS = ("hermes_default_config", "hermes_workspace_bytes", "hermes_create", "hermes_append_chunk",
           "hermes_append_chunk_host", "hermes_get_cache", "hermes_len", "hermes_layer_len", "hermes_layer_budget", "hermes_layer_budgets", "hermes_device_status",
           "hermes_set_profiling", "hermes_get_profile", "hermes_last_score_path", "hermes_v_pending",
           "hermes_last_launch_count", "hermes_destroy", "hermes_last_error",
           "hermes_topk_noalloc", "hermes_topk_noalloc_setup", "hermes_topk_noalloc_max_tokens", "hermes_topk_noalloc_error")


class HermesConfig(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_layers", "n_q_heads", "n_kv_heads", "head_dim", "dtype",
                                         "n_streams", "tokens_per_frame", "budget", "max_chunk_tokens",
                                         "max_tokens", "max_probe_tokens", "n_shallow", "n_deep",
                                         "l_short", "l_long")] + \
               [("omega0", C.c_float), ("gamma", C.c_float), ("forget_rate", C.c_float),
                ("norm_mode", C.c_int32), ("lambda_shallow", C.c_float), ("lambda_middle", C.c_float),
                ("lambda_deep", C.c_float), ("softmax_scale", C.c_float), ("rope_mode", C.c_int32),
                ("rope_theta", C.c_float), ("mrope_section", C.c_int32 * 3),
                ("mrope_compact_axes", C.c_int32), ("mrope_grid_h", C.c_int32),
                ("mrope_grid_w", C.c_int32), ("pos_offset", C.c_int32), ("reindex_mode", C.c_int32),
                ("max_position", C.c_int32), ("probe_deep_begin", C.c_int32), ("summary_token", C.c_int32), ("budget_weight", C.c_float * 3), ("defer_v", C.c_int32), ("score_path", C.c_int32),
                ("device", C.c_int32)]


class HermesCacheView(C.Structure):
    _fields_ = [("k", C.c_void_p), ("v", C.c_void_p), ("pos", C.c_void_p), ("n_axes", C.c_int32),
                ("pos_stride", C.c_int32), ("len", C.c_int32), ("last_scores", C.c_void_p),
                ("last_kept", C.c_void_p), ("last_T", C.c_int32)]


class HermesError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"hermes error {code}: {msg}")
        self.code = code


_lib = None


def load_library(rebuild_if_stale: bool = True) -> C.CDLL:
    """dlopen the in-tree library (building it with nvcc first if the sources are newer)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if rebuild_if_stale and _build.needs_build() and os.path.exists("/usr/local/cuda/bin/nvcc"):
        _build.build()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2601_14724_b200.build` (no CPU fallback exists)")
    lib = C.CDLL(path)
    vp, i32 = C.c_void_p, C.c_int32
    lib.hermes_default_config.argtypes = [C.POINTER(HermesConfig)]
    lib.hermes_default_config.restype = None
    lib.hermes_workspace_bytes.argtypes = [C.POINTER(HermesConfig)]
    lib.hermes_workspace_bytes.restype = C.c_size_t
    lib.hermes_create.argtypes = [C.POINTER(HermesConfig), vp, C.c_size_t, C.POINTER(vp)]
    lib.hermes_append_chunk.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp]
    lib.hermes_append_chunk_host.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp]
    lib.hermes_get_cache.argtypes = [vp, i32, i32, C.POINTER(HermesCacheView)]
    lib.hermes_len.argtypes = [vp]
    lib.hermes_layer_len.argtypes = [vp, i32]
    lib.hermes_layer_budget.argtypes = [vp, i32]
    lib.hermes_layer_budgets.argtypes = [C.POINTER(HermesConfig), C.POINTER(i32), i32]
    lib.hermes_device_status.argtypes = [vp, C.POINTER(i32)]
    lib.hermes_set_profiling.argtypes = [vp, i32]
    lib.hermes_get_profile.argtypes = [vp, C.POINTER(C.c_float), i32]
    lib.hermes_last_score_path.argtypes = [vp]
    lib.hermes_last_launch_count.argtypes = [vp]
    lib.hermes_v_pending.argtypes = [vp]
    lib.hermes_destroy.argtypes = [vp]
    lib.hermes_destroy.restype = None
    lib.hermes_last_error.argtypes = [vp]
    lib.hermes_last_error.restype = C.c_char_p
    lib.hermes_topk_noalloc.argtypes = [vp, i32, i32, vp, vp]
    lib.hermes_topk_noalloc_setup.argtypes = []
    lib.hermes_topk_noalloc_max_tokens.argtypes = []
    lib.hermes_topk_noalloc_max_tokens.restype = i32
    lib.hermes_topk_noalloc_error.argtypes = []
    lib.hermes_topk_noalloc_error.restype = C.c_char_p
    _lib = lib
    return lib


def hermes_default_config(**kw) -> HermesConfig:
    """hermes_default_config() + keyword overrides (mrope_section takes a 3-tuple)."""
    cfg = HermesConfig()
    load_library().hermes_default_config(C.byref(cfg))
    for k, v in kw.items():
        if k == "mrope_section":
            cfg.mrope_section = (C.c_int32 * 3)(*v)
        elif k == "budget_weight":
            cfg.budget_weight = (C.c_float * 3)(*v)
        elif not hasattr(cfg, k):
            raise TypeError(f"hermes_config has no field {k!r}")
        else:
            setattr(cfg, k, v)
    return cfg


def hermes_layer_budgets(cfg: HermesConfig) -> list:
    """Per-layer budgets of a config (host-only; no device needed)."""
    out = (C.c_int32 * max(int(cfg.n_layers), 1))()
    n = load_library().hermes_layer_budgets(C.byref(cfg), out, len(out))
    if n < 0:
        raise HermesError(n, (load_library().hermes_last_error(None) or b"").decode())
    return list(out[:n])


def hermes_workspace_bytes(cfg: HermesConfig) -> int:
    return int(load_library().hermes_workspace_bytes(C.byref(cfg)))


@dataclass
class Handle:
    ptr: C.c_void_p
    cfg: HermesConfig
    workspace: torch.Tensor

    @property
    def torch_dtype(self):
        return torch.bfloat16 if self.cfg.dtype == HERMES_BF16 else torch.float32


def _check(h, rc: int):
    if rc != HERMES_OK:
        msg = load_library().hermes_last_error(h.ptr if h is not None else None)
        raise HermesError(rc, msg.decode() if msg else "")


def hermes_create(cfg: HermesConfig) -> Handle:
    """Allocates the workspace with torch on cfg.device and calls hermes_create()."""
    lib = load_library()
    nbytes = hermes_workspace_bytes(cfg)
    if nbytes == 0:
        out = C.c_void_p()
        rc = lib.hermes_create(C.byref(cfg), None, 0, C.byref(out))   # collects the validation message
        raise HermesError(rc, (lib.hermes_last_error(None) or b"invalid config").decode())
    if not torch.cuda.is_available():
        raise HermesError(HERMES_ECUDA, "no CUDA device: the HERMES update has no CPU fallback")
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=f"cuda:{cfg.device}")
    off = (-ws.data_ptr()) % 256
    ws = ws[off:off + nbytes]
    out = C.c_void_p()
    rc = lib.hermes_create(C.byref(cfg), C.c_void_p(ws.data_ptr()), nbytes, C.byref(out))
    if rc != HERMES_OK:
        raise HermesError(rc, (lib.hermes_last_error(None) or b"").decode())
    return Handle(out, cfg, ws)


def _dev_ptr(h: Handle, t, shape, what: str):
    if t is None:
        return None
    if not (t.is_cuda and t.device.index == h.cfg.device):
        raise ValueError(f"{what} must live on cuda:{h.cfg.device}")
    if t.dtype != h.torch_dtype or tuple(t.shape) != tuple(shape) or not t.is_contiguous():
        raise ValueError(f"{what} must be contiguous {h.torch_dtype} of shape {tuple(shape)}, got {t.dtype} {tuple(t.shape)}")
    return C.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def hermes_append_chunk(h: Handle, K_new, V_new, Q_probe=None, pos_start: int = -1, stream=None):
    """K_new, V_new: [B, L, n_new, H_kv, d]; Q_probe: [B, L, H_q, P, d] or None (device tensors)."""
    c = h.cfg
    n_new = int(K_new.shape[2])
    kv_shape = (c.n_streams, c.n_layers, n_new, c.n_kv_heads, c.head_dim)
    n_probe = int(Q_probe.shape[3]) if Q_probe is not None else 0
    q_shape = (c.n_streams, c.n_layers, c.n_q_heads, n_probe, c.head_dim)
    rc = load_library().hermes_append_chunk(
        h.ptr, _dev_ptr(h, K_new, kv_shape, "K_new"), _dev_ptr(h, V_new, kv_shape, "V_new"),
        _dev_ptr(h, Q_probe, q_shape, "Q_probe"), n_new, n_probe, pos_start, _stream_ptr(stream))
    _check(h, rc)


def _host_ptr(h: Handle, t, what: str):
    if t is None:
        return None
    if t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{what} must be a contiguous host tensor")
    return C.c_void_p(t.data_ptr())


def hermes_append_chunk_host(h: Handle, K_new, V_new, Q_probe=None, pos_start: int = -1,
                             kept_out=None, stream=None):
    """Same update from HOST tensors (pinned recommended); kept_out: int32 host [B, L, budget]."""
    n_new = int(K_new.shape[2])
    n_probe = int(Q_probe.shape[3]) if Q_probe is not None else 0
    for t, what in ((K_new, "K_new"), (V_new, "V_new"), (Q_probe, "Q_probe")):
        if t is not None and t.dtype != h.torch_dtype:
            raise ValueError(f"{what} must be {h.torch_dtype}")
    rc = load_library().hermes_append_chunk_host(
        h.ptr, _host_ptr(h, K_new, "K_new"), _host_ptr(h, V_new, "V_new"), _host_ptr(h, Q_probe, "Q_probe"),
        n_new, n_probe, pos_start, _host_ptr(h, kept_out, "kept_out"), _stream_ptr(stream))
    _check(h, rc)


def _view(h: Handle, ptr, nbytes: int, dtype, shape):
    off = ptr - h.workspace.data_ptr()
    return h.workspace[off:off + nbytes].view(dtype).view(*shape)


def hermes_get_cache(h: Handle, stream: int, layer: int) -> dict:
    """Zero-copy torch views of one (stream, layer) slab: k, v [len, H_kv, d]; pos [A, len];
    last_scores [last_T]; last_kept [budget].  Synchronise the stream before reading them."""
    v = HermesCacheView()
    _check(h, load_library().hermes_get_cache(h.ptr, stream, layer, C.byref(v)))
    c = h.cfg
    es = 2 if c.dtype == HERMES_BF16 else 4
    row = c.n_kv_heads * c.head_dim
    out = {"len": v.len, "last_T": v.last_T, "n_axes": v.n_axes}
    out["k"] = _view(h, v.k, v.len * row * es, h.torch_dtype, (v.len, c.n_kv_heads, c.head_dim))
    out["v"] = _view(h, v.v, v.len * row * es, h.torch_dtype, (v.len, c.n_kv_heads, c.head_dim))
    pos = _view(h, v.pos, v.n_axes * v.pos_stride * 4, torch.int32, (v.n_axes, v.pos_stride))
    out["pos"] = pos[:, :v.len]
    if v.last_T:
        out["last_scores"] = _view(h, v.last_scores, v.last_T * 4, torch.float32, (v.last_T,))
        out["last_kept"] = _view(h, v.last_kept, v.len * 4, torch.int32, (v.len,))
    return out


def hermes_len(h: Handle) -> int:
    return int(load_library().hermes_len(h.ptr))


def hermes_layer_len(h: Handle, layer: int) -> int:
    return int(load_library().hermes_layer_len(h.ptr, layer))


def hermes_layer_budget(h: Handle, layer: int) -> int:
    return int(load_library().hermes_layer_budget(h.ptr, layer))


def hermes_device_status(h: Handle) -> int:
    s = C.c_int32()
    _check(h, load_library().hermes_device_status(h.ptr, C.byref(s)))
    return s.value


def hermes_set_profiling(h: Handle, enable: bool):
    _check(h, load_library().hermes_set_profiling(h.ptr, int(enable)))


def hermes_get_profile(h: Handle) -> dict:
    buf = (C.c_float * len(HERMES_K_NAMES))()
    n = load_library().hermes_get_profile(h.ptr, buf, len(HERMES_K_NAMES))
    if n < 0:
        _check(h, n)
    return {HERMES_K_NAMES[i]: float(buf[i]) for i in range(n)}


def hermes_last_score_path(h: Handle) -> int:
    return int(load_library().hermes_last_score_path(h.ptr))


def hermes_v_pending(h: Handle) -> int:
    return int(load_library().hermes_v_pending(h.ptr))


def hermes_last_launch_count(h: Handle) -> int:
    return int(load_library().hermes_last_launch_count(h.ptr))


def hermes_destroy(h: Handle):
    if h.ptr:
        load_library().hermes_destroy(h.ptr)
        h.ptr = None
        h.workspace = None


# ---- allocation-free Top-K (csrc/hermes_noalloc.cu): no handle, no workspace, scratch in a static device array ----
def hermes_topk_noalloc_max_tokens() -> int:
    return int(load_library().hermes_topk_noalloc_max_tokens())


def _noalloc_check(rc: int):
    if rc != HERMES_OK:
        msg = load_library().hermes_topk_noalloc_error()
        raise HermesError(rc, msg.decode() if msg else "")


def hermes_topk_noalloc_setup():
    """Resolves the static scratch address on the current CUDA device (do this before graph capture)."""
    _noalloc_check(load_library().hermes_topk_noalloc_setup())


def hermes_topk_noalloc(scores, k: int, kept_out, stream=None):
    """scores: contiguous fp32 device tensor [T]; kept_out: contiguous int32 device tensor [k] (caller-allocated).
    Enqueues one kernel on `stream` of the CURRENT device; nothing is allocated.  The pointers are passed as they are:
    the C entry point validates sizes (T > hermes_topk_noalloc_max_tokens() -> HERMES_ECAPACITY)."""
    if scores.dtype != torch.float32 or not scores.is_cuda or not scores.is_contiguous() or scores.dim() != 1:
        raise ValueError("scores must be a contiguous 1-D fp32 CUDA tensor")
    if kept_out.dtype != torch.int32 or not kept_out.is_cuda or not kept_out.is_contiguous() or kept_out.numel() < max(k, 0):
        raise ValueError("kept_out must be a contiguous int32 CUDA tensor with at least k elements")
    rc = load_library().hermes_topk_noalloc(C.c_void_p(scores.data_ptr()), int(scores.numel()), int(k),
                                            C.c_void_p(kept_out.data_ptr()), _stream_ptr(stream))
    _noalloc_check(rc)
