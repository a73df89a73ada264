"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/hermes.h
declares, validates configs, sizes workspaces, and fails loudly without a GPU (no compute calls)."""
import ctypes as C
import os
import re

import pytest
import torch

import paper_2601_14724_b200 as hb
from workloads import CONFIGS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    lib = hb.load_library()
    header = open(os.path.join(ROOT, "include", "hermes.h")).read()
    declared = set(re.findall(r"\b(hermes_[a-z_]+)\s*\(", header))
    declared -= {"hermes_append_chunk_"}
    assert declared == set(hb.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_config_struct_matches_header_size():
    # 15 int32 + 3 float + int32 + 4 float + int32 + float + 3 int32 + 8 int32 + 3 float + 3 int32 = 42 x 4 bytes
    assert C.sizeof(hb.HermesConfig) == 42 * 4
    assert list(hb.hermes_default_config().budget_weight) == [1.0, 1.0, 1.0]
    assert hb.hermes_default_config().reindex_mode == 0
    cfg = hb.hermes_default_config()
    assert (cfg.omega0, cfg.gamma) == (0.75, pytest.approx(0.6))
    assert (cfg.lambda_shallow, cfg.lambda_middle, cfg.lambda_deep) == (pytest.approx(0.1), pytest.approx(0.3), pytest.approx(0.4))
    assert list(cfg.mrope_section) == [16, 24, 24]


def test_workspace_bytes_accounts_for_double_buffered_cache():
    wl = CONFIGS["llava_ov_7b"]
    cfg = hb.config_for_workload(wl)
    n = hb.hermes_workspace_bytes(cfg)
    kv = 2 * 2 * wl.n_layers * wl.cap * wl.n_kv_heads * wl.head_dim * 2      # K+V, two buffers, bf16
    assert kv < n < kv * 1.5
    big = hb.config_for_workload(CONFIGS["batched_72b"])
    assert hb.hermes_workspace_bytes(big) < 120e9                              # fits one B200 (180 GB)


@pytest.mark.parametrize("field,value", [("n_kv_heads", 3), ("head_dim", 100), ("budget", 0), ("forget_rate", 0.0),
                                         ("n_shallow", 20), ("lambda_deep", 1.5), ("mrope_section", (16, 24, 20)),
                                         ("dtype", 7), ("max_tokens", 10)])
def test_invalid_configs_are_rejected(field, value):
    over = {field: value}
    if field == "mrope_section":
        over["rope_mode"] = hb.HERMES_ROPE_M3D
    if field == "n_shallow":
        over["n_deep"] = 20
    cfg = hb.config_for_workload(CONFIGS["llava_ov_7b"], **over)
    assert hb.hermes_workspace_bytes(cfg) == 0
    out = C.c_void_p()
    rc = hb.load_library().hermes_create(C.byref(cfg), None, 0, C.byref(out))
    assert rc == hb.HERMES_EINVAL and not out.value
    assert hb.load_library().hermes_last_error(None)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_lazy_reindex_needs_room_below_max_position():
    wl = CONFIGS["llava_ov_7b"]
    bad = hb.config_for_workload(wl, reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=wl.budget + wl.chunk_tokens)
    assert hb.hermes_workspace_bytes(bad) == 0
    ok = hb.config_for_workload(wl, reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=32768)
    assert hb.hermes_workspace_bytes(ok) > hb.hermes_workspace_bytes(hb.config_for_workload(wl))   # larger rotary table


def test_create_without_gpu_fails_loudly():
    cfg = hb.config_for_workload(CONFIGS["toy"])
    with pytest.raises(hb.HermesError) as e:
        hb.hermes_create(cfg)
    assert e.value.code == hb.HERMES_ECUDA
    buf = C.create_string_buffer(hb.hermes_workspace_bytes(cfg) + 512)
    addr = (C.addressof(buf) + 255) // 256 * 256
    out = C.c_void_p()
    rc = hb.load_library().hermes_create(C.byref(cfg), C.c_void_p(addr), hb.hermes_workspace_bytes(cfg), C.byref(out))
    assert rc == hb.HERMES_ECUDA and b"no CPU fallback" in hb.load_library().hermes_last_error(None)


def test_null_handle_calls_do_not_crash():
    lib = hb.load_library()
    assert lib.hermes_append_chunk(None, None, None, None, 1, 0, -1, None) == hb.HERMES_EINVAL
    assert lib.hermes_len(None) == 0
    lib.hermes_destroy(None)


def test_layer_dependent_budget_configs():
    wl = CONFIGS["llava_ov_7b"]
    assert hb.hermes_workspace_bytes(hb.config_for_workload(wl, budget_weight=(1.3, 1.0, 0.7))) == 0   # max_tokens < largest layer
    ok = hb.config_for_workload(wl, budget_weight=(1.3, 1.0, 0.7), max_tokens=0)
    assert hb.hermes_workspace_bytes(ok) > hb.hermes_workspace_bytes(hb.config_for_workload(wl))   # slabs sized for the largest layer
    for bad in (dict(budget_weight=(1.3, 1.0, 0.0)),
                dict(budget_weight=(0.7, 1.0, 1.3), rope_mode=hb.HERMES_ROPE_M3D)):
        assert hb.hermes_workspace_bytes(hb.config_for_workload(wl, max_tokens=0, **bad)) == 0
    assert hb.hermes_workspace_bytes(hb.config_for_workload(wl, max_tokens=0, budget_weight=(1.3, 1.0, 0.7), summary_token=1)) > 0
    # both scoring paths take per-layer candidate counts
    assert hb.hermes_workspace_bytes(hb.config_for_workload(wl, max_tokens=0, budget_weight=(1.3, 1.0, 0.7), score_path=hb.HERMES_SCORE_TCGEN05)) > 0


@pytest.mark.parametrize("w", [(1.0, 1.0, 1.0), (1.3, 1.0, 0.7), (0.7, 1.6, 0.7), (0.7, 1.0, 1.3), (0.31, 2.7, 1.9)])
@pytest.mark.parametrize("L,budget", [(4, 96), (28, 6000), (28, 6272), (80, 4096), (7, 785), (33, 1001)])
def test_host_layer_budgets_equal_the_oracle(L, budget, w):
    """The library's host-side allocation against oracle.layer_budgets for the Tab. 5 weightings and an
    awkward one: same fp32 weights, same fp64 quotient, same residue rule on both sides."""
    from oracle import hermes_oracle as ho
    wl = CONFIGS["llava_ov_7b"].scaled(n_layers=L, budget=budget)
    got = hb.hermes_layer_budgets(hb.config_for_workload(wl, budget_weight=w, max_tokens=0))
    ocfg = ho.OracleConfig(n_layers=L, n_q_heads=28, n_kv_heads=4, head_dim=128, budget=budget, forget_rate=0.1, budget_weights=w)
    assert got == ho.layer_budgets(ocfg).tolist() and sum(got) == budget * L
