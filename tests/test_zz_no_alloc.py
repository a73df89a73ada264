"""hermes_topk_noalloc (include/hermes.h, csrc/hermes_noalloc.cu): the allocation-free Top-K entry point, whose scratch
is a static device array, against the update path's own selection (hermes_cache_view.last_scores -> last_kept).

Index work: the comparison is bit-exact, like every kept-list comparison in tests/test_gpu_parity.py.
Named test_zz_* so that pytest collects it last: `pytest -x` then never hides another test behind a failure here."""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_2601_14724_b200 as hb
from workloads import CONFIGS


def _expected_topk(scores: np.ndarray, k: int) -> np.ndarray:
    """Eq. 6 written out: total order (score, index), the T - k smallest leave, survivors in ascending index order."""
    order = np.lexsort((np.arange(scores.size), scores))           # by score, ties by index
    return np.sort(order[scores.size - k:]).astype(np.int32)


def test_noalloc_rejects_bad_sizes_without_touching_cuda():
    lib = hb.load_library()
    mx = hb.hermes_topk_noalloc_max_tokens()
    assert mx == 65536
    fake = C.c_void_p(0x1000)                                       # never dereferenced: sizes are checked first
    assert lib.hermes_topk_noalloc(fake, mx + 1, 1, fake, None) == hb.HERMES_ECAPACITY
    msg = lib.hermes_topk_noalloc_error().decode()
    assert "65536" in msg and "exceeds" in msg, msg
    assert lib.hermes_topk_noalloc(fake, 10, 0, fake, None) == hb.HERMES_EINVAL
    assert lib.hermes_topk_noalloc(fake, 10, 11, fake, None) == hb.HERMES_EINVAL
    assert lib.hermes_topk_noalloc(fake, 0, 1, fake, None) == hb.HERMES_EINVAL
    assert lib.hermes_topk_noalloc(None, 10, 1, fake, None) == hb.HERMES_EINVAL
    assert lib.hermes_topk_noalloc(fake, 10, 1, None, None) == hb.HERMES_EINVAL


def _update_path_selection(wl):
    """Runs the existing path to its second eviction and returns [(last_scores, last_kept)] per layer (device clones)."""
    from gpu_harness import LockStep
    ls = LockStep(wl)
    ls.fill()
    ls.step(check=False)
    ls.step(check=False)
    torch.cuda.synchronize()
    out = []
    for l in range(wl.n_layers):
        v = hb.hermes_get_cache(ls.h, 0, l)
        assert v["last_T"] > v["len"] == wl.budget
        out.append((v["last_scores"].clone(), v["last_kept"].clone()))
    torch.cuda.synchronize()
    ls.close()
    return out


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["toy", "bf16_reduced"])
def test_noalloc_topk_equals_update_path_two_calls_in_a_row(name):
    wl = CONFIGS["toy"] if name == "toy" else CONFIGS["llava_ov_7b"].scaled(n_layers=6, budget=784, probe_tokens=64)
    ref = _update_path_selection(wl)
    hb.hermes_topk_noalloc_setup()
    la, lb = 0, wl.n_layers - 1                                     # a shallow (recency-only) and a deep layer
    outs = [torch.full((wl.budget,), -7, dtype=torch.int32, device="cuda") for _ in range(2)]
    # two calls in a row on one stream, no synchronisation between them: the second starts from the first one's scratch
    hb.hermes_topk_noalloc(ref[la][0], wl.budget, outs[0])
    hb.hermes_topk_noalloc(ref[lb][0], wl.budget, outs[1])
    torch.cuda.synchronize()
    assert torch.equal(outs[0], ref[la][1]), "first call differs from the update path's kept list"
    assert torch.equal(outs[1], ref[lb][1]), "second call differs from the update path's kept list"
    # and every layer, back to back, into one reused output buffer
    for scores, kept in ref:
        hb.hermes_topk_noalloc(scores, wl.budget, outs[0])
        torch.cuda.synchronize()
        assert torch.equal(outs[0], kept)


@pytest.mark.gpu
def test_noalloc_topk_stale_scratch_max_size_and_ties():
    """A maximum-size call leaves the array full of keys, prefixes and histograms; a small call right behind it must
    not see them.  Ties (quantised scores, and one all-equal vector) follow the (score, index) order."""
    rng = np.random.default_rng(20260114)
    mx = hb.hermes_topk_noalloc_max_tokens()
    big = np.round(rng.standard_normal(mx).astype(np.float32) * 8) / 8            # many equal scores, both signs
    small = rng.standard_normal(1000).astype(np.float32)
    flat = np.full(4133, 0.25, np.float32)                                       # ragged tail, every key equal
    cases = [(big, 6272), (small, 37), (flat, 4000), (big, mx), (small, 1), (big[:33], 32)]
    dev = [(torch.from_numpy(s).cuda(), k, torch.full((k,), -7, dtype=torch.int32, device="cuda")) for s, k in cases]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for s, k, out in dev:                                            # all enqueued back to back on one stream
        hb.hermes_topk_noalloc(s, k, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "device memory was allocated by hermes_topk_noalloc"
    for (s, k), (_, _, out) in zip(cases, dev):
        np.testing.assert_array_equal(out.cpu().numpy(), _expected_topk(s, k))


@pytest.mark.gpu
def test_noalloc_oversize_is_refused_on_the_gpu_too():
    mx = hb.hermes_topk_noalloc_max_tokens()
    s = torch.zeros(mx + 1, dtype=torch.float32, device="cuda")
    out = torch.zeros(8, dtype=torch.int32, device="cuda")
    with pytest.raises(hb.HermesError) as e:
        hb.hermes_topk_noalloc(s, 8, out)
    assert e.value.code == hb.HERMES_ECAPACITY and "exceeds" in str(e.value)
    hb.hermes_topk_noalloc(s[:mx], 8, out)                           # the maximum itself is accepted
    torch.cuda.synchronize()
    np.testing.assert_array_equal(out.cpu().numpy(), np.arange(mx - 8, mx, dtype=np.int32))
