"""GPU parity on seeded random geometries: head counts, head_dim, dtype, budget, chunk and probe sizes that are not
multiples of any tile (128-token K tiles, 32-row MMA blocks, 32-token flag chunks, 16-byte units), both scoring paths,
1D RoPE and M-RoPE, eager and lazy re-indexing, with and without the summary token, one or two streams.  Same lock-step comparison with the
oracle, same tolerances, as tests/test_gpu_parity.py; the fixed workloads there only cover the paper's geometries."""
import numpy as np
import pytest

import paper_2601_14724_b200 as hb
from gpu_harness import LockStep
from workloads import Workload

pytestmark = pytest.mark.gpu


def _draw(seed: int):
    """One random workload + config overrides.  Even seeds force the tcgen05 path's preconditions (bf16, d = 128,
    G * P >= 32, T >= 512); odd seeds roam over everything the CUDA-core path accepts."""
    r = np.random.default_rng(9000 + seed)
    tc = seed % 2 == 0
    d = 128 if tc else int(r.choice([32, 64, 128]))
    dtype = "bf16" if tc else str(r.choice(["bf16", "f32"]))
    hkv = int(r.choice([1, 2, 3, 4]))
    grp = int(r.choice([2, 4, 7] if tc else [1, 2, 3, 7]))
    L = int(r.integers(3, 7))
    m3d = seed % 3 == 2
    if m3d:
        gh, gw = int(r.choice([2, 4])), int(r.choice([2, 4, 8]))
        tpt = gh * gw
        chunk = tpt * int(r.integers(2, 7))
        sec_t = int(r.integers(1, d // 4))
        sec_h = int(r.integers(1, d // 2 - sec_t))
        section = (sec_t, sec_h, d // 2 - sec_t - sec_h)
        axes = int(r.choice([0b001, 0b111]))
    else:
        gh = gw = 8
        tpt = int(r.integers(5, 40))
        chunk = int(r.integers(3, 160))
        section, axes = (d // 2 - 2, 1, 1), 0b001
    budget = int(r.integers(520, 900)) if tc else int(r.integers(70, 700))
    probe = int(r.integers(max(1, -(-32 // grp)), 72)) if tc else int(r.integers(1, 40))
    wl = Workload(name=f"random{seed}", n_layers=L, n_q_heads=hkv * grp, n_kv_heads=hkv, head_dim=d, dtype=dtype,
                  tokens_per_frame=tpt, budget=budget, chunk_tokens=chunk, probe_tokens=probe,
                  rope_theta=float(r.choice([1.0e4, 1.0e6])), seed=7000 + seed, rope_mode="m3d" if m3d else "1d",
                  mrope_section=section, mrope_compact_axes=axes, mrope_grid_h=gh, mrope_grid_w=gw,
                  pos_offset=int(r.integers(0, 20)), n_streams=2 if seed % 4 == 3 else 1)
    over, oover = {}, {}
    if not m3d and r.integers(0, 3) == 0:                      # lazy re-indexing, re-index step somewhere in the run
        mp = wl.pos_offset + budget + chunk * int(r.integers(2, 5)) + 2
        over.update(reindex_mode=hb.HERMES_REINDEX_LAZY, max_position=mp)
        oover.update(reindex_mode="lazy", max_position=mp, max_chunk_span=chunk)
    if not m3d and r.integers(0, 3) == 0:
        over.update(summary_token=1); oover.update(summary_token=True)
    if r.integers(0, 2) == 0:
        over.update(norm_mode=hb.HERMES_NORM_SUM); oover.update(norm_mode="sum")
    return wl, over, oover, tc


@pytest.mark.parametrize("seed", range(24))
def test_random_geometry_lockstep(seed):
    wl, over, oover, tc = _draw(seed)
    what = f"seed {seed}: {wl} cfg {over}"
    ls = LockStep(wl, over, oover)
    try:
        ls.fill()
        reps = []
        for _ in range(4):
            reps += ls.step(check=True)
        assert all(r["evicted"] for r in reps), what
        assert all(r["max_score_rel"] < 1e-3 for r in reps), what
        if tc:
            assert hb.hermes_last_score_path(ls.h) == hb.HERMES_SCORE_TCGEN05, what
        assert hb.hermes_device_status(ls.h) & 1 == 0, what
    except AssertionError as e:
        raise AssertionError(f"{what}\n{e}") from e
    finally:
        ls.close()
