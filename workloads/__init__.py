"""Seeded synthetic inputs shared by the CPU oracle's tests and the CUDA path's tests / bench.

This package holds NONE of the method's arithmetic (no scoring, smoothing, selection,
compaction or rotary correction): only workload geometry and random tensors shaped like
what an MLLM would hand to the cache manager.  See DESIGN.md "Input recipe".
"""
from .synth import (CONFIGS, Workload, chunk_kv, probe_q, rope_at_arrival, round_storage,
                    storage_bits, stream_rng, sweep_point)

__all__ = ["CONFIGS", "Workload", "chunk_kv", "probe_q", "rope_at_arrival", "round_storage",
           "storage_bits", "stream_rng", "sweep_point"]
