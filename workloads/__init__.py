"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, and
therefore holds none of the method's arithmetic: no rotation, no codec, no slot
computation.  It describes workloads (shapes, segment lists, block tables,
position maps, frequency tables -- all of which are *inputs* of the kvr_* calls)
and draws K/V values from seeded generators.  See DESIGN.md "Input recipe".
"""
from .configs import (  # noqa: F401
    ADAPTERS, S0, SegmentSpec, Workload, adapter_config, adapter_small, config, config_small, inv_freq_llama3, inv_freq_mrope_temporal, inv_freq_standard,
    make_pool, make_sources, make_workload, pos_map_with_gaps, SENTINEL_BF16, SENTINEL_FP8,
)
from .attention import (  # noqa: F401
    READ_WORKLOADS, ReadSegmentSpec, ReadWorkload, attention_config, make_queries, make_read_sources, read_workload,
)
