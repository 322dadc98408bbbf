"""B200 (sm_100a) closed-shell CCSD(T) perturbative triples energy, arXiv:1609.08094 section 2.2.

The product is the C-ABI library of ``include/triples_b200.h`` (CUDA kernels in ``csrc/``); this package is
its thin Python binding (``binding``) plus the seeded synthetic-input generator (``synth``) shared by the
tests and the benchmark.  There is no CPU fallback: the binding raises if the CUDA library is missing.
"""
from .binding import (  # noqa: F401
    EMU64,
    FP64,
    MIXED,
    TriplesError,
    triples_cache_slots,
    triples_energy,
    triples_energy_host,
    triples_energy_noalloc,
    triples_energy_ri,
    triples_energy_sharded,
    triples_energy_streamed,
    triples_energy_subset,
    triples_last_launch_count,
    triples_last_profile,
    triples_plan_batches,
    triples_plan_shards,
    triples_plan_slices,
    triples_probe_fp64_peak,
    triples_probe_tc_peak,
    triples_set_profiling,
    triples_triplet_count,
    triples_triplet_list,
    triples_w_block,
    triples_workspace_bytes,
    triples_workspace_bytes_host,
    triples_workspace_bytes_ri,
    triples_workspace_bytes_streamed,
)
