"""paper_2607_05439_b200 -- B200-native pair-bias attention (the one-GPU core of Design-CP).

`csrc/` holds the CUDA kernels and the C ABI (include/designcp.h); `binding.py` is the thin
ctypes layer with the same names.  Importing the package requires the built library
(`python paper_2607_05439_b200/build.py`); there is no CPU fallback.
"""
from .binding import (  # noqa: F401
    DcpError, Event, dcp_atom_pair_bias_attention, dcp_attention_stack, dcp_attention_stack_cache_bytes, dcp_attention_stack_cached, dcp_attention_stack_cached_workspace_bytes, dcp_attention_stack_workspace_bytes, dcp_gather_pair_slice, dcp_kernel_supported, dcp_knn, dcp_knn_budget, dcp_last_launch_count, dcp_merge_states, dcp_no_alloc_scratch_bytes, dcp_pair_bias_attention_no_alloc,
    dcp_pair_bias_attention, dcp_pair_bias_attention_host, dcp_pair_transition, dcp_pairformer_stack, dcp_partial_states, dcp_plan_units, dcp_probe_l2_gather, dcp_probe_scan, dcp_shard_range,
    dcp_sparse_atom_attention, dcp_sparse_atom_workspace_bytes, dcp_workspace_bytes, status_string, version,
)
