"""B200-native Scattered Linear Attention (ScatterFormer, arxiv 2401.00912): a C-ABI CUDA library
(include/sla.h, csrc/) plus this thin ctypes binding.  `workloads` holds the seeded synthetic scene
generators shared by tests and bench (no method arithmetic)."""
from .binding import (  # noqa: F401
    SLA_BF16, SLA_F16, SLA_F32, SLA_PHI_ELU1, SLA_PHI_RELU, SYMBOLS, SlaError, load_library, sla_backward, sla_forward, sla_forward_static,
    sla_build_span_table, sla_forward_planned,
    sla_bench_stream_ceiling, sla_forward_host, sla_offsets_from_window_ids, workspace_bytes,
    sla_gather_rows, sla_scatter_rows, sla_sequence_from_coords, sla_sort_by_window, sla_window_count, sla_window_keys,
    sla_cwi_forward, sla_linear, sla_module_forward, sla_qkv_projection,
)
