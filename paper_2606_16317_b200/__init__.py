"""B200 (sm_100a) tile-skipping attention forward of arxiv/paper_2606_16317 (DynSparse).

Thin ctypes binding over the C ABI in include/sparse_attn.h; every step of the hot path runs in
the CUDA kernels of csrc/.  There is no CPU fallback: compute calls raise on a machine without
the built extension or without an sm_100 device.
"""
from .binding import (  # noqa: F401
    MODE_DENSE,
    MODE_DYNAMIC,
    MODE_FIXED,
    MODE_MASK,
    SELECT_TOPK,
    SELECT_TOPP,
    SparseAttnError,
    SparseAttnParams,
    lambda_from_preal,
    lambda_from_recall,
    last_error,
    launch_count,
    library_path,
    make_params,
    sparse_attn_block_mass,
    sparse_attn_block_stats,
    sparse_attn_brick_permutation,
    sparse_attn_fwd,
    sparse_attn_fwd_host,
    sparse_attn_reorder_tokens,
    sparse_attn_output_error,
    sparse_attn_recall_stats,
    sparse_attn_release_scratch,
    sparse_attn_row_topk_curve,
    sparse_attn_row_topk_curve_static,
    sparse_attn_select_blocks,
    sparse_attn_select_blocks_greedy,
    status_string,
    version,
)
