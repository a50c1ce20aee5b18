"""paper_2605_31500_b200 - fused CSR graph attention (Graph Transformer + GATv2, fwd + bwd) for B200.

Thin Python binding over the C-ABI library ``libgnn_attn.so`` (``include/gnn_attn.h``): argument
marshalling only; every step of the path runs in the library's sm_100a kernels.  PyTorch is used
for device memory and streams.  There is no CPU fallback: importing works without a GPU (the
library loads and exports its symbols), but any compute call without a CUDA device raises.
"""
from .binding import (  # noqa: F401
    GnnError, lib, Plan, PlanOpts,
    gnn_csr_validate, gnn_plan_bytes, gnn_plan_build, gnn_plan_destroy, gnn_plan_export, gnn_workspace_bytes,
    gnn_gt_attn_fwd, gnn_gt_attn_fwd_block, gnn_gt_attn_fwd_wsb, gnn_gt_attn_bwd_wsb, gnn_gt_attn_bwd_block, gnn_gt_attn_bwd, gnn_gatv2_fwd, gnn_gatv2_bwd,
    gnn_seg_minmax_fwd, gnn_seg_minmax_bwd, GNN_AGG_MIN, GNN_AGG_MAX, GNN_OP_SEG_MINMAX_FWD,
    gnn_last_error, gnn_version, gnn_launch_count, gnn_profile_enable, gnn_profile_collect, gnn_pdl_enable, gnn_probe_gather, gnn_ln_qkv_fwd, gnn_dot_aggr,
    gnn_static_workspace_limit, gnn_gt_attn_fwd_static,
    GNN_F32, GNN_BF16, GNN_OP_GT_FWD, GNN_OP_GT_BWD, GNN_OP_GATV2_FWD, GNN_OP_GATV2_BWD,
    GNN_TRANSPOSE_NONE, GNN_TRANSPOSE_BUILD, GNN_TRANSPOSE_UNDIRECTED, GNN_BLOCKS_DIAG, GNN_BLOCKS_WSB,
    EXPORTED_SYMBOLS,
)
