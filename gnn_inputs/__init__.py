"""Seeded synthetic inputs (graphs + feature tensors) for the five BASELINE.json configs.

This module is the ONLY code shared by the oracle side (``oracle/``, tests) and the
CUDA side (``paper_2605_31500_b200/``, ``bench.py``).  It holds none of the method's
arithmetic: no scores, no softmax, no aggregation, no gradients, no plan / binning /
transposition logic.  It only draws random graphs and random feature tensors, rounds
them to the storage dtype, and (for GATv2) applies the dense input projection that the
paper places outside the fused kernels ("not subject to optimization",
PAPER.md:488 "precomputed per-node features").

The paper's datasets (GraphLand, OGB, Planetoid; Table 8)
are not available; these graphs stand in for them (recipe in DESIGN.md section 4).
"""
from .graphs import (  # noqa: F401
    csr_from_pairs,
    erdos_renyi,
    chung_lu,
    rmat_symmetric,
    community_graph,
    rmat_hubs,
    degree_stats,
)
from .tensors import (  # noqa: F401
    f32_to_bf16_bits,
    bf16_bits_to_f32,
    normal_tensor,
    store,
)
from .configs import CONFIGS, make_config, config_name  # noqa: F401
