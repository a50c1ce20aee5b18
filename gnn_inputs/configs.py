"""The five BASELINE.json workloads as seeded synthetic inputs (recipe: DESIGN.md section 4).

``make_config(cfg, scale)`` returns a dict with the graph (int32 CSR, row = dst) and the
feature tensors in storage dtype (``*_st``: fp32 array, or uint16 bf16 bit patterns) plus
their exact fp32 up-casts (``*_f32``) for the oracle (``keep_f32=False`` skips the up-cast copies of
bf16 tensors to save host memory at full size; ``gnn_inputs.bf16_bits_to_f32`` recreates them).  ``scale`` < 1 shrinks node and edge
counts proportionally (parity tests); scale = 1 is the BASELINE.json size.
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor

import numpy as np

from . import graphs as G
from .tensors import rng_for, normal_tensor, store

CONFIGS = {
    1: dict(name="cfg1_gt_er1k_f32", layer="gt", dtype="f32", n=1_000, heads=4, head_dim=16),
    2: dict(name="cfg2_gatv2_chunglu170k_bf16", layer="gatv2", dtype="bf16", n=170_000, heads=8, head_dim=16,
            in_dim=128, slope=0.2),
    3: dict(name="cfg3_gt_rmat2p4m_bf16", layer="gt", dtype="bf16", n=2_400_000, heads=4, head_dim=64),
    4: dict(name="cfg4_gt_community1m_bf16", layer="gt", dtype="bf16", n=1_000_000, heads=8, head_dim=64),
    5: dict(name="cfg5_gatv2_rmat4m_hubs_bf16", layer="gatv2", dtype="bf16", n=4_000_000, heads=4, head_dim=32,
            in_dim=128, slope=0.2),
}


def config_name(cfg: int) -> str:
    return CONFIGS[cfg]["name"]


def _graph(cfg: int, scale: float, seed: int, relabel: bool = True, dense: bool = False):
    c = CONFIGS[cfg]
    n = max(64, int(round(c["n"] * scale)))
    r0, r1, r2, r3 = (rng_for(cfg, s, seed) for s in (0, 1, 2, 3))
    if cfg == 1:
        return n, G.erdos_renyi(n, 8.0, r0)
    if cfg == 2:
        n_pairs = int(round(1_200_000 * scale))
        w_max = max(16.0, 10_000.0 * min(1.0, scale * 4))
        return n, G.chung_lu(n, n_pairs, 2.1, w_max, r0, r1)
    if cfg == 3:
        bits = max(7, int(np.ceil(np.log2(n))))
        samples = 85_000_000 if dense else 41_500_000   # dense = "cfg 3b": ~124 M stored entries, average degree ~50 (ogbn-products' shape)
        return n, G.rmat_symmetric(n, bits, int(round(samples * scale)), (0.57, 0.19, 0.19), r0, r1 if relabel else None)
    if cfg == 4:
        n = (n // 16) * 16
        return n, G.community_graph(n, 16, 0.6, 2, r0, r3)
    if cfg == 5:
        bits = max(7, int(np.ceil(np.log2(n))))
        hubs = [int(round(h * scale)) for h in (3_000_000, 2_000_000, 1_500_000, 1_100_000)]
        return n, G.rmat_hubs(n, bits, int(round(100_000_000 * scale)), (0.65, 0.15, 0.15), hubs, r0, r1, r2)
    raise ValueError(cfg)


def make_config(cfg: int, scale: float = 1.0, seed: int = 0, with_grads: bool = True, keep_f32: bool = True,
                relabel: bool = True, dense: bool = False) -> dict:
    """relabel=False (cfg 3 only) keeps the natural R-MAT ids: the locality study of SURVEY section 8(d), not the headline."""
    c = dict(CONFIGS[cfg])
    if (not relabel or dense) and cfg != 3:
        raise ValueError("relabel=False / dense=True are defined for cfg 3 only")
    n, (rowptr, colidx) = _graph(cfg, scale, seed, relabel, dense)
    if dense:
        c["name"] = c["name"].replace("cfg3_", "cfg3b_deg50_")
    h, d, dt = c["heads"], c["head_dim"], c["dtype"]
    out = dict(c, cfg=cfg, scale=scale, seed=seed, relabel=relabel, n=n, e=int(colidx.size), rowptr=rowptr, colidx=colidx)
    if c["layer"] == "gt":
        names = (("q", 10), ("k", 11), ("v", 12)) + ((("do", 13),) if with_grads else ())
        # independent streams -> drawn in parallel threads (numpy releases the GIL); same values either way
        with ThreadPoolExecutor(max_workers=len(names)) as ex:
            res = list(ex.map(lambda ns: store(normal_tensor(rng_for(cfg, ns[1], seed), (n, h, d)), dt, keep_f32), names))
        for (name, _), (st, f32) in zip(names, res):
            out[name + "_st"], out[name + "_f32"] = st, f32
    else:
        fin = c["in_dim"]
        x = normal_tensor(rng_for(cfg, 20, seed), (n, fin))
        w_s = normal_tensor(rng_for(cfg, 21, seed), (h * d, fin), std=fin ** -0.5)   # N(0, var 1/in_dim)
        w_t = normal_tensor(rng_for(cfg, 22, seed), (h * d, fin), std=fin ** -0.5)
        a = normal_tensor(rng_for(cfg, 23, seed), (h, d), std=d ** -0.5)            # N(0, var 1/head_dim)
        # dense input projections: outside the fused kernels
        for name, w in (("xl", w_s), ("xr", w_t)):
            st, f32 = store((x @ w.T).reshape(n, h, d), dt, keep_f32)
            out[name + "_st"], out[name + "_f32"] = st, f32
        out["a_f32"] = np.ascontiguousarray(a, dtype=np.float32)
        if with_grads:
            st, f32 = store(normal_tensor(rng_for(cfg, 24, seed), (n, h, d)), dt, keep_f32)
            out["do_st"], out["do_f32"] = st, f32
    return out
