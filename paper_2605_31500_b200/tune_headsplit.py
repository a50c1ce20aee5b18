"""Tuning experiment: does one pass per head group (a smaller gather working set, hence more L2 hits) beat one pass
over all heads of a row?  Each group gets its own contiguous [n, heads_per_pass, d] tensors, so the bytes gathered per
edge are the same and only the working set changes.  Result (profiles/r01_bench_results.md): no - all heads of a row
keep travelling together.

    python -m paper_2605_31500_b200.tune_headsplit <cfg>
"""
import os, sys
import numpy as np, torch
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import gnn_inputs as GI
import paper_2605_31500_b200 as G

cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 3
c = GI.make_config(cfg, keep_f32=False)
n, H, d = c["n"], c["heads"], c["head_dim"]
dev = "cuda"
rp, ci = torch.from_numpy(c["rowptr"]).to(dev), torch.from_numpy(c["colidx"]).to(dev)
plan = G.Plan(rp, ci, transpose="undirected" if cfg == 3 else True)
gt = c["layer"] == "gt"
names = ("q", "k", "v", "do") if gt else ("xl", "xr", "do")
T = {nm: torch.from_numpy(c[nm + "_st"]).view(torch.bfloat16).to(dev) for nm in names}
if not gt:
    a = torch.from_numpy(c["a_f32"]).to(dev)

def timeit(fn, it=5):
    for _ in range(2): fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(True), torch.cuda.Event(True)
    e0.record()
    for _ in range(it): fn()
    e1.record(); torch.cuda.synchronize()
    return e0.elapsed_time(e1) / it

res = {}
for hs in (H, H // 2, 1):
    groups = [slice(g, g + hs) for g in range(0, H, hs)]
    parts = []
    for g in groups:
        P = {nm: T[nm][:, g, :].contiguous() for nm in names}
        P["out"] = torch.empty_like(P[names[0]])
        P["lse"] = torch.empty((n, hs), dtype=torch.float32, device=dev)
        P["stat"] = torch.empty_like(P["lse"])
        P["g1"], P["g2"] = (torch.empty((n, hs, d), dtype=torch.float32, device=dev) for _ in range(2))
        P["g3"] = torch.empty((n, hs, d), dtype=torch.float32, device=dev) if gt else torch.empty((hs, d), dtype=torch.float32, device=dev)
        if not gt: P["a"] = a[g].contiguous()
        parts.append(P)
    def fwd():
        for P in parts:
            if gt: G.gnn_gt_attn_fwd(plan, P["q"], P["k"], P["v"], P["out"], P["lse"])
            else: G.gnn_gatv2_fwd(plan, P["xl"], P["xr"], P["a"], c["slope"], P["out"], P["lse"])
    def bwd():
        for P in parts:
            if gt: G.gnn_gt_attn_bwd(plan, P["q"], P["k"], P["v"], P["lse"], P["do"], P["stat"], P["g1"], P["g2"], P["g3"])
            else: G.gnn_gatv2_bwd(plan, P["xl"], P["xr"], P["a"], P["lse"], P["do"], c["slope"], P["stat"], P["g1"], P["g2"], P["g3"])
    res[hs] = (timeit(fwd), timeit(bwd))
    print(f"cfg{cfg} heads/pass={hs}: fwd {res[hs][0]:.3f} ms  bwd {res[hs][1]:.3f} ms", flush=True)
    del parts
    torch.cuda.empty_cache()
