"""Tuning sweep: lane width (bytes per lane, GNN_MAX_CB_FWD / GNN_MAX_CB_BWD) and plan thresholds on one of the
BASELINE.json workloads.  The paper autotunes its kernels per graph; this library ships one
fixed configuration and this script is how it was chosen (results: profiles/r01_lane_width_sweep.md).

    python -m paper_2605_31500_b200.tune <cfg> [warp_max,cta_max,split_chunk ...]
"""
import os, sys, time
import numpy as np, torch
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import gnn_inputs as GI
import paper_2605_31500_b200 as G
cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 3
opts = [dict(warp_max_deg=int(a), cta_max_deg=int(b), split_chunk=int(c)) for a, b, c in (x.split(',') for x in sys.argv[2:])] or [dict()]
c = GI.make_config(cfg, keep_f32=False)
n, H, d, dt = c["n"], c["heads"], c["head_dim"], c["dtype"]
gt = c["layer"] == "gt"
def dev(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    return (t.view(torch.bfloat16) if a.dtype == np.uint16 else t).cuda()
rp, ci = dev(c["rowptr"]), dev(c["colidx"])
names = ("q", "k", "v", "do") if gt else ("xl", "xr", "do")
T = {nm: dev(c[nm + "_st"]) for nm in names}
if not gt: T["a"] = dev(c["a_f32"])
out = torch.empty_like(T[names[0]]); lse = torch.empty((n, H), device="cuda"); stat = torch.empty_like(lse)
g1, g2 = (torch.empty((n, H, d), device="cuda") for _ in range(2))
g3 = torch.empty((n, H, d), device="cuda") if gt else torch.empty((H, d), device="cuda")
def timeit(fn, k=5):
    fn(); torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(k): fn()
    b.record(); torch.cuda.synchronize()
    return a.elapsed_time(b) / k
for o in opts:
    plan = G.Plan(rp, ci, **o)
    if gt:
        fwd = lambda: G.gnn_gt_attn_fwd(plan, T["q"], T["k"], T["v"], out, lse)
        bwd = lambda: G.gnn_gt_attn_bwd(plan, T["q"], T["k"], T["v"], lse, T["do"], stat, g1, g2, g3)
    else:
        fwd = lambda: G.gnn_gatv2_fwd(plan, T["xl"], T["xr"], T["a"], c["slope"], out, lse)
        bwd = lambda: G.gnn_gatv2_bwd(plan, T["xl"], T["xr"], T["a"], lse, T["do"], c["slope"], stat, g1, g2, g3)
    for cbf in (32, 16):
        os.environ["GNN_MAX_CB_FWD"] = str(cbf)
        G.gnn_profile_enable(True); fwd(); G.gnn_profile_enable(False)
        pr = {k: round(v, 3) for k, v in G.gnn_profile_collect()}
        print(f"cfg{cfg} {o} fwd cb={cbf}: {timeit(fwd):.3f} ms {pr}", flush=True)
    for cbb in (32, 16):
        os.environ["GNN_MAX_CB_BWD"] = str(cbb)
        G.gnn_profile_enable(True); bwd(); G.gnn_profile_enable(False)
        pr = {k: round(v, 3) for k, v in G.gnn_profile_collect()}
        print(f"cfg{cfg} {o} bwd cb={cbb}: {timeit(bwd):.3f} ms  {pr}", flush=True)
    del plan
