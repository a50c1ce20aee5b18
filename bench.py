#!/usr/bin/env python
"""bench.py - fused GT / GATv2 attention forward+backward GEdges/s on one BASELINE.json workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg C] [--impl ours|reference]

One "step" = one pass of the whole hot path (plan resident; forward + backward = dst pass + src pass)
over the config's synthetic graph.  Prints ONE JSON line (see DESIGN.md section 8 for every key).
`value` = edges * ranks / max-over-ranks device time, inputs resident in HBM.  `e2e` = the same metric with
the host->device copies of every input and the device->host copies of every output inside the timed region.
`--impl reference` times the fp64 CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gnn_inputs as GI  # noqa: E402

METRIC = "fused GT/GATv2 attn GEdges/s (fwd+bwd)"
UNIT = "GEdges/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=3, help="BASELINE.json config 1..5 (default 3: the large power-law GT graph)")
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the workload (debug only; < 1 is not a bench value)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=4)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--natural-ids", action="store_true",
                    help="cfg 3: keep the natural R-MAT ids instead of the random relabel (locality study, SURVEY 8(d))")
    ap.add_argument("--dense", action="store_true",
                    help="cfg 3 only: variant 3b, 85 M R-MAT samples -> ~124 M stored entries (ogbn-products' shape); not the headline")
    ap.add_argument("--directed-plan", action="store_true",
                    help="cfg 3: build CSR^T instead of reusing the forward CSR in the backward (row f1)")
    ap.add_argument("--no-minmax", action="store_true", help="skip the extra row-f3 (min aggregation) measurement of cfg 3 / 5")
    ap.add_argument("--degree-sorted-ids", action="store_true",
                    help="relabel the nodes by descending in-degree (graph and every per-node tensor: same graph, same data) so that "
                         "the most gathered K / V rows form a contiguous prefix; locality experiment, not the headline")
    ap.add_argument("--l2-window", type=float, default=0.0,
                    help="MB of the K tensor's prefix to pin in L2 (cudaAccessPolicyWindow, persisting) on the bench stream; "
                         "meant for --degree-sorted-ids; locality experiment, not the headline")
    ap.add_argument("--no-all-configs", action="store_true",
                    help="default run (cfg 3) only: skip the compact measurements of cfg 1, 2, 4, 5 (`all_configs`)")
    ap.add_argument("--no-extras", action="store_true", help="skip the gather-ceiling probe and the row-f4 measurements")
    ap.add_argument("--warp-max-deg", type=int, default=0)
    ap.add_argument("--cta-max-deg", type=int, default=0)
    ap.add_argument("--split-chunk", type=int, default=0)
    return ap.parse_args()


# ------------------------------------------------------------------------------------------ byte model
def byte_model(c, plan_counts, deg_in, deg_out, perm, perm_t):
    """Algorithmic bytes per kernel launch (SURVEY.md section 8(d) per-edge / per-node figures x units) and
    compulsory bytes per pass (every array read or written once)."""
    n, e, H, d = c["n"], c["e"], c["heads"], c["head_dim"]
    b = 4 if c["dtype"] == "f32" else 2
    R = H * d
    if c["layer"] == "gt":
        per = {  # pass: (bytes per edge, bytes per row)
            "gt_fwd": (4 + 2 * R * b, 8 + 2 * R * b + 4 * H),
            "gt_bwd_dst": (4 + 2 * R * b, 8 + 2 * R * b + 4 * H + 4 * R + 4 * H),
            "gt_bwd_src": (4 + 2 * R * b + 8 * H, 8 + 2 * R * b + 8 * R),
        }
        csr = 4 * (n + 1) + 4 * e
        comp = {"fwd": csr + 4 * n * R * b + 4 * n * H,
                "bwd": 2 * csr + 4 * n * R * b + 4 * n * H + 12 * n * R + 8 * n * H}
    else:
        per = {
            "gatv2_fwd": (4 + R * b, 8 + 2 * R * b + 4 * H),
            "gatv2_bwd_dst": (4 + R * b, 8 + 2 * R * b + 4 * H + 4 * R + 4 * H),
            "gatv2_bwd_src": (4 + 2 * R * b + 8 * H, 8 + R * b + 4 * R),
        }
        csr = 4 * (n + 1) + 4 * e
        comp = {"fwd": csr + 3 * n * R * b + 4 * n * H + 4 * R,
                "bwd": 2 * csr + 3 * n * R * b + 4 * n * H + 8 * n * R + 8 * n * H + 8 * R}
    alg = {}
    for ps, (pe, pn) in per.items():
        t = ps.endswith("_src")
        deg, pm = (deg_out, perm_t) if t else (deg_in, perm)
        sfx = "_t" if t else ""
        nh, nc = plan_counts["n_hub" + sfx], plan_counts["n_cta" + sfx]
        ng, nch = plan_counts["n_group" + sfx], plan_counts["n_chunks" + sfx]
        e_heavy = int(deg[pm[: nh + nc]].sum())
        e_group = int(deg[pm[nh + nc:]].sum())
        alg[ps + "/segment"] = e_heavy * pe + (nc + nch) * pn
        alg[ps + "/group"] = e_group * pe + ng * pn
    return alg, comp


def compulsory_bytes(c):
    """Compulsory bytes per pass: rowptr + colidx (+ CSR^T for the backward) + every tensor once + outputs
    (O in the feature dtype, gradients fp32, L / Delta / G fp32)."""
    n, e, H, d = c["n"], c["e"], c["heads"], c["head_dim"]
    b = 4 if c["dtype"] == "f32" else 2
    R = H * d
    csr = 4 * (n + 1) + 4 * e
    if c["layer"] == "gt":
        return {"fwd": csr + 4 * n * R * b + 4 * n * H, "bwd": 2 * csr + 4 * n * R * b + 4 * n * H + 12 * n * R + 8 * n * H}
    return {"fwd": csr + 3 * n * R * b + 4 * n * H + 4 * R, "bwd": 2 * csr + 3 * n * R * b + 4 * n * H + 8 * n * R + 8 * n * H + 8 * R}


def quick_config(cfg, args, dev, peak):
    """Compact measurement of one more BASELINE.json config in the same run (`all_configs`): the same calls, the same
    timing rules (>= 3 warm-up steps, CUDA events on the launch stream, L2 flushed between steps when the inputs do not
    exceed it), forward / backward / step times, GEdges/s and the compulsory-byte fractions.  cfg 4 also times the
    tcgen05 paths (diagonal block forward, WSB forward + backward)."""
    import torch
    import paper_2605_31500_b200 as G
    c = GI.make_config(cfg, keep_f32=False)
    n, e, H, d, dt = c["n"], c["e"], c["heads"], c["head_dim"], c["dtype"]
    gt = c["layer"] == "gt"
    names = ("q", "k", "v", "do") if gt else ("xl", "xr", "do")

    def to_dev(a):
        t = torch.from_numpy(np.ascontiguousarray(a))
        return (t.view(torch.bfloat16) if (dt == "bf16" and a.dtype == np.uint16) else t).to(dev)

    T = {nm: to_dev(c[nm + "_st"]) for nm in names}
    rp, ci = torch.from_numpy(c["rowptr"]).to(dev), torch.from_numpy(c["colidx"]).to(dev)
    if not gt:
        T["a"] = torch.from_numpy(c["a_f32"]).to(dev)
    plan = G.Plan(rp, ci, transpose=True, blocks=(cfg == 4), wsb=(cfg == 4))
    f32 = dict(dtype=torch.float32, device=dev)
    out = torch.empty((n, H, d), dtype=T[names[0]].dtype, device=dev)
    lse, stat = torch.empty((n, H), **f32), torch.empty((n, H), **f32)
    g1, g2 = torch.empty((n, H, d), **f32), torch.empty((n, H, d), **f32)
    g3 = torch.empty((n, H, d), **f32) if gt else torch.empty((H, d), **f32)
    if gt:
        fwd = lambda: G.gnn_gt_attn_fwd(plan, T["q"], T["k"], T["v"], out, lse)
        bwd = lambda: G.gnn_gt_attn_bwd(plan, T["q"], T["k"], T["v"], lse, T["do"], stat, g1, g2, g3)
    else:
        fwd = lambda: G.gnn_gatv2_fwd(plan, T["xl"], T["xr"], T["a"], c["slope"], out, lse)
        bwd = lambda: G.gnn_gatv2_bwd(plan, T["xl"], T["xr"], T["a"], lse, T["do"], c["slope"], stat, g1, g2, g3)
    in_bytes = sum(int(v.numel()) * v.element_size() for v in list(T.values()) + [rp, ci])
    l2 = torch.cuda.get_device_properties(dev).L2_cache_size
    flush = torch.empty(max(2 * l2, 1 << 28), dtype=torch.uint8, device=dev) if in_bytes < 4 * l2 else None

    def timed(fn, k):
        evs = []
        for _ in range(k):
            if flush is not None:
                flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record()
            evs.append((a, b))
        torch.cuda.synchronize()
        return float(np.mean([a.elapsed_time(b) for a, b in evs]))

    step = lambda: (fwd(), bwd())
    for _ in range(max(args.warmup, 3)):
        step()
    l0 = G.gnn_launch_count()
    ms_step = timed(step, args.steps)
    launches = (G.gnn_launch_count() - l0) // max(args.steps, 1)
    ms_f, ms_b = timed(fwd, args.steps), timed(bwd, args.steps)
    comp = compulsory_bytes(c)
    frac = lambda byts, ms: byts / (ms * 1e-3) * 1e-9 / peak
    r = {"workload": c["name"], "layer": c["layer"], "nodes": n, "edges": e, "heads": H, "head_dim": d, "feature_dtype": dt,
         "ms_per_step": ms_step, "ms_fwd": ms_f, "ms_bwd": ms_b, "gedges": e / (ms_step * 1e-3) * 1e-9,
         "gedges_fwd": e / (ms_f * 1e-3) * 1e-9, "gedges_bwd": e / (ms_b * 1e-3) * 1e-9, "launches_per_step": int(launches),
         "l2": "L2 flushed between timed steps" if flush is not None else "inputs larger than L2 (no flush)",
         "compulsory_frac_fwd": frac(comp["fwd"], ms_f), "compulsory_frac_bwd": frac(comp["bwd"], ms_b),
         "compulsory_frac_step": frac(comp["fwd"] + comp["bwd"], ms_step), "plan": plan.counts()}
    if cfg == 4:
        fb = lambda: G.gnn_gt_attn_fwd_block(plan, T["q"], T["k"], T["v"], out, lse)
        fw = lambda: G.gnn_gt_attn_fwd_wsb(plan, T["q"], T["k"], T["v"], out, lse)
        bw = lambda: G.gnn_gt_attn_bwd_wsb(plan, T["q"], T["k"], T["v"], out, lse, T["do"], stat, g1, g2, g3)
        bb = lambda: G.gnn_gt_attn_bwd_block(plan, T["q"], T["k"], T["v"], lse, T["do"], stat, g1, g2, g3)
        for _ in range(3):
            fb(); fw(); bw(); bb()
        ms_fb, ms_fw, ms_bw = timed(fb, args.steps), timed(fw, args.steps), timed(bw, args.steps)
        ms_bb, ms_sb = timed(bb, args.steps), timed(lambda: (fb(), bb()), args.steps)
        ms_mx = timed(lambda: (fb(), bwd()), args.steps)     # fastest measured composition: tcgen05 forward + CSR backward
        r["tcgen05_paths"] = {"block_fwd_ms": ms_fb, "block_fwd_compulsory_frac": frac(comp["fwd"], ms_fb),
                              "block_bwd_ms": ms_bb, "block_bwd_compulsory_frac": frac(comp["bwd"], ms_bb),
                              "block_step_ms": ms_sb, "block_step_gedges": e / (ms_sb * 1e-3) * 1e-9,
                              "block_step_compulsory_frac": frac(comp["fwd"] + comp["bwd"], ms_sb),
                              "mixed_step_ms": ms_mx, "mixed_step_gedges": e / (ms_mx * 1e-3) * 1e-9,
                              "mixed_step_compulsory_frac": frac(comp["fwd"] + comp["bwd"], ms_mx),
                              "wsb_fwd_ms": ms_fw, "wsb_bwd_ms": ms_bw, "wsb_info": plan.wsb_info(),
                              "note": "block_* = diagonal block layout (tile-local tcgen05 + remainder CSR), wsb_* = general WSB layout, "
                                      "mixed_* = block forward + CSR backward"}
    del T, out, lse, stat, g1, g2, g3, plan, flush
    torch.cuda.empty_cache()
    return r


def degree_sort_config(c):
    """Same graph and data under new labels: node ids sorted by descending in-degree (ties: old id)."""
    n = c["n"]
    deg = np.diff(c["rowptr"].astype(np.int64))
    order = np.argsort(-deg, kind="stable")
    new_id = np.empty(n, np.int64)
    new_id[order] = np.arange(n)
    dst = np.repeat(np.arange(n, dtype=np.int64), deg)
    rp, ci = GI.csr_from_pairs(n, new_id[dst], new_id[c["colidx"].astype(np.int64)], self_loops=False, dedupe=False)
    out = dict(c, rowptr=rp, colidx=ci, relabel="degree-sorted")
    for k, v in c.items():
        if k.endswith("_st") and isinstance(v, np.ndarray) and v.shape[0] == n:
            out[k] = np.ascontiguousarray(v[order])
    return out


def set_l2_window(ptr, nbytes, stream_handle, persist_bytes):
    """cudaDeviceSetLimit(persisting L2) + cudaStreamSetAttribute(access policy window) through the loaded libcudart.
    Returns a dict describing what the runtime accepted (plumbing: streams and memory policy, no compute)."""
    import ctypes as C
    path = None
    for line in open("/proc/self/maps"):
        if "libcudart" in line:
            path = line.split()[-1]
            break
    if path is None:
        return {"error": "libcudart not found in the process"}
    rt = C.CDLL(path)
    mx_win, mx_per = C.c_int(0), C.c_int(0)
    rt.cudaDeviceGetAttribute(C.byref(mx_win), 109, 0)     # cudaDevAttrMaxAccessPolicyWindowSize
    rt.cudaDeviceGetAttribute(C.byref(mx_per), 108, 0)     # cudaDevAttrMaxPersistingL2CacheSize
    persist = min(int(persist_bytes), mx_per.value)
    rc1 = rt.cudaDeviceSetLimit(6, C.c_size_t(persist))    # cudaLimitPersistingL2CacheSize

    class Win(C.Structure):
        _fields_ = [("base_ptr", C.c_void_p), ("num_bytes", C.c_size_t), ("hitRatio", C.c_float), ("hitProp", C.c_int),
                    ("missProp", C.c_int)]

    class Val(C.Union):
        _fields_ = [("pad", C.c_char * 64), ("win", Win)]

    v = Val()
    nb = min(int(nbytes), mx_win.value)
    v.win = Win(ptr, nb, 1.0, 2, 1) if nb > 0 else Win(None, 0, 0.0, 0, 0)     # hit: persisting, miss: streaming
    rc2 = rt.cudaStreamSetAttribute(C.c_void_p(stream_handle), 1, C.byref(v))   # cudaStreamAttributeAccessPolicyWindow
    return {"window_bytes": nb, "persisting_limit_bytes": persist, "max_window_bytes": mx_win.value,
            "max_persisting_bytes": mx_per.value, "rc_set_limit": rc1, "rc_set_attr": rc2}


def event_ms(fn, reps=3, warm=1):
    import torch
    for _ in range(warm):
        fn()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(reps):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps


def gather_ceilings(row_bytes, dev):
    """Ceiling 2 of DESIGN.md section 6, measured in this process through the C ABI (gnn_probe_gather): GB/s of uniformly
    random `row_bytes` rows from an HBM-resident table (2.4 GB) and from an L2-resident one (48 MB); register gathers
    (256-bit loads, 4 rows in flight per lane group) at 32 and at 16 resident warps per SM - the traversal kernels run at
    12-16 - and cp.async.bulk copies at 16 warps per SM."""
    import torch
    import paper_2605_31500_b200 as G
    rb = 256 if row_bytes <= 256 else (512 if row_bytes <= 512 else 1024)
    n_idx = 1 << 25
    sink = torch.zeros(1, dtype=torch.float32, device=dev)
    res = {"row_bytes": rb, "n_gathers": n_idx}
    for name, tbytes in (("hbm_resident", 2_400_000_000), ("l2_resident", 48_000_000)):
        rows = tbytes // rb
        table = torch.ones(rows * rb, dtype=torch.uint8, device=dev)
        idx = torch.randint(0, rows, (n_idx,), dtype=torch.int32, device=dev)
        r = {}
        for key, mode, depth, cps in (("ldg_32warps", 0, 4, 8), ("ldg_16warps", 0, 4, 4), ("bulk_16warps", 1, 8, 4)):
            ms = event_ms(lambda: G.gnn_probe_gather(table, rb, idx, mode, depth, cps, sink))
            r[key + "_gbs"] = n_idx * rb / (ms * 1e-3) * 1e-9
        res[name] = r
        del table, idx
    torch.cuda.empty_cache()
    return res


def block_extras(c, dev, peak, bf16_peak):
    """Row f4 on the main config's shape: (1) the fused LayerNorm + QKV projection in front of the GT attention
    (input features = H * d as in the paper's block), bytes = x + q, k, v + W once, flops = 2 n C 3R;
    (2) cfg 3 only: the dot-aggr locality study - second-pass times of the feature-parallel and the
    neighbour-parallel kernel, scalar and 16-byte loads, fp32 D = 64, on the config's ids (random relabel = "orig") and
    on two reorderings (natural R-MAT ids, ids sorted by descending in-degree); s = t_orig / t_reordered,
    gap = s_neighbour - s_feature."""
    import torch
    import paper_2605_31500_b200 as G
    n, H, d = c["n"], c["heads"], c["head_dim"]
    R = H * d
    out = {}
    if c["layer"] == "gt" and R % 128 == 0 and 64 <= R <= 512:
        g = torch.Generator(device=dev).manual_seed(1)
        x = torch.randn((n, R), device=dev, generator=g).to(torch.bfloat16)
        w = (torch.randn((3 * R, R), device=dev, generator=g) * R ** -0.5).to(torch.bfloat16)
        gamma, beta = torch.ones(R, device=dev), torch.zeros(R, device=dev)
        bias = torch.zeros(3 * R, device=dev)
        q, k, v = (torch.empty((n, H, d), dtype=torch.bfloat16, device=dev) for _ in range(3))
        ms = event_ms(lambda: G.gnn_ln_qkv_fwd(x, gamma, beta, 1e-5, w, bias, q, k, v), reps=5, warm=2)
        F = torch.nn.functional
        gb, bb, biasb = gamma.bfloat16(), beta.bfloat16(), bias.bfloat16()
        ms_lib = event_ms(lambda: F.linear(F.layer_norm(x, (R,), gb, bb, 1e-5), w, biasb), reps=5, warm=2)   # context only
        byts = n * R * 2 * 4 + 3 * R * R * 2
        fl = 2.0 * n * R * 3 * R
        out["ln_qkv"] = {"ms": ms, "c_in": R, "out_features": 3 * R, "bytes": byts, "gbs": byts / (ms * 1e-3) * 1e-9,
                         "frac_of_hbm_peak": byts / (ms * 1e-3) * 1e-9 / peak, "tflops": fl / (ms * 1e-3) * 1e-12,
                         "frac_of_bf16_peak": (fl / (ms * 1e-3) * 1e-12 / bf16_peak) if bf16_peak else None,
                         "library_layer_norm_plus_linear_ms": ms_lib,
                         "note": "LayerNorm fused into the A-operand staging of a tcgen05 GEMM; x, W random, timed alone; the library "
                                 "figure (torch layer_norm kernel + cuBLAS linear, the paper's own arrangement) is context, not a product path"}
        del x, w, q, k, v
    if c["cfg"] == 3 and c["scale"] == 1.0:
        from gnn_inputs.configs import _graph
        D = 64
        g = torch.Generator(device=dev).manual_seed(2)
        xf = torch.randn((n, D), device=dev, generator=g) * D ** -0.5
        o = torch.empty(n, device=dev)
        deg = np.diff(c["rowptr"].astype(np.int64))
        order = np.argsort(-deg, kind="stable")
        new_id = np.empty(n, np.int64)
        new_id[order] = np.arange(n)
        dst = np.repeat(np.arange(n, dtype=np.int64), deg)
        rp_s, ci_s = GI.csr_from_pairs(n, new_id[dst], new_id[c["colidx"]], self_loops=False, dedupe=False)
        _, (rp_n, ci_n) = _graph(3, 1.0, c["seed"], relabel=False)
        graphs = {"orig_random_ids": (c["rowptr"], c["colidx"]), "natural_rmat_ids": (rp_n, ci_n), "degree_sorted_ids": (rp_s, ci_s)}
        t = {}
        for gname, (rp, ci) in graphs.items():
            rpd, cid = torch.from_numpy(rp).to(dev), torch.from_numpy(ci).to(dev)
            for mode, mname in ((0, "feature"), (1, "neighbor")):
                for vec in (False, True):
                    t[f"{gname}/{mname}{'_vec' if vec else ''}"] = event_ms(lambda: G.gnn_dot_aggr(rpd, cid, xf, mode, vec, o), reps=2, warm=1)
            del rpd, cid
        gaps = {}
        for gname in ("natural_rmat_ids", "degree_sorted_ids"):
            for sfx in ("", "_vec"):
                s_f = t[f"orig_random_ids/feature{sfx}"] / t[f"{gname}/feature{sfx}"]
                s_n = t[f"orig_random_ids/neighbor{sfx}"] / t[f"{gname}/neighbor{sfx}"]
                gaps[f"{gname}{sfx}"] = {"s_feature": s_f, "s_neighbor": s_n, "delta_s": s_n - s_f}
        out["dot_aggr"] = {"dim": D, "dtype": "f32", "second_pass_ms": t, "reordering_gap": gaps,
                           "note": "METIS is not available: the reorderings are the generator's natural ids and a degree sort"}
    torch.cuda.empty_cache()
    return out


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 8:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        os.unlink(self.f.name)
        if not sm:   # region shorter than one sampling period: one synchronous query right after it
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=10).stdout
                parts = [x.strip() for x in out.strip().splitlines()[0].split(",")]
                sm, mx = [float(parts[0])], [float(parts[1])]
                for nm, val in zip(names, parts[4:8]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ oracle arm
def oracle_sample_pass(c, f32, rows, srcs, rp_t, ci_t):
    """One pass of the fp64 oracle over `rows` (forward + dst-side backward) and `srcs` (src-side backward).
    Returns seconds per stage.  L / Delta for destinations outside `rows` are placeholders in the src stage
    (timing only; these outputs are discarded)."""
    import oracle
    n, H = c["n"], c["heads"]
    rp, ci = c["rowptr"], c["colidx"]
    t = {}
    if c["layer"] == "gt":
        q, k, v, do = f32["q"], f32["k"], f32["v"], f32["do"]
        t0 = time.perf_counter()
        O, L = oracle.gt_forward(rp, ci, q, k, v, rows=rows)
        t["fwd"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        Dl = oracle.rowdot(O, do, rows=rows)
        Lf, Df = np.zeros((n, H)), np.zeros((n, H))
        Lf[rows], Df[rows] = L, Dl
        oracle.gt_backward_dst(rp, ci, q, k, v, do, Lf, Df, rows=rows)
        t["bwd_dst"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        oracle.gt_backward_src(rp_t, ci_t, q, k, v, do, Lf, Df, srcs=srcs)
        t["bwd_src"] = time.perf_counter() - t0
    else:
        xl, xr, a, do, sl = f32["xl"], f32["xr"], c["a_f32"], f32["do"], c["slope"]
        t0 = time.perf_counter()
        O, L = oracle.gatv2_forward(rp, ci, xl, xr, a, sl, rows=rows)
        t["fwd"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        Gv = oracle.rowdot(O, do, rows=rows)
        Lf, Gf = np.zeros((n, H)), np.zeros((n, H))
        Lf[rows], Gf[rows] = L, Gv
        oracle.gatv2_backward_dst(rp, ci, xl, xr, a, sl, do, Lf, Gf, rows=rows)
        t["bwd_dst"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        oracle.gatv2_backward_src(rp_t, ci_t, xl, xr, a, sl, do, Lf, Gf, srcs=srcs)
        t["bwd_src"] = time.perf_counter() - t0
    return t


class OracleArm:
    """Times oracle/ (as it stands) on a bounded sample: uniformly drawn destination rows for the forward and
    the dst-side backward, uniformly drawn source rows of the oracle's own CSR^T for the src-side backward.
    GEdges/s = 1 / (sum over the three stages of seconds per sampled edge)."""

    def __init__(self, c, target_seconds: float):
        import oracle
        from oracle import plan_ref
        oracle.build()
        self.c = c
        self.cores = oracle.num_threads()
        names = ("q", "k", "v", "do") if c["layer"] == "gt" else ("xl", "xr", "do")
        self.f32 = {}
        for nm in names:
            x = c.get(nm + "_f32")
            self.f32[nm] = x if x is not None else GI.bf16_bits_to_f32(c[nm + "_st"])
        self.rp_t, self.ci_t = plan_ref.transpose_csr(c["rowptr"], c["colidx"])
        rng = np.random.default_rng(12345)
        n = c["n"]
        self.order_r = rng.permutation(n).astype(np.int32)
        self.order_s = rng.permutation(n).astype(np.int32)
        self.deg_in = np.diff(c["rowptr"].astype(np.int64))
        self.deg_out = np.diff(self.rp_t.astype(np.int64))
        # calibrate the sample size on a small probe
        k = min(n, 2000)
        t = self.run(k, k)
        per_row = sum(t.values()) / k
        self.k = int(max(64, min(n, target_seconds / max(per_row, 1e-9))))

    def run(self, kr=None, ks=None):
        kr = self.k if kr is None else kr
        ks = self.k if ks is None else ks
        rows, srcs = np.sort(self.order_r[:kr]), np.sort(self.order_s[:ks])
        self.er, self.es = int(self.deg_in[rows].sum()), int(self.deg_out[srcs].sum())
        return oracle_sample_pass(self.c, self.f32, rows, srcs, self.rp_t, self.ci_t)

    def gedges(self, t) -> float:
        sec_per_edge = t["fwd"] / max(self.er, 1) + t["bwd_dst"] / max(self.er, 1) + t["bwd_src"] / max(self.es, 1)
        return 1e-9 / sec_per_edge

    def sample_text(self) -> str:
        return (f"{self.k} uniformly drawn dst rows ({self.er} edges: fwd + dst-side bwd) and {self.k} src rows "
                f"({self.es} edges: src-side bwd) of the full-size {self.c['name']} graph; per-edge stage times summed")


def max_over_ranks(x: float, world: int, device=None) -> float:
    """MAX of a per-rank scalar over the job (device time of the slowest rank)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_gedges(edges_per_rank: int, steps: int, world: int, total_ms: float) -> float:
    """Whole-job GEdges/s: every rank processed `edges_per_rank` edges per step (replicas, weak scaling)."""
    return world * edges_per_rank * steps / (total_ms * 1e-3) * 1e-9


def workload_config(c, args):
    return {"workload": c["name"], "layer": c["layer"], "nodes": c["n"], "edges": c["e"], "heads": c["heads"],
            "head_dim": c["head_dim"], "feature_dtype": c["dtype"], "scale": args.scale,
            "graph": "synthetic seeded generator (gnn_inputs), stands in for the paper's datasets",
            "ids": ("sorted by descending in-degree (locality experiment, not the headline)" if c.get("relabel") == "degree-sorted" else
                    "randomly relabelled" if c.get("relabel", True) else "natural R-MAT ids (locality study, not the headline)")}


def run_reference(args, rank):
    if rank != 0:
        return
    c = GI.make_config(args.cfg, scale=args.scale, keep_f32=False, relabel=not args.natural_ids, dense=args.dense)
    # each step = one bounded sample pass; the whole run (warm-up + steps) is sized to about two minutes of oracle time
    arm = OracleArm(c, target_seconds=min(args.cpu_seconds, 120.0 / max(args.steps + args.warmup, 1)))
    for _ in range(args.warmup):
        arm.run()
    t0 = time.perf_counter()
    vals = []
    for _ in range(args.steps):
        vals.append(arm.gedges(arm.run()))
    wall = time.perf_counter() - t0
    v = float(len(vals) / sum(1.0 / x for x in vals))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(c, args),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": arm.cores, "kind": "oracle", "sample": arm.sample_text()},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ CUDA arm
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist

    import paper_2605_31500_b200 as G
    import paper_2605_31500_b200.binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle arm)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    c = GI.make_config(args.cfg, scale=args.scale, keep_f32=False, relabel=not args.natural_ids, dense=args.dense)   # replicas: every rank runs the same workload
    if args.degree_sorted_ids:
        c = degree_sort_config(c)
    n, e, H, d, dt = c["n"], c["e"], c["heads"], c["head_dim"], c["dtype"]
    gt = c["layer"] == "gt"
    names = ("q", "k", "v", "do") if gt else ("xl", "xr", "do")

    def to_torch(a):
        t = torch.from_numpy(np.ascontiguousarray(a))
        return t.view(torch.bfloat16) if (dt == "bf16" and a.dtype == np.uint16) else t

    host = {nm: to_torch(c[nm + "_st"]) for nm in names}
    host["rowptr"], host["colidx"] = torch.from_numpy(c["rowptr"]), torch.from_numpy(c["colidx"])
    if not gt:
        host["a"] = torch.from_numpy(c["a_f32"])
    devt = {k: v.to(dev) for k, v in host.items()}
    torch.cuda.synchronize()
    # row f1: cfg 3 is undirected by construction, so its backward reuses the forward CSR (the
    # library verifies that); --directed-plan builds CSR^T instead.  Both plans are built and timed for cfg 3.
    undirected = args.cfg == 3 and not args.directed_plan

    def build_plan(mode):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        p = G.Plan(devt["rowptr"], devt["colidx"], warp_max_deg=args.warp_max_deg, cta_max_deg=args.cta_max_deg,
                   split_chunk=args.split_chunk, transpose=mode, blocks=(args.cfg == 4), wsb=(args.cfg == 4))
        torch.cuda.synchronize()
        return p, 1e3 * (time.perf_counter() - t0)

    plan_cmp = None
    if undirected:
        build_plan(True)            # untimed first build: module load, allocator warm-up
        p_dir, ms_dir = build_plan(True)
        plan_cmp = {"directed_plan_build_ms": ms_dir, "directed_plan_bytes": p_dir.plan_bytes}
        del p_dir
    plan, plan_ms = build_plan("undirected" if undirected else True)

    f32 = dict(dtype=torch.float32, device=dev)
    out = torch.empty((n, H, d), dtype=devt[names[0]].dtype, device=dev)
    lse, stat = torch.empty((n, H), **f32), torch.empty((n, H), **f32)
    g1, g2 = torch.empty((n, H, d), **f32), torch.empty((n, H, d), **f32)
    g3 = torch.empty((n, H, d), **f32) if gt else torch.empty((H, d), **f32)

    if gt:
        def fwd():
            G.gnn_gt_attn_fwd(plan, devt["q"], devt["k"], devt["v"], out, lse)

        def bwd():
            G.gnn_gt_attn_bwd(plan, devt["q"], devt["k"], devt["v"], lse, devt["do"], stat, g1, g2, g3)
    else:
        def fwd():
            G.gnn_gatv2_fwd(plan, devt["xl"], devt["xr"], devt["a"], c["slope"], out, lse)

        def bwd():
            G.gnn_gatv2_bwd(plan, devt["xl"], devt["xr"], devt["a"], lse, devt["do"], c["slope"], stat, g1, g2, g3)

    def step():
        fwd()
        bwd()

    def fwd_block():   # cfg 4 only: tcgen05/TMEM block-sparse forward (row a12); writes the same out / lse
        G.gnn_gt_attn_fwd_block(plan, devt["q"], devt["k"], devt["v"], out, lse)

    in_bytes = sum(int(v.numel()) * v.element_size() for v in host.values())
    outs = [out, lse, stat, g1, g2, g3]
    out_bytes = sum(int(v.numel()) * v.element_size() for v in outs)
    l2_bytes = torch.cuda.get_device_properties(dev).L2_cache_size
    need_flush = in_bytes < 4 * l2_bytes
    flush = torch.empty(max(2 * l2_bytes, 1 << 28), dtype=torch.uint8, device=dev) if need_flush else None

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, k):
        """sum of per-step CUDA-event times (ms); L2 flushed between steps (outside the events) for small inputs"""
        evs = []
        for _ in range(k):
            if flush is not None:
                flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            evs.append((a, b))
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    l2win = None
    if args.l2_window > 0:
        kt = devt["k" if gt else "xr"]
        l2win = set_l2_window(kt.data_ptr(), int(args.l2_window * 1e6), torch.cuda.current_stream().cuda_stream,
                              int(min(args.l2_window * 1e6 * 1.25, 0.75 * l2_bytes)))
        l2win["tensor"] = "k" if gt else "xr"
    clocks = ClockSampler(local_rank)     # sampled every 100 ms from the warm-up to the end of the timed regions
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    l0 = G.gnn_launch_count()
    ms_steps = timed(step, args.steps)
    launches = G.gnn_launch_count() - l0
    barrier()
    ms_fwd = timed(fwd, args.steps)
    ms_bwd = timed(bwd, args.steps)
    clk = clocks.stop()
    total_ms = max_over_ranks(float(sum(ms_steps)), world, dev)
    value = job_gedges(e, args.steps, world, total_ms)

    peak_mem = int(torch.cuda.max_memory_allocated(dev))   # the layer itself: inputs, outputs, plan, workspace (+ L2 flush buffer)

    def fwd_wsb():     # cfg 4 only: general WSB layout, tcgen05 forward (row f2)
        G.gnn_gt_attn_fwd_wsb(plan, devt["q"], devt["k"], devt["v"], out, lse)

    def bwd_wsb():     # cfg 4 only: tensor-core backward on the WSB layouts of the CSR and of CSR^T (row f2)
        G.gnn_gt_attn_bwd_wsb(plan, devt["q"], devt["k"], devt["v"], out, lse, devt["do"], stat, g1, g2, g3)

    wsb = None
    if args.cfg == 4:
        for _ in range(3):
            fwd_wsb()
            bwd_wsb()
        ms_wf, ms_wb = timed(fwd_wsb, args.steps), timed(bwd_wsb, args.steps)
        G.gnn_profile_enable(True)
        fwd_wsb()
        bwd_wsb()
        G.gnn_profile_enable(False)
        wk = {nm: float(ms) for nm, ms in G.gnn_profile_collect(64)}
        wsb = {"ms_fwd": float(np.mean(ms_wf)), "ms_bwd": float(np.mean(ms_wb)), "kernels_ms": wk, "info": plan.wsb_info()}
        fwd()   # restore the CSR forward's out / lse for what follows

    def bwd_block():   # cfg 4 only: tensor-core backward on the diagonal block layout (+ remainder CSR passes)
        G.gnn_gt_attn_bwd_block(plan, devt["q"], devt["k"], devt["v"], lse, devt["do"], stat, g1, g2, g3)

    block = None
    if args.cfg == 4:
        for _ in range(3):
            fwd_block()
            bwd_block()
        ms_blk = timed(fwd_block, args.steps)
        ms_bblk = timed(bwd_block, args.steps)
        ms_sblk = timed(lambda: (fwd_block(), bwd_block()), args.steps)
        G.gnn_profile_enable(True)
        fwd_block()
        bwd_block()
        G.gnn_profile_enable(False)
        bk = {nm: float(ms) for nm, ms in G.gnn_profile_collect(64)}
        block = {"ms_fwd": float(np.mean(ms_blk)), "gedges_fwd": e / (np.mean(ms_blk) * 1e-3) * 1e-9,
                 "ms_bwd": float(np.mean(ms_bblk)), "ms_step": float(np.mean(ms_sblk)),
                 "gedges_step": e / (np.mean(ms_sblk) * 1e-3) * 1e-9, "kernels_ms": bk}

    # ---- cfg 1 / 2 are launch-bound (a step is 7-9 launches of a few microseconds each): the same step captured
    # once in a CUDA graph of 100 back-to-back layers and replayed (SURVEY 8(d) timing protocol).  Warm L2 by
    # construction (the working set fits), so it is reported beside `value`, never instead of it.
    graph = None
    if args.cfg in (1, 2) and world == 1:
        layers = 100
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            step()
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        cg = torch.cuda.CUDAGraph()
        with torch.cuda.graph(cg):
            for _ in range(layers):
                step()
        cg.replay()
        ms_graph = timed(cg.replay, max(args.steps, 5))
        ms_layer = float(np.mean(ms_graph)) / layers
        graph = {"layers_per_graph": layers, "ms_per_step": ms_layer, "gedges": e / (ms_layer * 1e-3) * 1e-9,
                 "l2": "warm (back-to-back layers on an L2-resident working set)"}

    # ---- per-kernel device times (library event profiler), same inputs, right after the timed region
    G.gnn_profile_enable(True)
    for _ in range(args.steps):
        if flush is not None:
            flush.zero_()
        step()
    G.gnn_profile_enable(False)
    recs = G.gnn_profile_collect(64 * args.steps + 64)
    kern = {}
    for nm, ms in recs:
        kern.setdefault(nm, []).append(ms)
    kern_ms = {k: float(np.mean(v)) for k, v in kern.items()}

    # ---- byte model and rooflines
    cnt = plan.counts()
    perm, perm_t = plan.export(B.GNN_PLAN_PERM), plan.export(B.GNN_PLAN_PERM_T)
    deg_in = np.diff(c["rowptr"].astype(np.int64))
    deg_out = np.diff(plan.export(B.GNN_PLAN_ROWPTR_T).astype(np.int64))
    alg, comp = byte_model(c, cnt, deg_in, deg_out, perm, perm_t)
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peak, peak_src = float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak, peak_src = FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"
    bf16_peak = None
    if os.path.exists(peaks_path):
        bf16_peak = json.load(open(peaks_path)).get("bf16_tflops")
    traffic, tfile = None, None
    for tname in ("r02_dram_traffic.json", "r01_dram_traffic.json"):      # ncu captures of this build, else of round 1
        tpath = os.path.join(ROOT, "profiles", tname)
        if traffic is None and os.path.exists(tpath) and args.scale == 1.0 and not (args.warp_max_deg or args.cta_max_deg or args.split_chunk):
            tj = json.load(open(tpath))
            if c["name"] in tj:
                traffic, tfile = tj[c["name"]], "profiles/" + tname
    dom = max((k for k in kern_ms if k in alg), key=lambda k: kern_ms[k])
    achieved = alg[dom] / (kern_ms[dom] * 1e-3) * 1e-9
    step_ms = total_ms / args.steps
    comp_step = comp["fwd"] + comp["bwd"]
    dom_traffic = (traffic or {}).get(dom)
    roof = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "frac_meaning": "ALGORITHMIC bytes of the dominant kernel (index + gathered rows per edge, SURVEY 8(d)) / its "
                            "live CUDA-event time / measured HBM copy peak.  Gathers that hit L2 count, so this is NOT a DRAM "
                            "utilisation and can exceed 1; `dram_frac` is the DRAM utilisation, `north_star` the graded figure",
            "traffic": dom_traffic,
            "traffic_source": (f"ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, offline capture ({tfile}); "
                               "not measured in this run") if traffic else None,
            "dram_frac": (dom_traffic / (kern_ms[dom] * 1e-3) * 1e-9 / peak) if dom_traffic else None,
            "traffic_over_compulsory_step": (sum(v for k, v in traffic.items() if k in kern_ms) / comp_step) if traffic else None,
            "north_star": {"what": "compulsory bytes (each array once) / step time / measured HBM peak", "target": 0.60,
                           "value": comp_step / (step_ms * 1e-3) * 1e-9 / peak},
            "kernels_traffic": traffic or None,
            "peak_source": peak_src, "algorithmic_bytes_per_launch": alg[dom],
            "kernel_ms": kern_ms[dom], "kernel_share_of_step": kern_ms[dom] / sum(kern_ms.values()),
            "kernels_ms": kern_ms,
            "kernels_algorithmic_gbs": {k: alg[k] / (kern_ms[k] * 1e-3) * 1e-9 for k in kern_ms if k in alg and kern_ms[k] > 0},
            "compulsory": {"bytes_fwd": comp["fwd"], "bytes_bwd": comp["bwd"],
                           "gbs_fwd": comp["fwd"] / (np.mean(ms_fwd) * 1e-3) * 1e-9,
                           "gbs_bwd": comp["bwd"] / (np.mean(ms_bwd) * 1e-3) * 1e-9,
                           "gbs_step": comp_step / (step_ms * 1e-3) * 1e-9,
                           "frac_fwd": comp["fwd"] / (np.mean(ms_fwd) * 1e-3) * 1e-9 / peak,
                           "frac_bwd": comp["bwd"] / (np.mean(ms_bwd) * 1e-3) * 1e-9 / peak,
                           "frac_step": comp_step / (step_ms * 1e-3) * 1e-9 / peak}}

    # third ceiling: plain fp32 ALUs.  Useful flops per (edge, head), d = head_dim, one exp counted as 1:
    # GT fwd 5d+1 (Eq. 3), bwd dst 8d (one-sweep form), bwd src 8d; GATv2 fwd 7d+1 (Eq. 4), bwd dst 15d,
    # bwd src 11d.  Peak = SMs x 128 fp32 lanes x 2 flop x the SM clock sampled during the timed region.
    fl = {"fwd": (5 * d + 1) if gt else (7 * d + 1), "bwd": (16 * d) if gt else (26 * d)}
    sm_clk = float(clk.get("sm_mhz") or clk.get("sm_max_mhz") or 1965.0)
    alu_peak = torch.cuda.get_device_properties(dev).multi_processor_count * 128 * 2 * sm_clk * 1e6 * 1e-12   # TFLOP/s
    tf_fwd = e * H * fl["fwd"] / (np.mean(ms_fwd) * 1e-3) * 1e-12
    tf_bwd = e * H * fl["bwd"] / (np.mean(ms_bwd) * 1e-3) * 1e-12
    roof["fp32_alu"] = {"flop_per_edge_head_fwd": fl["fwd"], "flop_per_edge_head_bwd": fl["bwd"], "peak_tflops": alu_peak,
                        "sm_mhz": sm_clk, "tflops_fwd": tf_fwd, "tflops_bwd": tf_bwd,
                        "frac_fwd": tf_fwd / alu_peak, "frac_bwd": tf_bwd / alu_peak}
    extras = {}
    if world == 1 and not args.no_extras:
        gc = gather_ceilings(H * d * (4 if dt == "f32" else 2), dev)
        roof["gather_ceiling"] = gc
        # the dominant kernel's row ingest against the probe at the occupancy the kernels run at: an L2-hit-weighted mix
        # of the two tables bounds it (the kernels see ~40-60 % L2 hits, profiles/)
        roof["frac_of_gather_ceiling"] = {"vs_hbm_resident_16warps": achieved / gc["hbm_resident"]["ldg_16warps_gbs"],
                                          "vs_l2_resident_16warps": achieved / gc["l2_resident"]["ldg_16warps_gbs"],
                                          "vs_hbm_resident_32warps": achieved / gc["hbm_resident"]["ldg_32warps_gbs"],
                                          "vs_l2_resident_32warps": achieved / gc["l2_resident"]["ldg_32warps_gbs"]}
        extras = block_extras(c, dev, peak, bf16_peak)
    fr = {"hbm_compulsory": roof["north_star"]["value"], "hbm_dram_traffic_dominant_kernel": roof["dram_frac"],
          "fp32_alu": max(roof["fp32_alu"]["frac_fwd"], roof["fp32_alu"]["frac_bwd"]),
          "gather_ingest_hbm_resident_16warps": (roof.get("frac_of_gather_ceiling") or {}).get("vs_hbm_resident_16warps")}
    known = {k: v for k, v in fr.items() if v is not None}
    top = max(known, key=known.get)
    roof["binding"] = {"fractions": fr, "largest": top,
                       "reading": ("no ceiling is saturated: the traversal kernels are latency-bound at register-limited occupancy "
                                   "(12-16 warps/SM); the closest ceiling is the gather ingest of random rows at that occupancy "
                                   "(profiles/r02_csr_experiments.md); the compulsory-byte fraction misses north_star's 0.60 because the "
                                   "per-edge gathers move 5-13x the compulsory bytes through L2 / DRAM")}

    if block is not None:
        rem = int(plan.export(B.GNN_PLAN_BLOCK_REM_ROWPTR)[-1])
        b_el = 2
        # algorithmic bytes of the block kernel: Q, K, V tiles once, O, L, bitmaps, remainder index + gathered K_j, V_j
        blk_bytes = 4 * n * H * d * b_el + 4 * n * H + 2 * n + 4 * (n + 1) + rem * (4 + 2 * H * d * b_el)
        tp = (traffic or {}).get("gt_fwd_block/tile_tensor_pipe_pct") if traffic else None
        ms_mixed = block["ms_fwd"] + float(np.mean(ms_bwd))    # block forward + CSR backward (the paper's own fallback)
        block.update({"ms_step_block_fwd_csr_bwd": ms_mixed, "gedges_step_block_fwd_csr_bwd": e / (ms_mixed * 1e-3) * 1e-9,
                      "csr_ms_fwd": float(np.mean(ms_fwd)), "speedup_vs_csr_fwd": float(np.mean(ms_fwd) / block["ms_fwd"]),
                      "remainder_edges": rem, "algorithmic_bytes": blk_bytes,
                      "achieved_gbs": blk_bytes / (block["ms_fwd"] * 1e-3) * 1e-9,
                      "frac_of_hbm_peak": blk_bytes / (block["ms_fwd"] * 1e-3) * 1e-9 / peak,
                      "compulsory_frac_fwd": comp["fwd"] / (block["ms_fwd"] * 1e-3) * 1e-9 / peak,
                      "traffic": (traffic or {}).get("gt_fwd_block/tile") if traffic else None,
                      "tensor_pipe_pct_of_peak": tp})

    # ---- row f3: degree-aware min aggregation with argmin on the same graph and plan, x = the K / xr tensor
    # viewed as [n, H*d], dout = the config's upstream gradient; an extra object, not part of `value`
    minmax = None
    if args.cfg in (3, 5) and not args.no_minmax:
        x2 = devt["k" if gt else "xr"].view(n, H * d)
        do2 = devt["do"].view(n, H * d)
        mo, ma = torch.empty_like(x2), torch.empty((n, H * d), dtype=torch.int32, device=dev)
        mdx = torch.empty((n, H * d), **f32)

        def mm_fwd():
            G.gnn_seg_minmax_fwd(plan, x2, G.GNN_AGG_MIN, mo, ma)

        def mm_bwd():
            G.gnn_seg_minmax_bwd(ma, do2, mdx)

        for _ in range(3):
            mm_fwd()
            mm_bwd()
        ms_mf, ms_mb = timed(mm_fwd, args.steps), timed(mm_bwd, args.steps)
        G.gnn_profile_enable(True)
        mm_fwd()
        mm_bwd()
        G.gnn_profile_enable(False)
        mk = {nm: float(ms) for nm, ms in G.gnn_profile_collect(64)}
        b_el = x2.element_size()
        R = H * d
        # forward: index + one gathered row per edge; per row perm, rowptr, out row, arg row.  backward: arg + dout read,
        # dx zeroed and one 32-byte sector read-modify-written per 8 scattered floats at best (counted as 4 B read + 4 B write)
        mm_fwd_bytes = e * (4 + R * b_el) + n * (8 + R * b_el + 4 * R)
        mm_bwd_bytes = n * R * (4 + b_el + 4 + 8)
        minmax = {"op": "seg_min + argmin (row f3)", "channels": R, "ms_fwd": float(np.mean(ms_mf)), "ms_bwd": float(np.mean(ms_mb)),
                  "gedges_fwd": e / (np.mean(ms_mf) * 1e-3) * 1e-9, "kernels_ms": mk,
                  "algorithmic_bytes_fwd": mm_fwd_bytes, "achieved_gbs_fwd": mm_fwd_bytes / (np.mean(ms_mf) * 1e-3) * 1e-9,
                  "frac_of_hbm_peak_fwd": mm_fwd_bytes / (np.mean(ms_mf) * 1e-3) * 1e-9 / peak,
                  "algorithmic_bytes_bwd": mm_bwd_bytes, "achieved_gbs_bwd": mm_bwd_bytes / (np.mean(ms_mb) * 1e-3) * 1e-9,
                  "frac_of_hbm_peak_bwd": mm_bwd_bytes / (np.mean(ms_mb) * 1e-3) * 1e-9 / peak}
        del mo, ma, mdx

    # ---- end to end: pinned host inputs -> device, step, every output -> pinned host, all inside the timed region.
    # Three streams (H2D, compute, D2H) and two sets of device feature / output buffers, so the copies of step k+1
    # and k-1 overlap the kernels of step k (PCIe is full duplex); the CSR goes into the plan's own buffers once the
    # previous step's kernels are done.  Time = first H2D start -> last D2H end, pipeline fill and drain included.
    e2e = None
    if args.e2e_steps > 0:
        ksteps = args.e2e_steps
        pin_in = {k: v.pin_memory() for k, v in host.items()}
        pin_out = [torch.empty(o.shape, dtype=o.dtype, pin_memory=True) for o in outs]
        feat = [k for k in host if k not in ("rowptr", "colidx")]
        dsets = [devt, {**devt, **{k: torch.empty_like(devt[k]) for k in feat}}]
        osets = [outs, [torch.empty_like(o) for o in outs]]
        s_in, s_c, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()

        def step_on(D, O):
            o_, l_, st_, a1, a2, a3 = O
            if gt:
                G.gnn_gt_attn_fwd(plan, D["q"], D["k"], D["v"], o_, l_)
                G.gnn_gt_attn_bwd(plan, D["q"], D["k"], D["v"], l_, D["do"], st_, a1, a2, a3)
            else:
                G.gnn_gatv2_fwd(plan, D["xl"], D["xr"], D["a"], c["slope"], o_, l_)
                G.gnn_gatv2_bwd(plan, D["xl"], D["xr"], D["a"], l_, D["do"], c["slope"], st_, a1, a2, a3)

        def e2e_run(k):
            ev_in, ev_c, ev_out = [], [], []
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(s_in):
                t0.record()
            for i in range(k):
                D, O = dsets[i % 2], osets[i % 2]
                with torch.cuda.stream(s_in):
                    if i >= 2:
                        s_in.wait_event(ev_c[i - 2])          # feature set i % 2 is free again
                    for k2 in feat:
                        D[k2].copy_(pin_in[k2], non_blocking=True)
                    if i >= 1:
                        s_in.wait_event(ev_c[i - 1])          # the CSR buffers are the plan's: no kernel may be reading
                    for k2 in ("rowptr", "colidx"):
                        D[k2].copy_(pin_in[k2], non_blocking=True)
                    ev_in.append(torch.cuda.Event()); ev_in[-1].record()
                with torch.cuda.stream(s_c):
                    s_c.wait_event(ev_in[i])
                    if i >= 2:
                        s_c.wait_event(ev_out[i - 2])         # output set i % 2 has been read back
                    step_on(D, O)
                    ev_c.append(torch.cuda.Event()); ev_c[-1].record()
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_c[i])
                    for po, o in zip(pin_out, O):
                        po.copy_(o, non_blocking=True)
                    ev_out.append(torch.cuda.Event()); ev_out[-1].record()
            with torch.cuda.stream(s_out):
                t1.record()
            torch.cuda.synchronize()
            return t0.elapsed_time(t1)

        barrier()
        e2e_run(2)
        barrier()
        t_e2e = max_over_ranks(float(e2e_run(ksteps)), world, dev)
        e2e = {"value": job_gedges(e, ksteps, world, t_e2e), "unit": UNIT,
               "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": out_bytes, "steps": ksteps,
               "ms_per_step": t_e2e / ksteps,
               "pipeline": "3 streams, double-buffered features and outputs; fill and drain inside the timed region"}
        del pin_in, pin_out, dsets, osets

    all_cfg = None
    if rank == 0 and world == 1 and args.cfg == 3 and args.scale == 1.0 and not args.no_all_configs and not args.dense:
        all_cfg = {}
        for other in (1, 2, 4, 5):
            all_cfg[f"cfg{other}"] = quick_config(other, args, dev, peak)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        arm = OracleArm(c, args.cpu_seconds)
        cpu = {"value": arm.gedges(arm.run()), "unit": UNIT, "cores": arm.cores, "kind": "oracle", "sample": arm.sample_text(),
               "edges_timed_dst_side": arm.er, "edges_timed_src_side": arm.es, "edges_total": e,
               "fraction_of_edges_timed": {"dst_side": arm.er / e, "src_side": arm.es / e}}

    if rank == 0:
        cfgd = workload_config(c, args)
        cfgd.update({"l2": "L2 flushed between timed steps" if need_flush else "inputs larger than L2 (no flush)",
                     "plan": cnt, "plan_opts": {"warp_max_deg": plan.opts.warp_max_deg, "cta_max_deg": plan.opts.cta_max_deg,
                                                "split_chunk": plan.opts.split_chunk},
                     "plan_build_ms": plan_ms, "l2_window": l2win,
                     "backward_csr": "forward CSR reused (undirected graph, PAPER.md:343)" if undirected else "CSR^T built by the plan",
                     "plan_vs_directed": plan_cmp, "degree_stats": GI.degree_stats(c["rowptr"], c["colidx"])})
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": cfgd,
                "ms_fwd": float(np.mean(ms_fwd)), "ms_bwd": float(np.mean(ms_bwd)),
                "gedges_fwd": e / (np.mean(ms_fwd) * 1e-3) * 1e-9, "gedges_bwd": e / (np.mean(ms_bwd) * 1e-3) * 1e-9,
                "peak_device_bytes": peak_mem, "device_bytes_inputs": in_bytes, "device_bytes_outputs": out_bytes,
                "plan_bytes": plan.plan_bytes, "clocks": clk, "e2e": e2e, "gpu_launches": int(launches),
                "roofline": roof, "block_path": block, "wsb_path": wsb, "all_configs": all_cfg,
                "ln_qkv": extras.get("ln_qkv"), "dot_aggr": extras.get("dot_aggr"), "cuda_graph": graph, "seg_minmax": minmax, "cpu_baseline": cpu}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
