"""Full-size parity (BASELINE.json sizes, default plan = the launch configuration bench.py times).

EVERY output element of every config is compared with the fp64 oracle: the oracle is evaluated in row chunks
(destination rows for O, L, Delta / G, dQ / dxl and the per-row da terms; source rows of the oracle's own CSR^T for
dK, dV / dxr), the error norms are accumulated per output tensor and the north_star tolerances are applied to the
whole tensor at the end.  da - the one output that sums over every edge with cancellation - is compared element by
element with the sum of the oracle's per-row terms.  Plus the conservation identities that hold at any size
(SURVEY.md section 8(c)), the plan metadata bit-exact on the full graph, and the O(N*H*d) memory assertions."""
import numpy as np
import pytest

import gnn_inputs as GI
import oracle
from oracle import plan_ref
from test_gpu_parity import check, _dev, DEFAULT_OPTS

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

CHUNK = 400_000     # rows per oracle call


def _f32(c, nm):
    x = c.get(nm + "_f32")
    return x if x is not None else GI.bf16_bits_to_f32(c[nm + "_st"])


class TensorErr:
    """north_star's per-tensor criteria accumulated over row chunks: max-abs <= 1e-4 (fp32 features); max-abs <= 2e-2
    AND relative Frobenius <= 5e-3 (bf16 features); non-finite pattern (L of empty rows) must match exactly."""

    def __init__(self, name, dtype):
        self.name, self.dtype, self.mx, self.e2, self.w2, self.count = name, dtype, 0.0, 0.0, 0.0, 0

    def add(self, got, want):
        got, want = np.asarray(got, np.float64), np.asarray(want, np.float64)
        assert got.shape == want.shape, self.name
        fin = np.isfinite(want)
        assert np.array_equal(np.isfinite(got), fin), f"{self.name}: non-finite pattern differs"
        assert np.array_equal(got[~fin], want[~fin]), f"{self.name}: inf values differ"
        err = got[fin] - want[fin]
        if err.size:
            self.mx = max(self.mx, float(np.abs(err).max()))
        self.e2 += float((err * err).sum())
        self.w2 += float((want[fin] ** 2).sum())
        self.count += int(err.size)

    def finish(self, expect_count):
        assert self.count == expect_count, f"{self.name}: compared {self.count} of {expect_count} elements"
        rel = (self.e2 / self.w2) ** 0.5 if self.w2 > 0 else 0.0
        if self.dtype == "f32":
            assert self.mx <= 1e-4, f"{self.name}: max abs err {self.mx:.3e} > 1e-4"
        else:
            assert self.mx <= 2e-2, f"{self.name}: max abs err {self.mx:.3e} > 2e-2"
            assert rel <= 5e-3, f"{self.name}: rel Frobenius err {rel:.3e} > 5e-3"
        return self.mx, rel


@pytest.mark.parametrize("cfg", [2, 3, 4, 5])
def test_fullsize_sampled_parity(cfg):
    import torch
    import paper_2605_31500_b200 as G
    import paper_2605_31500_b200.binding as B
    c = GI.make_config(cfg, keep_f32=False)
    n, H, d, dt, gt = c["n"], c["heads"], c["head_dim"], c["dtype"], c["layer"] == "gt"
    rp, ci = torch.from_numpy(c["rowptr"]).cuda(), torch.from_numpy(c["colidx"]).cuda()
    # cfg 3 is undirected: same launch configuration as bench.py (backward over the forward CSR, row f1)
    plan = G.Plan(rp, ci, transpose="undirected" if cfg == 3 else True, blocks=(cfg == 4), **DEFAULT_OPTS)
    assert plan.undirected() == (cfg == 3)
    names = ("q", "k", "v", "do") if gt else ("xl", "xr", "do")
    T = {nm: _dev(c[nm + "_st"], dt) for nm in names}
    out = torch.empty_like(T[names[0]])
    lse = torch.empty((n, H), dtype=torch.float32, device="cuda")
    stat = torch.empty_like(lse)
    g1, g2 = (torch.empty((n, H, d), dtype=torch.float32, device="cuda") for _ in range(2))
    # saved state and workspace are O(N*H*d), never O(E*H): the library allocates nothing, the
    # binding allocates only the workspace the library asks for, and that is far below one E x H fp32 tensor
    code = B.GNN_BF16 if dt == "bf16" else B.GNN_F32
    ops = (B.GNN_OP_GT_FWD, B.GNN_OP_GT_BWD) if gt else (B.GNN_OP_GATV2_FWD, B.GNN_OP_GATV2_BWD)
    ws_need = max(G.gnn_workspace_bytes(plan.handle, op, H, d, code) for op in ops)
    assert ws_need <= 4 * n * H * d                      # at most one [n,H,d] fp32 tensor
    if c["e"] >= 20 * n:                                 # cfg 3 / 5: a small fraction of one E x H fp32 tensor
        assert ws_need <= 0.1 * (4 * c["e"] * H)
    torch.cuda.synchronize()
    torch.cuda.reset_peak_memory_stats()
    mem0 = torch.cuda.memory_allocated()
    if gt:
        g3 = torch.empty((n, H, d), dtype=torch.float32, device="cuda")
        G.gnn_gt_attn_fwd(plan, T["q"], T["k"], T["v"], out, lse)
        G.gnn_gt_attn_bwd(plan, T["q"], T["k"], T["v"], lse, T["do"], stat, g1, g2, g3)
    else:
        a = torch.from_numpy(c["a_f32"]).cuda()
        g3 = torch.empty((H, d), dtype=torch.float32, device="cuda")
        G.gnn_gatv2_fwd(plan, T["xl"], T["xr"], a, c["slope"], out, lse)
        G.gnn_gatv2_bwd(plan, T["xl"], T["xr"], a, lse, T["do"], c["slope"], stat, g1, g2, g3)
    torch.cuda.synchronize()
    extra = torch.cuda.max_memory_allocated() - mem0 - g3.numel() * 4
    assert extra <= ws_need + (4 << 20), f"forward + backward allocated {extra} bytes beyond the workspace ({ws_need})"

    # ---- metadata, bit-exact on the full graph
    rp_t, ci_t = plan_ref.transpose_csr(c["rowptr"], c["colidx"])
    assert np.array_equal(plan.export(B.GNN_PLAN_ROWPTR_T), rp_t)
    assert np.array_equal(plan.export(B.GNN_PLAN_COLIDX_T), ci_t)
    cnt = plan.counts()
    ref = plan_ref.build_bins(c["rowptr"], *_resolved_opts(c["e"]))
    assert np.array_equal(plan.export(B.GNN_PLAN_PERM), ref["perm"])
    assert np.array_equal(plan.export(B.GNN_PLAN_CHUNKS).reshape(-1, 4), ref["chunks"])
    ref_t = plan_ref.build_bins(rp_t, *_resolved_opts(c["e"]))
    assert np.array_equal(plan.export(B.GNN_PLAN_PERM_T), ref_t["perm"])
    assert np.array_equal(plan.export(B.GNN_PLAN_CHUNKS_T).reshape(-1, 4), ref_t["chunks"])
    assert cnt["n_chunks"] == ref["chunks"].shape[0] and cnt["n_chunks_t"] == ref_t["chunks"].shape[0]

    # ---- conservation identities on the full outputs (fp64 sums on the device)
    do64 = T["do"].double()
    sum_do = do64.sum(0)
    if gt:
        dq, dk, dv = g1.double(), g2.double(), g3.double()
        scale = float(do64.abs().sum(0).max())
        assert float((dv.sum(0) - sum_do).abs().max()) <= 1e-5 * scale + 1e-3
        lhs = float((T["q"].double() * dq).sum())
        rhs = float((T["k"].double() * dk).sum())
        den = float((T["q"].double() * dq).abs().sum())
        assert abs(lhs - rhs) <= 1e-5 * den
    else:
        dxl, dxr = g1.double(), g2.double()
        scale = float(do64.abs().sum(0).max())
        assert float((dxr.sum(0) - dxl.sum(0) - sum_do).abs().max()) <= 1e-5 * scale + 1e-3

    # ---- every bin the plan has is exercised by construction (all rows are compared); say what this graph covers
    if cfg in (3, 5):
        assert cnt["n_hub"] > 0 and cnt["n_cta"] > 0 and cnt["n_group"] > 0 and cnt["n_chunks"] > cnt["n_hub"]
        assert cnt["n_cta_t"] > 0 and cnt["n_group_t"] > 0
    if cfg == 5:
        assert cnt["n_chunks"] >= 733          # the 3 M-edge hub alone is 733 chunks of <= 4096 edges

    # ---- the whole output against the oracle, chunk by chunk
    f = {nm: _f32(c, nm) for nm in names}
    host = lambda t, lo, hi: t[lo:hi].float().cpu().numpy().astype(np.float64)
    Lf, Sf = np.empty((n, H)), np.empty((n, H))                 # oracle L and Delta / G of every destination
    keys_dst = ("O", "L", "Delta", "dQ") if gt else ("O", "L", "G", "dxl")
    keys_src = ("dK", "dV") if gt else ("dxr",)
    E = {k: TensorErr(f"cfg{cfg}:{k}", dt) for k in keys_dst + keys_src}
    da_ref = np.zeros((H, d))
    out_b = lse_b = None
    if cfg == 4:   # row a12 at full size: the tcgen05 block path on the same inputs, every row against the oracle
        out_b, lse_b = torch.full_like(out, float("nan")), torch.full_like(lse, float("nan"))
        G.gnn_gt_attn_fwd_block(plan, T["q"], T["k"], T["v"], out_b, lse_b)
        torch.cuda.synchronize()
        assert float((out_b.float() - out.float()).abs().max()) <= 4e-2     # two bf16 roundings of nearby values
        assert float((lse_b - lse).abs().max()) <= 1e-3
        E["block:O"], E["block:L"] = TensorErr(f"cfg{cfg}:block:O", dt), TensorErr(f"cfg{cfg}:block:L", dt)
    for lo in range(0, n, CHUNK):
        hi = min(n, lo + CHUNK)
        rows = np.arange(lo, hi, dtype=np.int32)
        if gt:
            O, L = oracle.gt_forward(c["rowptr"], c["colidx"], f["q"], f["k"], f["v"], rows=rows)
        else:
            O, L = oracle.gatv2_forward(c["rowptr"], c["colidx"], f["xl"], f["xr"], c["a_f32"], c["slope"], rows=rows)
        S = oracle.rowdot(O, f["do"], rows=rows)
        Lf[lo:hi], Sf[lo:hi] = L, S
        E["O"].add(host(out, lo, hi), O)
        E["L"].add(host(lse, lo, hi), L)
        E[keys_dst[2]].add(host(stat, lo, hi), S)
        if out_b is not None:
            E["block:O"].add(host(out_b, lo, hi), O)
            E["block:L"].add(host(lse_b, lo, hi), L)
        del O
    Lz = np.where(np.isfinite(Lf), Lf, 0.0)                      # empty rows have no entries: their L is never read
    for lo in range(0, n, CHUNK):
        hi = min(n, lo + CHUNK)
        rows = np.arange(lo, hi, dtype=np.int32)
        if gt:
            dQ = oracle.gt_backward_dst(c["rowptr"], c["colidx"], f["q"], f["k"], f["v"], f["do"], Lz, Sf, rows=rows)
            E["dQ"].add(host(g1, lo, hi), dQ)
        else:
            dxl, da_rows = oracle.gatv2_backward_dst(c["rowptr"], c["colidx"], f["xl"], f["xr"], c["a_f32"], c["slope"],
                                                     f["do"], Lz, Sf, rows=rows)
            E["dxl"].add(host(g1, lo, hi), dxl)
            da_ref += da_rows.sum(axis=0)
            del da_rows
    for lo in range(0, n, CHUNK):
        hi = min(n, lo + CHUNK)
        srcs = np.arange(lo, hi, dtype=np.int32)
        if gt:
            dK, dV = oracle.gt_backward_src(rp_t, ci_t, f["q"], f["k"], f["v"], f["do"], Lz, Sf, srcs=srcs)
            E["dK"].add(host(g2, lo, hi), dK)
            E["dV"].add(host(g3, lo, hi), dV)
        else:
            dxr = oracle.gatv2_backward_src(rp_t, ci_t, f["xl"], f["xr"], c["a_f32"], c["slope"], f["do"], Lz, Sf, srcs=srcs)
            E["dxr"].add(host(g2, lo, hi), dxr)
    report = {}
    for k, te in E.items():
        report[k] = te.finish(n * H * (1 if k.endswith("L") or k in ("Delta", "G") else d))
    if not gt:
        # da [H, d]: a sum over all E edges with cancellation (fp32 per CTA, fp64 across CTAs in the kernel)
        check(f"cfg{cfg}:da", g3.cpu().numpy(), da_ref, dt)
        report["da"] = float(np.abs(g3.cpu().numpy() - da_ref).max())
    print(f"cfg{cfg} full-size (max abs, rel Frobenius):", {k: (f"{v[0]:.2e}", f"{v[1]:.2e}") if isinstance(v, tuple) else f"{v:.2e}"
                                                             for k, v in report.items()})


def _resolved_opts(nnz):
    """the library's default thresholds (include/gnn_attn.h)"""
    return (4096, 16384, 4096) if nnz >= (1 << 24) else (256, 1024, 512)
