"""GPU parity for SURVEY section 8 row f3: degree-aware min / max aggregation with argmin
through the C ABI vs ``oracle/agg_ref.py``.  The forward selects values and indices, so it is compared BIT-EXACTLY
(out is a copy of an input element, arg an integer with a fixed tie rule); the backward is an fp32 scatter-add whose
addition order is not fixed: max-abs <= 1e-4 relative to the largest gradient magnitude."""
import numpy as np
import pytest

import gnn_inputs as GI
from oracle import agg_ref
from test_gpu_parity import SMALL_OPTS, DEFAULT_OPTS, _host

pytestmark = pytest.mark.gpu


def _to_dev(x64, dtype):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(x64, dtype=np.float32)).cuda()
    return t.to(torch.bfloat16) if dtype == "bf16" else t


def _run(rowptr, colidx, x_dev, mode, opts, dout_dev=None):
    import torch
    import paper_2605_31500_b200 as G
    n, ch = x_dev.shape
    plan = G.Plan(torch.from_numpy(rowptr).cuda(), torch.from_numpy(colidx).cuda(), transpose=False, **opts)
    out = torch.full_like(x_dev, float("nan"))
    arg = torch.full((n, ch), -7, dtype=torch.int32, device="cuda")
    G.gnn_seg_minmax_fwd(plan, x_dev, G.GNN_AGG_MIN if mode == "min" else G.GNN_AGG_MAX, out, arg)
    res = dict(out=_host(out), arg=arg.cpu().numpy(), plan=plan)
    if dout_dev is not None:
        dx = torch.full((n, ch), float("nan"), dtype=torch.float32, device="cuda")
        G.gnn_seg_minmax_bwd(arg, dout_dev, dx)
        res["dx"] = _host(dx)
    torch.cuda.synchronize()
    return res


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("mode", ["min", "max"])
@pytest.mark.parametrize("channels,opts", [(128, SMALL_OPTS), (96, SMALL_OPTS), (64, DEFAULT_OPTS), (8, SMALL_OPTS),
                                              (640, SMALL_OPTS), (1024, DEFAULT_OPTS)])   # channel groups (> 1024-byte rows)
def test_seg_minmax_parity(dtype, mode, channels, opts):
    """Power-law graph (cfg 2 scaled: hubs, CTA rows and packed rows under the small bins), random features AND a
    tie-heavy variant (three value levels, -0.0 included) that exercises the smaller-index rule in every merge."""
    if dtype == "f32" and channels == 8:
        channels = 12                                  # 48-byte rows: three 16-byte lanes
    c = GI.make_config(2, scale=0.03)
    rp, ci, n = c["rowptr"], c["colidx"], c["n"]
    rng = np.random.default_rng(channels)
    ci_shuffled = ci.copy()
    for i in range(n):
        ci_shuffled[rp[i]:rp[i + 1]] = rng.permutation(ci[rp[i]:rp[i + 1]])
    for ties, shuffled in ((False, False), (True, False), (True, True)):
        ci = ci_shuffled if shuffled else c["colidx"]   # sorted rows: strict-minimum fast path; shuffled: general path
        x = rng.standard_normal((n, channels)) if not ties else rng.integers(-1, 2, size=(n, channels)).astype(np.float64)
        if ties:
            x[rng.random((n, channels)) < 0.1] = -0.0
        xd = _to_dev(x, dtype)
        xq = _host(xd)                                 # the values the kernel sees (bf16-rounded)
        dout = rng.standard_normal((n, channels))
        dd = _to_dev(dout, dtype)
        got = _run(rp, ci, xd, mode, opts, dd)
        assert got["plan"].rows_sorted() == (not shuffled)
        if opts is SMALL_OPTS:
            cnt = got["plan"].counts()
            assert cnt["n_hub"] > 0 and cnt["n_cta"] > 0
        want_out, want_arg = agg_ref.seg_minmax_forward(rp, ci, xq, mode)
        assert np.array_equal(got["arg"], want_arg), f"arg differs ({dtype}, {mode}, C={channels}, ties={ties})"
        assert np.array_equal(got["out"], want_out), f"out differs ({dtype}, {mode}, C={channels}, ties={ties})"
        want_dx = agg_ref.seg_minmax_backward(want_arg, _host(dd), n)
        err = np.abs(got["dx"] - want_dx).max()
        assert err <= 1e-4 * max(1.0, np.abs(want_dx).max()), f"dx max abs err {err:.3e}"


def test_seg_minmax_degenerate():
    """Empty rows give 0 / -1 and no gradient; a multigraph with duplicate entries, a single self-loop graph and a
    row count that leaves ragged warps; errors are reported."""
    import torch
    import paper_2605_31500_b200 as G
    rng = np.random.default_rng(11)
    n, C = 1037, 32
    deg = rng.poisson(3.0, size=n)
    deg[rng.integers(0, n, 200)] = 0
    rp = np.concatenate([[0], np.cumsum(deg)]).astype(np.int32)
    ci = rng.integers(0, n, size=int(rp[-1])).astype(np.int32)      # duplicates allowed, unsorted
    x = rng.standard_normal((n, C))
    xd = _to_dev(x, "f32")
    dout = rng.standard_normal((n, C))
    got = _run(rp, ci, xd, "min", DEFAULT_OPTS, _to_dev(dout, "f32"))
    wo, wa = agg_ref.seg_minmax_forward(rp, ci, _host(xd), "min")
    assert np.array_equal(got["arg"], wa) and np.array_equal(got["out"], wo)
    assert np.all(got["arg"][deg == 0] == -1) and np.all(got["out"][deg == 0] == 0.0)
    wdx = agg_ref.seg_minmax_backward(wa, _host(_to_dev(dout, "f32")), n)
    assert np.abs(got["dx"] - wdx).max() <= 1e-5
    # self-loops only: identity
    rp1, ci1 = np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32)
    g1 = _run(rp1, ci1, xd, "max", DEFAULT_OPTS)
    assert np.array_equal(g1["out"], _host(xd)) and np.array_equal(g1["arg"], np.repeat(ci1[:, None], C, 1))
    # errors
    plan = g1["plan"]
    x3 = torch.zeros((n, 6), device="cuda")
    with pytest.raises(G.GnnError, match="unsupported shape"):
        G.gnn_seg_minmax_fwd(plan, x3, G.GNN_AGG_MIN, torch.empty_like(x3), torch.empty((n, 6), dtype=torch.int32, device="cuda"))
    with pytest.raises(G.GnnError, match="mode"):
        G.gnn_seg_minmax_fwd(plan, xd, 7, torch.empty_like(xd), torch.empty((n, C), dtype=torch.int32, device="cuda"))


@pytest.mark.parametrize("mode", ["min", "max"])
@pytest.mark.parametrize("shuffled", [False, True])
def test_seg_minmax_infinite_values(mode, shuffled):
    """+-inf are ordinary IEEE values (include/gnn_attn.h): a candidate whose signed value is +inf (x = +inf for min,
    -inf for max) must still beat "no candidate yet" - rows whose sources are all +inf return +inf and the smallest
    such source, not the empty-row answer 0 / -1 - through the per-lane update, the CTA-row merge and the hub merge."""
    c = GI.make_config(2, scale=0.03)
    rp, ci, n = c["rowptr"], c["colidx"].copy(), c["n"]
    rng = np.random.default_rng(5)
    if shuffled:
        for i in range(n):
            ci[rp[i]:rp[i + 1]] = rng.permutation(ci[rp[i]:rp[i + 1]])
    C = 64
    x = rng.standard_normal((n, C))
    bad = np.inf if mode == "min" else -np.inf
    x[rng.random((n, C)) < 0.3] = bad                  # scattered: some rows see only +-inf, most see a mix
    x[rng.random((n, C)) < 0.05] = -bad                # and the value that must always win
    x[:, :16] = bad                                    # whole channels: every row, hubs included, sees only +-inf there
    for dtype in ("f32", "bf16"):
        xd = _to_dev(x, dtype)
        got = _run(rp, ci, xd, mode, SMALL_OPTS)
        cnt = got["plan"].counts()
        assert cnt["n_hub"] > 0 and cnt["n_cta"] > 0
        want_out, want_arg = agg_ref.seg_minmax_forward(rp, ci, _host(xd), mode)
        assert np.array_equal(got["arg"], want_arg)
        assert np.array_equal(got["out"], want_out)
        deg = np.diff(rp)
        assert np.all(got["arg"][deg > 0] >= 0) and np.all(got["out"][deg > 0][:, :16] == bad)


@pytest.mark.slow
def test_seg_minmax_fullsize_cfg5():
    """BASELINE.json cfg 5 graph (4 M nodes, 94 M edges, hubs of in-degree up to 3 M = 733 chunks each) with the default
    plan, x = the config's xr tensor viewed as [n, 128] bf16: sampled rows (uniform + the heaviest) bit-exact against
    the oracle, every arg a stored in-neighbour whose value equals out, and gradient mass conserved."""
    import torch
    import paper_2605_31500_b200 as G
    c = GI.make_config(5, keep_f32=False, with_grads=False)
    n, rp, ci = c["n"], c["rowptr"], c["colidx"]
    x_st = c["xr_st"].reshape(n, -1)
    C = x_st.shape[1]
    xd = torch.from_numpy(np.ascontiguousarray(x_st)).view(torch.bfloat16).cuda()
    plan = G.Plan(torch.from_numpy(rp).cuda(), torch.from_numpy(ci).cuda(), transpose=False, **DEFAULT_OPTS)
    assert plan.counts()["n_hub"] > 0 and plan.rows_sorted()
    out = torch.empty_like(xd)
    arg = torch.empty((n, C), dtype=torch.int32, device="cuda")
    G.gnn_seg_minmax_fwd(plan, xd, G.GNN_AGG_MIN, out, arg)
    dout = torch.randn((n, C), device="cuda", generator=torch.Generator(device="cuda").manual_seed(0)).to(torch.bfloat16)
    dx = torch.empty((n, C), dtype=torch.float32, device="cuda")
    G.gnn_seg_minmax_bwd(arg, dout, dx)
    torch.cuda.synchronize()
    # properties at full size
    deg = np.diff(rp.astype(np.int64))
    nonempty = torch.from_numpy(deg > 0).cuda()
    assert bool(((arg >= 0).all(dim=1) == nonempty).all())
    sel = torch.gather(xd.float(), 0, arg.clamp(min=0).long())           # x[arg[i,c], c]
    assert bool((sel[nonempty] == out.float()[nonempty]).all())
    mass_in = dout.float()[nonempty].double().sum(0)
    mass_out = dx.double().sum(0)
    assert float((mass_in - mass_out).abs().max()) <= 1e-3 * float(mass_in.abs().max() + 1.0)
    # sampled rows against the oracle
    rng = np.random.default_rng(0)
    rows = np.unique(np.concatenate([rng.choice(n, size=3000, replace=False), np.argsort(-deg)[:4]]))
    rp_s = np.concatenate([[0], np.cumsum(deg[rows])]).astype(np.int64)
    ci_s = np.concatenate([ci[rp[r]:rp[r + 1]] for r in rows])
    xq = GI.bf16_bits_to_f32(x_st).astype(np.float64)
    wo, wa = agg_ref.seg_minmax_forward(rp_s, ci_s, xq, "min")
    rows_t = torch.from_numpy(rows).cuda().long()
    assert np.array_equal(arg[rows_t].cpu().numpy(), wa)
    assert np.array_equal(out[rows_t].float().cpu().numpy().astype(np.float64), wo)
