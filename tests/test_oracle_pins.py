"""Pins for the fp64 CPU oracle (oracle/): everything here is `-m "not gpu"`.

Each oracle function is checked against something other than itself:
  * hand-worked closed forms (tests/golden/*.json, with citations),
  * an independent dense numpy brute force (adjacency COUNT matrix, dense softmax),
  * library SDPA on the complete graph (textbook special case),
  * torch.autograd through a dense formulation (gradients never typed by hand),
  * central finite differences through the double-input build of the oracle,
  * invariants the mathematics fixes (north_star list) and conservation identities,
  * brute-force python loops / scipy for the integer plan metadata.
"""
import json
import math
import os

import numpy as np
import pytest
import torch

import oracle
from oracle import plan_ref

GOLD = os.path.join(os.path.dirname(__file__), "golden")
_NS = {"ln2": math.log(2.0), "ln3": math.log(3.0), "ln4": math.log(4.0), "ln34": math.log(34.0)}


def _val(x):
    return float(eval(x, {"__builtins__": {}}, _NS)) if isinstance(x, str) else float(x)


def _arr(x):
    if isinstance(x, list):
        return np.array([_arr(y) for y in x], dtype=np.float64)
    return _val(x)


def _rand_graph(rng, n, avg, multigraph=False, empty_rows=False):
    """Random directed (multi)graph as CSR (row = dst), unsorted neighbour order."""
    deg = rng.poisson(avg, size=n) + (0 if empty_rows else 1)
    if empty_rows:
        deg[rng.integers(0, n, size=max(1, n // 5))] = 0
    rowptr = np.zeros(n + 1, np.int32)
    rowptr[1:] = np.cumsum(deg)
    if multigraph:
        colidx = rng.integers(0, n, size=rowptr[-1]).astype(np.int32)
    else:
        colidx = np.concatenate([rng.choice(n, size=min(d, n), replace=False) if d else np.zeros(0, int)
                                 for d in np.minimum(deg, n)]).astype(np.int32)
        rowptr[1:] = np.cumsum(np.minimum(deg, n))
    return rowptr, colidx


def _count_matrix(rowptr, colidx):
    n = rowptr.size - 1
    C = np.zeros((n, n))
    for i in range(n):
        for e in range(rowptr[i], rowptr[i + 1]):
            C[i, colidx[e]] += 1.0
    return C


# --------------------------------------------------------------------------- dense brute force
def dense_gt(C, q, k, v):
    """Dense masked attention: S = QK^T/sqrt(d); alpha_ij = C_ij e^{S_ij} / sum_j C_ij e^{S_ij}."""
    n, H, d = q.shape
    O = np.zeros((n, H, d))
    L = np.full((n, H), -np.inf)
    for h in range(H):
        S = q[:, h, :] @ k[:, h, :].T / math.sqrt(d)
        with np.errstate(divide="ignore"):
            W = np.log(C) + S
        m = W.max(axis=1, keepdims=True)
        ok = np.isfinite(m[:, 0])
        E = np.exp(W[ok] - m[ok])
        Z = E.sum(axis=1, keepdims=True)
        O[ok, h, :] = (E / Z) @ v[:, h, :]
        L[ok, h] = (m[ok] + np.log(Z))[:, 0]
    return O, L


def dense_gatv2(C, xl, xr, a, slope):
    n, H, d = xl.shape
    O = np.zeros((n, H, d))
    L = np.full((n, H), -np.inf)
    for h in range(H):
        Z3 = xl[:, None, h, :] + xr[None, :, h, :]            # [i, j, c]
        S = (np.where(Z3 > 0, Z3, slope * Z3) * a[h][None, None, :]).sum(-1)
        with np.errstate(divide="ignore"):
            W = np.log(C) + S
        m = W.max(axis=1, keepdims=True)
        ok = np.isfinite(m[:, 0])
        E = np.exp(W[ok] - m[ok])
        Zs = E.sum(axis=1, keepdims=True)
        O[ok, h, :] = (E / Zs) @ xr[:, h, :]
        L[ok, h] = (m[ok] + np.log(Zs))[:, 0]
    return O, L


def _feat(rng, n, H, d, scale=1.0):
    return (rng.standard_normal((n, H, d)) * scale).astype(np.float32)


# --------------------------------------------------------------------------- golden fixtures
def test_golden_gt_two_node():
    g = json.load(open(os.path.join(GOLD, "gt_two_node.json")))
    rp, ci = np.array(g["rowptr"], np.int32), np.array(g["colidx"], np.int32)
    q, k, v = (_arr(g[x]) for x in "qkv")
    O, L = oracle.gt_forward(rp, ci, q, k, v)
    np.testing.assert_allclose(O, _arr(g["O"]), rtol=0, atol=1e-14)
    np.testing.assert_allclose(L, _arr(g["L"]), rtol=0, atol=1e-14)
    for case in ("case_a", "case_b"):
        r = oracle.gt_backward(rp, ci, q, k, v, _arr(g[case]["dO"]))
        for name in ("dQ", "dK", "dV"):
            np.testing.assert_allclose(r[name], _arr(g[case][name]), rtol=0, atol=1e-14, err_msg=f"{case} {name}")


def test_golden_gatv2_two_node():
    g = json.load(open(os.path.join(GOLD, "gatv2_two_node.json")))
    rp, ci = np.array(g["rowptr"], np.int32), np.array(g["colidx"], np.int32)
    xl, xr, a, dO = _arr(g["xl"]), _arr(g["xr"]), _arr(g["a"]), _arr(g["dO"])
    r = oracle.gatv2_backward(rp, ci, xl, xr, a, g["slope"], dO)
    for name in ("O", "L", "G", "da", "dxl", "dxr"):
        np.testing.assert_allclose(r[name], _arr(g[name]), rtol=0, atol=1e-14, err_msg=name)


# --------------------------------------------------------------------------- forward vs dense brute force
@pytest.mark.parametrize("seed,n,H,d,multi,empty", [(0, 9, 1, 4, False, False), (1, 23, 3, 8, True, False),
                                                     (2, 40, 2, 16, True, True), (3, 64, 4, 5, False, True)])
def test_gt_forward_vs_dense(seed, n, H, d, multi, empty):
    rng = np.random.default_rng(seed)
    rp, ci = _rand_graph(rng, n, 4.0, multi, empty)
    q, k, v = (_feat(rng, n, H, d) for _ in range(3))
    O, L = oracle.gt_forward(rp, ci, q, k, v)
    Od, Ld = dense_gt(_count_matrix(rp, ci), q.astype(np.float64), k.astype(np.float64), v.astype(np.float64))
    np.testing.assert_allclose(O, Od, rtol=0, atol=1e-12)
    np.testing.assert_array_equal(np.isinf(L), np.isinf(Ld))
    np.testing.assert_allclose(L[np.isfinite(L)], Ld[np.isfinite(Ld)], rtol=0, atol=1e-12)
    if empty:   # reading A5: empty row -> O = 0, L = -inf
        z = np.diff(rp) == 0
        assert z.any() and np.all(O[z] == 0) and np.all(np.isneginf(L[z]))


@pytest.mark.parametrize("seed,n,H,d,multi,slope", [(0, 9, 1, 4, False, 0.2), (1, 23, 3, 8, True, 0.2),
                                                     (2, 33, 2, 16, True, 0.01), (3, 20, 4, 5, False, 1.7)])
def test_gatv2_forward_vs_dense(seed, n, H, d, multi, slope):
    rng = np.random.default_rng(100 + seed)
    rp, ci = _rand_graph(rng, n, 4.0, multi, seed == 2)
    xl, xr = _feat(rng, n, H, d), _feat(rng, n, H, d)
    a = rng.standard_normal((H, d)).astype(np.float32)
    O, L = oracle.gatv2_forward(rp, ci, xl, xr, a, slope)
    Od, Ld = dense_gatv2(_count_matrix(rp, ci), xl.astype(np.float64), xr.astype(np.float64), a.astype(np.float64), slope)
    np.testing.assert_allclose(O, Od, rtol=0, atol=1e-12)
    fin = np.isfinite(Ld)
    np.testing.assert_array_equal(np.isfinite(L), fin)
    np.testing.assert_allclose(L[fin], Ld[fin], rtol=0, atol=1e-12)


def test_gt_complete_graph_is_library_sdpa():
    """Textbook special case: the complete graph with self-loops is plain dense softmax attention."""
    rng = np.random.default_rng(7)
    n, H, d = 17, 3, 8
    rp = (np.arange(n + 1) * n).astype(np.int32)
    ci = np.tile(np.arange(n, dtype=np.int32), n)
    q, k, v = (_feat(rng, n, H, d) for _ in range(3))
    O, L = oracle.gt_forward(rp, ci, q, k, v)
    tq, tk, tv = (torch.from_numpy(x.astype(np.float64)).permute(1, 0, 2) for x in (q, k, v))   # [H, n, d]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv)                        # scale 1/sqrt(d)
    np.testing.assert_allclose(O, ref.permute(1, 0, 2).numpy(), rtol=0, atol=1e-12)
    lse = torch.logsumexp(tq @ tk.transpose(1, 2) / math.sqrt(d), dim=-1)                     # [H, n]
    np.testing.assert_allclose(L, lse.T.numpy(), rtol=0, atol=1e-12)


# --------------------------------------------------------------------------- backward vs autograd (dense)
def _torch_dense_gt(C, q, k, v):
    d = q.shape[-1]
    S = torch.einsum("ihc,jhc->hij", q, k) / math.sqrt(d)
    W = S + torch.log(C)[None]
    A = torch.softmax(W, dim=-1)
    return torch.einsum("hij,jhc->ihc", A, v)


def _torch_dense_gatv2(C, xl, xr, a, slope):
    Z = xl[:, None] + xr[None, :]                        # [i, j, h, c]
    S = (torch.nn.functional.leaky_relu(Z, slope) * a[None, None]).sum(-1).permute(2, 0, 1)   # [h, i, j]
    A = torch.softmax(S + torch.log(C)[None], dim=-1)
    return torch.einsum("hij,jhc->ihc", A, xr)


@pytest.mark.parametrize("seed,multi", [(0, False), (1, True)])
def test_gt_backward_vs_autograd(seed, multi):
    rng = np.random.default_rng(200 + seed)
    n, H, d = 21, 2, 8
    rp, ci = _rand_graph(rng, n, 3.0, multi)
    q, k, v, dO = (_feat(rng, n, H, d) for _ in range(4))
    r = oracle.gt_backward(rp, ci, q, k, v, dO)
    C = torch.from_numpy(_count_matrix(rp, ci))
    tq, tk, tv = (torch.from_numpy(x.astype(np.float64)).requires_grad_() for x in (q, k, v))
    out = _torch_dense_gt(C, tq, tk, tv)
    out.backward(torch.from_numpy(dO.astype(np.float64)))
    np.testing.assert_allclose(r["O"], out.detach().numpy(), rtol=0, atol=1e-12)
    for name, t in (("dQ", tq), ("dK", tk), ("dV", tv)):
        np.testing.assert_allclose(r[name], t.grad.numpy(), rtol=0, atol=1e-11, err_msg=name)
    # Delta = <O, dO> equals sum_j alpha_ij dP_ij (PAPER.md:494 / :539)
    np.testing.assert_allclose(r["Delta"], (r["O"] * dO).sum(-1), rtol=0, atol=1e-12)


@pytest.mark.parametrize("seed,multi,slope", [(0, False, 0.2), (1, True, 0.2), (2, True, 1.5)])
def test_gatv2_backward_vs_autograd(seed, multi, slope):
    rng = np.random.default_rng(300 + seed)
    n, H, d = 19, 3, 4
    rp, ci = _rand_graph(rng, n, 3.0, multi)
    xl, xr, dO = (_feat(rng, n, H, d) for _ in range(3))
    a = rng.standard_normal((H, d)).astype(np.float32)
    r = oracle.gatv2_backward(rp, ci, xl, xr, a, slope, dO)
    C = torch.from_numpy(_count_matrix(rp, ci))
    txl, txr, ta = (torch.from_numpy(x.astype(np.float64)).requires_grad_() for x in (xl, xr, a))
    out = _torch_dense_gatv2(C, txl, txr, ta, slope)
    out.backward(torch.from_numpy(dO.astype(np.float64)))
    np.testing.assert_allclose(r["O"], out.detach().numpy(), rtol=0, atol=1e-12)
    for name, t in (("dxl", txl), ("dxr", txr), ("da", ta)):
        np.testing.assert_allclose(r[name], t.grad.numpy(), rtol=0, atol=1e-11, err_msg=name)


# --------------------------------------------------------------------------- backward vs finite differences
def _fd(fun, x, eps=1e-6):
    g = np.zeros_like(x)
    it = np.nditer(x, flags=["multi_index"])
    for _ in it:
        ix = it.multi_index
        old = x[ix]
        x[ix] = old + eps
        fp = fun()
        x[ix] = old - eps
        fm = fun()
        x[ix] = old
        g[ix] = (fp - fm) / (2 * eps)
    return g


def test_gt_backward_vs_finite_differences():
    """north_star: backward matches central finite differences to 1e-6 relative."""
    rng = np.random.default_rng(11)
    n, H, d = 7, 2, 4
    rp, ci = _rand_graph(rng, n, 2.5, multigraph=True)
    q, k, v, dO = (rng.standard_normal((n, H, d)) for _ in range(4))      # float64 -> double-input build
    r = oracle.gt_backward(rp, ci, q, k, v, dO)
    loss = lambda: float((oracle.gt_forward(rp, ci, q, k, v)[0] * dO).sum())
    for name, x in (("dQ", q), ("dK", k), ("dV", v)):
        g = _fd(loss, x)
        assert np.abs(r[name] - g).max() <= 1e-6 * max(1.0, np.abs(g).max()), name


def test_gatv2_backward_vs_finite_differences():
    rng = np.random.default_rng(12)
    n, H, d = 7, 2, 3
    rp, ci = _rand_graph(rng, n, 2.5, multigraph=True)
    xl, xr, dO = (rng.standard_normal((n, H, d)) for _ in range(3))
    a = rng.standard_normal((H, d))
    r = oracle.gatv2_backward(rp, ci, xl, xr, a, 0.2, dO)
    loss = lambda: float((oracle.gatv2_forward(rp, ci, xl, xr, a, 0.2)[0] * dO).sum())
    for name, x in (("dxl", xl), ("dxr", xr), ("da", a)):
        g = _fd(loss, x)
        assert np.abs(r[name] - g).max() <= 1e-6 * max(1.0, np.abs(g).max()), name


# --------------------------------------------------------------------------- invariants (north_star list)
def test_invariants_gt():
    rng = np.random.default_rng(21)
    n, H, d = 50, 2, 8
    rp, ci = _rand_graph(rng, n, 5.0)
    q, k, v = (_feat(rng, n, H, d) for _ in range(3))
    O, L = oracle.gt_forward(rp, ci, q, k, v)
    # alpha sums to 1: V = const vector -> O = that vector
    ones = np.ones_like(v)
    np.testing.assert_allclose(oracle.gt_forward(rp, ci, q, k, ones)[0], 1.0, rtol=0, atol=1e-14)
    # degree-1 row returns its neighbour's value exactly, and L = the single score
    rp1 = np.arange(n + 1, dtype=np.int32)
    ci1 = rng.permutation(n).astype(np.int32)
    O1, L1 = oracle.gt_forward(rp1, ci1, q, k, v)
    np.testing.assert_array_equal(O1, v[ci1].astype(np.float64))
    s = (q.astype(np.float64) * k[ci1].astype(np.float64)).sum(-1) / math.sqrt(d)
    np.testing.assert_allclose(L1, s, rtol=0, atol=1e-14)
    # constant scores (Q = 0) -> neighbour mean, L = ln deg
    O0, L0 = oracle.gt_forward(rp, ci, np.zeros_like(q), k, v)
    deg = np.diff(rp)
    mean = np.stack([v[ci[rp[i]:rp[i + 1]]].astype(np.float64).mean(0) for i in range(n)])
    np.testing.assert_allclose(O0, mean, rtol=0, atol=1e-13)
    np.testing.assert_allclose(L0, np.log(deg)[:, None].repeat(H, 1), rtol=0, atol=1e-13)
    # neighbour-order invariance
    ci_p = ci.copy()
    for i in range(n):
        ci_p[rp[i]:rp[i + 1]] = rng.permutation(ci[rp[i]:rp[i + 1]])
    Op, Lp = oracle.gt_forward(rp, ci_p, q, k, v)
    np.testing.assert_allclose(Op, O, rtol=0, atol=1e-13)
    np.testing.assert_allclose(Lp, L, rtol=0, atol=1e-13)
    # key shift: k_j + c leaves O unchanged and shifts L by <q_i, c>/sqrt(d)
    c = rng.standard_normal((1, H, d))
    Os, Ls = oracle.gt_forward(rp, ci, q.astype(np.float64), k.astype(np.float64) + c, v.astype(np.float64))
    np.testing.assert_allclose(Os, O, rtol=0, atol=1e-12)
    np.testing.assert_allclose(Ls - L, (q.astype(np.float64) * c).sum(-1) / math.sqrt(d), rtol=0, atol=1e-12)


def test_invariants_gatv2():
    rng = np.random.default_rng(22)
    n, H, d = 40, 3, 4
    rp, ci = _rand_graph(rng, n, 4.0)
    xl, xr, dO = (_feat(rng, n, H, d) for _ in range(3))
    a = rng.standard_normal((H, d)).astype(np.float32)
    # a = 0 -> constant scores -> neighbour mean of xr, L = ln deg
    O0, L0 = oracle.gatv2_forward(rp, ci, xl, xr, np.zeros_like(a), 0.2)
    mean = np.stack([xr[ci[rp[i]:rp[i + 1]]].astype(np.float64).mean(0) for i in range(n)])
    np.testing.assert_allclose(O0, mean, rtol=0, atol=1e-13)
    np.testing.assert_allclose(L0, np.log(np.diff(rp))[:, None].repeat(H, 1), rtol=0, atol=1e-13)
    # slope = 1: e_ij = a.xl_i + a.xr_j, alpha independent of xl -> dxl == 0 (up to cancellation) and
    # O does not depend on xl at all
    r = oracle.gatv2_backward(rp, ci, xl, xr, a, 1.0, dO)
    assert np.abs(r["dxl"]).max() < 1e-13
    O2, _ = oracle.gatv2_forward(rp, ci, _feat(rng, n, H, d), xr, a, 1.0)
    np.testing.assert_allclose(O2, r["O"], rtol=0, atol=1e-12)
    # sigma'(0) = slope (reading A8): xl = -xr on a self-loop-only graph makes z = 0 exactly
    rp1, ci1 = np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32)
    r1 = oracle.gatv2_backward(rp1, ci1, -xr, xr, a, 0.2, dO)
    np.testing.assert_array_equal(r1["O"], xr.astype(np.float64))          # degree 1
    np.testing.assert_allclose(r1["dxl"], 0.0, atol=1e-15)                 # de = alpha (dP - G) = 0 at degree 1
    np.testing.assert_allclose(r1["dxr"], dO.astype(np.float64), atol=1e-15)


def test_conservation_identities():
    """Identities usable at full scale: sum_j dV_j = sum_i dO_i;
    sum_i <q_i,dQ_i> = sum_j <k_j,dK_j>; sum_j dxr_j - sum_i dxl_i = sum_i dO_i."""
    rng = np.random.default_rng(23)
    n, H, d = 60, 2, 8
    rp, ci = _rand_graph(rng, n, 6.0, multigraph=True)
    q, k, v, dO = (_feat(rng, n, H, d) for _ in range(4))
    r = oracle.gt_backward(rp, ci, q, k, v, dO)
    np.testing.assert_allclose(r["dV"].sum(0), dO.astype(np.float64).sum(0), rtol=0, atol=1e-12)
    np.testing.assert_allclose((q * r["dQ"]).sum((0, 2)), (k * r["dK"]).sum((0, 2)), rtol=0, atol=1e-11)
    a = rng.standard_normal((H, d)).astype(np.float32)
    g = oracle.gatv2_backward(rp, ci, q, k, a, 0.2, dO)
    np.testing.assert_allclose(g["dxr"].sum(0) - g["dxl"].sum(0), dO.astype(np.float64).sum(0), rtol=0, atol=1e-12)


def test_row_subsets_match_full():
    rng = np.random.default_rng(24)
    n, H, d = 80, 2, 8
    rp, ci = _rand_graph(rng, n, 5.0)
    q, k, v, dO = (_feat(rng, n, H, d) for _ in range(4))
    full = oracle.gt_backward(rp, ci, q, k, v, dO)
    rows = rng.choice(n, size=13, replace=False).astype(np.int32)
    O, L = oracle.gt_forward(rp, ci, q, k, v, rows=rows)
    np.testing.assert_array_equal(O, full["O"][rows])
    np.testing.assert_array_equal(L, full["L"][rows])
    dQ = oracle.gt_backward_dst(rp, ci, q, k, v, dO, full["L"], full["Delta"], rows=rows)
    np.testing.assert_array_equal(dQ, full["dQ"][rows])
    rpt, cit = plan_ref.transpose_csr(rp, ci)
    dK, dV = oracle.gt_backward_src(rpt, cit, q, k, v, dO, full["L"], full["Delta"], srcs=rows)
    np.testing.assert_array_equal(dK, full["dK"][rows])
    np.testing.assert_array_equal(dV, full["dV"][rows])


# --------------------------------------------------------------------------- integer plan metadata
def test_transpose_csr_vs_bruteforce_and_scipy():
    import scipy.sparse as sp
    rng = np.random.default_rng(31)
    for multi in (False, True):
        n = 37
        rp, ci = _rand_graph(rng, n, 4.0, multi, empty_rows=True)
        rpt, cit = plan_ref.transpose_csr(rp, ci)
        # brute force: scan edges in CSR order, append dst to the source's list (stable by construction)
        lists = [[] for _ in range(n)]
        for i in range(n):
            for e in range(rp[i], rp[i + 1]):
                lists[ci[e]].append(i)
        np.testing.assert_array_equal(rpt, np.concatenate([[0], np.cumsum([len(x) for x in lists])]))
        np.testing.assert_array_equal(cit, np.concatenate([np.array(x, np.int32) for x in lists]))
        if not multi:
            A = sp.csr_matrix((np.ones(ci.size), ci, rp), shape=(n, n)).T.tocsr()
            A.sort_indices()
            np.testing.assert_array_equal(rpt, A.indptr)
            np.testing.assert_array_equal(cit, A.indices)
    # symmetric graph with sorted rows: CSR^T == CSR bit for bit
    m = rng.random((30, 30)) < 0.2
    m = m | m.T | np.eye(30, dtype=bool)
    A = sp.csr_matrix(m.astype(np.float64))
    A.sort_indices()
    rpt, cit = plan_ref.transpose_csr(A.indptr.astype(np.int32), A.indices.astype(np.int32))
    np.testing.assert_array_equal(rpt, A.indptr)
    np.testing.assert_array_equal(cit, A.indices)


def test_is_undirected_vs_dense_and_implies_self_transpose():
    """Row f1: is_undirected == (dense 0/1 adjacency equals its transpose, no repeated entry,
    ascending rows), and whenever it holds the stable transpose is the CSR itself; one removed mirror entry, one
    repeated entry or one swapped pair of neighbours breaks it."""
    import scipy.sparse as sp
    rng = np.random.default_rng(35)
    for trial in range(6):
        n = 23 + trial
        m = rng.random((n, n)) < 0.15
        if trial % 2 == 0:
            m = m | m.T
        A = sp.csr_matrix(m.astype(np.float64))
        A.sort_indices()
        rp, ci = A.indptr.astype(np.int32), A.indices.astype(np.int32)
        dense = np.zeros((n, n), np.int64)
        for i in range(n):
            for e in range(rp[i], rp[i + 1]):
                dense[i, ci[e]] += 1
        want = bool(np.array_equal(dense, dense.T) and dense.max() <= 1)
        assert plan_ref.is_undirected(rp, ci) == want == (trial % 2 == 0)
        if want:
            rpt, cit = plan_ref.transpose_csr(rp, ci)
            np.testing.assert_array_equal(rpt, rp)
            np.testing.assert_array_equal(cit, ci)
            i = int(np.argmax(np.diff(rp) >= 2))                      # a row with two neighbours
            swapped = ci.copy()
            swapped[rp[i]], swapped[rp[i] + 1] = ci[rp[i] + 1], ci[rp[i]]
            assert not plan_ref.is_undirected(rp, swapped)            # same edge set, row not ascending
            e = int(np.argmax(ci != np.repeat(np.arange(n), np.diff(rp))))   # first off-diagonal entry
            rp_cut = rp.copy()
            rp_cut[np.searchsorted(rp, e, side="right"):] -= 1
            assert not plan_ref.is_undirected(rp_cut, np.delete(ci, e))       # mirror entry missing
            rp_dup = rp.copy()
            rp_dup[np.searchsorted(rp, e, side="right"):] += 1
            assert not plan_ref.is_undirected(rp_dup, np.insert(ci, e, ci[e]))  # repeated entry
    assert plan_ref.is_undirected(np.array([0, 0, 0], np.int32), np.zeros(0, np.int32))   # no edges
    assert not plan_ref.is_undirected(np.array([0, 1], np.int32), np.array([3], np.int32))  # out-of-range source


def test_build_bins_vs_bruteforce():
    rng = np.random.default_rng(32)
    deg = np.concatenate([rng.integers(0, 6, 200), rng.integers(30, 300, 40), [1000, 2500, 4097, 9000, 0, 1, 64, 65]])
    rng.shuffle(deg)
    rp = np.concatenate([[0], np.cumsum(deg)]).astype(np.int32)
    wmax, cmax, sc = 64, 1024, 1000
    b = plan_ref.build_bins(rp, wmax, cmax, sc)

    def key(g):
        bl = int(g).bit_length()
        if g > cmax:
            return 0
        if g > wmax:
            return 1 + (32 - bl)
        return 34 + (32 - bl)

    order = sorted(range(deg.size), key=lambda r: (key(deg[r]), r))
    np.testing.assert_array_equal(b["perm"], np.array(order, np.int32))
    assert b["n_hub"] == int((deg > cmax).sum()) and b["n_cta"] == int(((deg > wmax) & (deg <= cmax)).sum())
    assert b["n_hub"] + b["n_cta"] + b["n_group"] == deg.size
    # chunk table: covers each hub row exactly once, contiguous, each chunk <= split_chunk, balanced to +-1
    ch = b["chunks"]
    for slot in range(b["n_hub"]):
        r = order[slot]
        mine = ch[b["hub_chunk_ptr"][slot]:b["hub_chunk_ptr"][slot + 1]]
        assert np.all(mine[:, 0] == r) and np.all(mine[:, 3] == slot)
        assert mine[0, 1] == rp[r] and mine[-1, 2] == rp[r + 1]
        np.testing.assert_array_equal(mine[1:, 1], mine[:-1, 2])
        sizes = mine[:, 2] - mine[:, 1]
        assert sizes.max() <= sc and sizes.max() - sizes.min() <= 1 and len(mine) == -(-deg[r] // sc)
    # heaviest first inside each class (bit-length buckets)
    dperm = deg[b["perm"]]
    bl = np.array([int(x).bit_length() for x in dperm])
    assert np.all(np.diff(bl[b["n_hub"]:b["n_hub"] + b["n_cta"]]) <= 0)
    assert np.all(np.diff(bl[b["n_hub"] + b["n_cta"]:]) <= 0)


def test_build_blocks_vs_bruteforce():
    rng = np.random.default_rng(33)
    n = 70                                   # ragged last window (70 = 4*16 + 6)
    rp, ci = _rand_graph(rng, n, 3.0, multigraph=True, empty_rows=True)
    # add many in-window edges
    extra_d = rng.integers(0, n, 300)
    extra_s = np.minimum((extra_d // 16) * 16 + rng.integers(0, 16, 300), n - 1)
    d_all = np.concatenate([np.repeat(np.arange(n), np.diff(rp)), extra_d])
    s_all = np.concatenate([ci, extra_s])
    o = np.argsort(d_all, kind="stable")
    d_all, s_all = d_all[o], s_all[o]
    rp = np.concatenate([[0], np.cumsum(np.bincount(d_all, minlength=n))]).astype(np.int32)
    ci = s_all.astype(np.int32)
    b = plan_ref.build_blocks(rp, ci)
    nw = (n + 15) // 16
    bm = np.zeros((nw, 16), np.uint16)
    rem_rows = [[] for _ in range(n)]
    for i in range(n):
        seen = set()
        for e in range(rp[i], rp[i + 1]):
            j = int(ci[e])
            if j // 16 == i // 16 and j not in seen:
                seen.add(j)
                bm[i // 16, i % 16] |= np.uint16(1 << (j % 16))
            else:
                rem_rows[i].append(j)
    np.testing.assert_array_equal(b["bitmap"], bm)
    np.testing.assert_array_equal(b["rem_rowptr"], np.concatenate([[0], np.cumsum([len(x) for x in rem_rows])]))
    np.testing.assert_array_equal(b["rem_colidx"], np.concatenate([np.array(x, np.int32) for x in rem_rows]))
    # every CSR entry is accounted for exactly once
    assert int(sum(bin(int(x)).count("1") for x in bm.ravel())) + b["rem_colidx"].size == ci.size


def _wsb_bruteforce(rp, ci, n):
    """PAPER.md:545 read literally, with Python sets and loops."""
    nw = (n + 15) // 16
    offs, cols, bms = [0], [], []
    for w in range(nw):
        rows = range(16 * w, min(n, 16 * w + 16))
        uniq = sorted({int(ci[e]) for i in rows for e in range(rp[i], rp[i + 1])})
        for t in range(0, len(uniq), 8):
            blk = uniq[t:t + 8]
            cols.append(blk + [0] * (8 - len(blk)))
            bm = [0] * 16
            for i in rows:
                present = {int(ci[e]) for e in range(rp[i], rp[i + 1])}
                for c, j in enumerate(blk):
                    if j in present:
                        bm[i - 16 * w] |= 1 << c
            bms.append(bm)
        offs.append(len(cols))
    return np.array(offs, np.int32), np.array(cols, np.int32).reshape(-1, 8), np.array(bms, np.uint8).reshape(-1, 16)


@pytest.mark.parametrize("multigraph", [False, True])
def test_build_wsb_vs_bruteforce_and_roundtrip(multigraph):
    """Row f2 layout: per 16-row window the sorted unique source columns cut into width-8 TCBs,
    zero-padded column lists, 128-bit bitmaps, tcb_row_offset - against a literal set-and-loop construction, and
    expanding the layout back gives exactly the set of distinct (dst, src) pairs of the CSR."""
    rng = np.random.default_rng(41 + multigraph)
    n = 103                                   # ragged last window (103 = 6*16 + 7)
    rp, ci = _rand_graph(rng, n, 5.0, multigraph=multigraph, empty_rows=True)
    # overlapping column sets between windows + a dense window + a row with > 8 * 3 distinct sources
    extra_d = np.concatenate([rng.integers(0, n, 400), np.full(40, 17), rng.integers(32, 48, 200)])
    extra_s = np.concatenate([rng.integers(0, 12, 400), rng.integers(0, n, 40), rng.integers(32, 48, 200)])
    d_all = np.concatenate([np.repeat(np.arange(n), np.diff(rp)), extra_d])
    s_all = np.concatenate([ci, extra_s])
    if not multigraph:
        key = np.unique(d_all.astype(np.int64) * n + s_all)
        d_all, s_all = key // n, key % n
    o = np.lexsort((s_all, d_all)) if not multigraph else np.argsort(d_all, kind="stable")
    d_all, s_all = d_all[o], s_all[o]
    rp = np.concatenate([[0], np.cumsum(np.bincount(d_all, minlength=n))]).astype(np.int32)
    ci = s_all.astype(np.int32)
    w = plan_ref.build_wsb(rp, ci)
    offs, cols, bms = _wsb_bruteforce(rp, ci, n)
    np.testing.assert_array_equal(w["tcb_row_offset"], offs)
    np.testing.assert_array_equal(w["tcb_cols"], cols)
    np.testing.assert_array_equal(w["tcb_bitmap"], bms)
    assert w["n_windows"] == 7 and w["n_tcb"] == cols.shape[0]
    # round trip: the layout encodes exactly the distinct (dst, src) pairs
    pairs = set()
    for win in range(w["n_windows"]):
        for t in range(w["tcb_row_offset"][win], w["tcb_row_offset"][win + 1]):
            for r in range(16):
                for c in range(8):
                    if (int(w["tcb_bitmap"][t, r]) >> c) & 1:
                        pairs.add((16 * win + r, int(w["tcb_cols"][t, c])))
    want = {(i, int(ci[e])) for i in range(n) for e in range(rp[i], rp[i + 1])}
    assert pairs == want
    assert w["n_dup"] == ci.size - len(want) and (w["n_dup"] > 0) == multigraph
    # columns inside a window ascend across its TCBs; padding sits only at the end of a window's last TCB
    for win in range(w["n_windows"]):
        t0, t1 = w["tcb_row_offset"][win], w["tcb_row_offset"][win + 1]
        used = w["tcb_bitmap"][t0:t1].reshape(t1 - t0, 16)
        colmask = np.bitwise_or.reduce(used, axis=1) if t1 > t0 else np.zeros(0, np.uint8)
        flat = [(int(w["tcb_cols"][t0 + k, c]), (int(colmask[k]) >> c) & 1) for k in range(t1 - t0) for c in range(8)]
        valid = [j for j, u in flat if u]
        assert valid == sorted(set(valid))
        assert all(u for _, u in flat[:len(valid)]) and all(j == 0 and not u for j, u in flat[len(valid):])


# --------------------------------------------------------------------------- min / max aggregation (row f3)
from oracle import agg_ref  # noqa: E402


@pytest.mark.parametrize("mode", ["min", "max"])
def test_seg_minmax_vs_bruteforce(mode):
    """Pin: the definition evaluated pair by pair with Python tuples - lexicographic (value, source id) over the
    neighbour set, PAPER.md:462/:474 - on a multigraph with empty rows and heavy ties (values drawn from 3 levels)."""
    rng = np.random.default_rng(5)
    n, C = 41, 6
    rp, ci = _rand_graph(rng, n, 4.0, multigraph=True, empty_rows=True)
    x = rng.integers(-1, 2, size=(n, C)).astype(np.float64)          # many ties
    x[rng.integers(0, n, 5)] *= 0.5
    out, arg = agg_ref.seg_minmax_forward(rp, ci, x, mode)
    sgn = 1.0 if mode == "min" else -1.0
    for i in range(n):
        nb = sorted(set(int(j) for j in ci[rp[i]:rp[i + 1]]))
        for c in range(C):
            if not nb:
                assert out[i, c] == 0.0 and arg[i, c] == -1
                continue
            v, j = min((sgn * x[j, c], j) for j in nb)
            assert out[i, c] == sgn * v and arg[i, c] == j


def test_seg_minmax_closed_forms():
    rng = np.random.default_rng(6)
    n, C = 30, 4
    rp, ci = _rand_graph(rng, n, 3.0)
    x = rng.standard_normal((n, C))
    # degree-1 rows return their neighbour; constant features pick the smallest neighbour id
    rp1 = np.arange(n + 1, dtype=np.int32)
    ci1 = rng.permutation(n).astype(np.int32)
    out, arg = agg_ref.seg_minmax_forward(rp1, ci1, x, "min")
    np.testing.assert_array_equal(out, x[ci1])
    np.testing.assert_array_equal(arg, np.repeat(ci1[:, None], C, 1))
    out, arg = agg_ref.seg_minmax_forward(rp, ci, np.ones((n, C)), "max")
    for i in range(n):
        assert np.all(out[i] == 1.0) and np.all(arg[i] == ci[rp[i]:rp[i + 1]].min())
    # neighbour order and duplicate entries do not matter; max(x) = -min(-x) with the same sources
    out0, arg0 = agg_ref.seg_minmax_forward(rp, ci, x, "min")
    ci2 = ci.copy()
    for i in range(n):
        ci2[rp[i]:rp[i + 1]] = rng.permutation(ci[rp[i]:rp[i + 1]])
    out1, arg1 = agg_ref.seg_minmax_forward(rp, ci2, x, "min")
    np.testing.assert_array_equal(out0, out1)
    np.testing.assert_array_equal(arg0, arg1)
    rpd = (2 * rp.astype(np.int64)).astype(np.int32)
    cid = np.concatenate([np.tile(ci[rp[i]:rp[i + 1]], 2) for i in range(n)]).astype(np.int32)
    out2, arg2 = agg_ref.seg_minmax_forward(rpd, cid, x, "min")
    np.testing.assert_array_equal(out0, out2)
    np.testing.assert_array_equal(arg0, arg2)
    outm, argm = agg_ref.seg_minmax_forward(rp, ci, -x, "max")
    np.testing.assert_array_equal(outm, -out0)
    np.testing.assert_array_equal(argm, arg0)
    # -0.0 and +0.0 tie: the smaller source id wins
    rpz, ciz = np.array([0, 2], np.int32), np.array([1, 0], np.int32)
    oz, az = agg_ref.seg_minmax_forward(np.array([0, 2, 2], np.int32), ciz, np.array([[0.0], [-0.0]]), "min")
    assert az[0, 0] == 0 and az[1, 0] == -1 and oz[1, 0] == 0.0
    del rpz


@pytest.mark.parametrize("mode", ["min", "max"])
def test_seg_minmax_backward_vs_autograd(mode):
    """Pin: gradient of the dense masked amin / amax (continuous values => no ties, so autograd's even split among
    equal elements never triggers) equals the scatter through the saved indices."""
    rng = np.random.default_rng(7)
    n, C = 25, 5
    rp, ci = _rand_graph(rng, n, 3.0, empty_rows=True)
    x = rng.standard_normal((n, C))
    dout = rng.standard_normal((n, C))
    out, arg = agg_ref.seg_minmax_forward(rp, ci, x, mode)
    dx = agg_ref.seg_minmax_backward(arg, dout, n)
    M = torch.from_numpy(_count_matrix(rp, ci) > 0)
    tx = torch.from_numpy(x).requires_grad_(True)
    fill = math.inf if mode == "min" else -math.inf
    dense = torch.where(M[:, :, None], tx[None, :, :], torch.tensor(fill, dtype=torch.float64))
    red = dense.amin(dim=1) if mode == "min" else dense.amax(dim=1)
    nonempty = M.any(dim=1)
    red = torch.where(nonempty[:, None], red, torch.zeros_like(red))
    np.testing.assert_allclose(red.detach().numpy(), out, rtol=0, atol=0)
    red.backward(torch.from_numpy(dout))
    np.testing.assert_allclose(tx.grad.numpy(), dx, rtol=0, atol=1e-15)
    # gradient mass is conserved: every non-empty (i, c) sends its dout to exactly one source
    np.testing.assert_allclose(dx.sum(0), dout[nonempty.numpy()].sum(0), rtol=0, atol=1e-12)


# --------------------------------------------------------------------------- row f4: LayerNorm + QKV projection, dot-aggr
from oracle import block_ref  # noqa: E402


def test_layer_norm_vs_library_and_closed_forms():
    """block_ref.layer_norm against the library routine (torch.nn.functional.layer_norm, fp64) and closed forms: with
    gamma = 1, beta = 0 every row has mean 0 and variance var / (var + eps); a constant row maps to beta; the result
    is invariant to a per-row shift and (up to eps) to a per-row positive scale."""
    rng = np.random.default_rng(5)
    x = rng.standard_normal((37, 96)) * rng.uniform(0.1, 5.0, (37, 1)) + rng.standard_normal((37, 1))
    g, b = rng.standard_normal(96), rng.standard_normal(96)
    got = block_ref.layer_norm(x, g, b, 1e-5)
    want = torch.nn.functional.layer_norm(torch.from_numpy(x), (96,), torch.from_numpy(g), torch.from_numpy(b), 1e-5).numpy()
    np.testing.assert_allclose(got, want, rtol=1e-12, atol=1e-12)
    y = block_ref.layer_norm(x, np.ones(96), np.zeros(96), 1e-5)
    var = x.var(axis=1)
    np.testing.assert_allclose(y.mean(axis=1), 0.0, atol=1e-12)
    np.testing.assert_allclose(y.var(axis=1), var / (var + 1e-5), rtol=1e-10)
    np.testing.assert_allclose(block_ref.layer_norm(np.full((3, 96), 7.25), g, b), np.tile(b, (3, 1)), atol=1e-12)
    np.testing.assert_allclose(block_ref.layer_norm(x + 3.0, g, b), got, atol=1e-10)
    np.testing.assert_allclose(block_ref.layer_norm(x * 1e3, g, b, 0.0), block_ref.layer_norm(x, g, b, 0.0), atol=1e-9)


def test_ln_qkv_vs_loops_and_library():
    """block_ref.ln_qkv: the projection against explicit loops on a tiny case (which row block of W feeds Q, K, V; the
    head / channel order of the outputs) and against torch layer_norm + linear in fp64."""
    rng = np.random.default_rng(6)
    n, C, H, d = 5, 16, 2, 4
    x, g, b = rng.standard_normal((n, C)), rng.standard_normal(C), rng.standard_normal(C)
    w, bias = rng.standard_normal((3 * H * d, C)), rng.standard_normal(3 * H * d)
    q, k, v = block_ref.ln_qkv(x, g, b, w, bias, H, d)
    y = torch.nn.functional.layer_norm(torch.from_numpy(x), (C,), torch.from_numpy(g), torch.from_numpy(b), 1e-5).numpy()
    for t, out in enumerate((q, k, v)):
        for i in range(n):
            for h in range(H):
                for c in range(d):
                    row = t * H * d + h * d + c
                    want = sum(y[i, m] * w[row, m] for m in range(C)) + bias[row]
                    assert abs(out[i, h, c] - want) < 1e-12
    lin = torch.nn.functional.linear(torch.from_numpy(y), torch.from_numpy(w), torch.from_numpy(bias)).numpy()
    np.testing.assert_allclose(np.concatenate([q.reshape(n, -1), k.reshape(n, -1), v.reshape(n, -1)], axis=1), lin, atol=1e-12)
    q0, _, _ = block_ref.ln_qkv(x, g, b, w, None, H, d)
    np.testing.assert_allclose(q0, q - bias[:H * d].reshape(1, H, d), atol=1e-12)


def test_dot_aggr_vs_dense():
    """block_ref.dot_aggr against the dense form diag(C X X^T) with C the edge-count matrix (multigraph), and the
    closed form on a graph of self-loops only (out[i] = |x_i|^2)."""
    rng = np.random.default_rng(7)
    n = 23
    rp, ci = _rand_graph(rng, n, 3.0, multigraph=True, empty_rows=True)
    x = rng.standard_normal((n, 12))
    C = _count_matrix(rp, ci)
    np.testing.assert_allclose(block_ref.dot_aggr(rp, ci, x), np.einsum("ij,ij->i", C, x @ x.T), atol=1e-12)
    rp1, ci1 = np.arange(n + 1), np.arange(n)
    np.testing.assert_allclose(block_ref.dot_aggr(rp1, ci1, x), (x * x).sum(axis=1), atol=1e-12)
