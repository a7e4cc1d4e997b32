"""Pins for the CPU oracle (no GPU).  Each test checks oracle/ against something other than itself:
invariants named by BASELINE.json:north_star, closed forms, torch CPU fp64 library routines on
special cases, the dense every-expert-runs-every-token formulation with torch autograd, central
finite differences, and the literal (quadratic) statement of the permutation rule.
Citations: SURVEY.md §8(c) "What pins the oracle"; BASELINE.json:north_star."""
import dataclasses
import json
import os

import numpy as np
import pytest
import torch

from inputs import configs as C
from oracle import oracle as O

torch.set_default_dtype(torch.float64)


def small_cfg(**kw):
    base = dict(name="t", T=24, d=12, E=6, k=3, I=20, seed=77, dtype=C.DT_F32)
    base.update(kw)
    return C.MoeConfig(**base)


def spread_logits(cfg, rng, gap=0.05):
    """Logits whose values within a row differ by at least `gap` (top-k locally constant, no ties)."""
    z = np.empty((cfg.T, cfg.E), np.float32)
    for t in range(cfg.T):
        z[t] = (rng.permutation(cfg.E) * gap * 4 + rng.uniform(0, gap, cfg.E) - 1.0).astype(np.float32)
    return z


# ------------------------------------------------------------------------------------- router
def test_router_closed_forms_and_library_special_case():
    """oracle_router_fwd / _bwd against what the mathematics fixes: one-hot tokens read a row of
    W_r (+ bias), an all-ones token sums its columns, integer-valued inputs give exact integers; dW_r of a one-hot dz
    is a token row of x and dX_r a column of W_r; on random data numpy's fp64 matmul; and the generator's logits
    (inputs/configs.py, reading c-18) are this sum rounded to fp32 plus one fp32 add of the bias."""
    cfg = small_cfg(T=6, d=12, E=6, k=3, dtype=C.DT_F32)
    rng = np.random.default_rng(9)
    w = rng.integers(-4, 5, size=(cfg.d, cfg.E)).astype(np.float32)
    bias = rng.integers(-3, 4, size=cfg.E).astype(np.float32)
    x = np.zeros((cfg.T, cfg.d), np.float32)
    for t in range(5):
        x[t, 2 * t] = 1.0
    x[5] = 1.0
    z = O.router_fwd(cfg, x, w, bias)
    for t in range(5):
        assert (z[t] == w[2 * t].astype(np.float64) + bias).all()
    assert (z[5] == w.sum(0, dtype=np.float64) + bias).all()
    assert (O.router_fwd(cfg, x, w) == z - bias).all()
    xr = rng.normal(size=(cfg.T, cfg.d)).astype(np.float32)
    dz = np.zeros((cfg.T, cfg.E))
    dz[3, 4] = 2.0
    dw, dx = O.router_bwd(cfg, xr, w, dz)
    assert (dw[:, 4] == 2.0 * xr[3].astype(np.float64)).all() and not np.delete(dw, 4, axis=1).any()
    assert (dx[3] == 2.0 * w[:, 4].astype(np.float64)).all() and not np.delete(dx, 3, axis=0).any()
    dzr = rng.normal(size=(cfg.T, cfg.E))
    dw, dx = O.router_bwd(cfg, xr, w, dzr)
    np.testing.assert_allclose(dw, xr.astype(np.float64).T @ dzr, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(dx, dzr @ w.astype(np.float64).T, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(O.router_fwd(cfg, xr, w, bias), xr.astype(np.float64) @ w + bias, rtol=1e-13, atol=1e-14)
    # central differences of <dz, z(x, W)>: the backward terms are the gradients of the forward
    eps = 1e-6
    xd, wd = xr.astype(np.float64), w.astype(np.float64)
    for (t, i) in ((0, 0), (4, 7)):
        xp_, xm_ = xd.copy(), xd.copy()
        xp_[t, i] += eps
        xm_[t, i] -= eps
        num = ((xp_ @ wd - xm_ @ wd) * dzr).sum() / (2 * eps)
        assert abs(num - dx[t, i]) < 1e-6 * max(1.0, abs(num))
    # bf16 configs: the generator's logits = fl32(fl32(sum in fp64) + bias)
    cfgb = dataclasses.replace(C.C3S, T=40)
    inp = C.make_inputs(cfgb, weights=False, with_dy=False)
    zb = O.router_fwd(cfgb, inp["x"], inp["w_r"])
    assert (inp["logits"] == (zb.astype(np.float32) + inp["bias"][None, :]).astype(np.float32)).all()
    # dense_dz scatters the k selected entries of each token to their experts' columns and leaves zeros elsewhere
    idx = np.array([[2, 0, 5], [1, 4, 3]], np.int32)
    dsel = np.array([[1.0, 2.0, 3.0], [4.0, 5.0, 6.0]])
    dd = O.dense_dz(small_cfg(T=2, E=6, k=3), idx, dsel)
    assert dd.tolist() == [[2.0, 0, 1.0, 0, 0, 3.0], [0, 4.0, 0, 6.0, 5.0, 0]]


# ------------------------------------------------------------------------------------ routing
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_route_invariants(mode):
    cfg = small_cfg(T=300, E=16, k=4, gate_mode=mode)
    z = np.random.default_rng(1).normal(size=(cfg.T, cfg.E)).astype(np.float32)
    idx, gates, cg = O.route_topk(cfg, z)
    assert cg.sum() == cfg.T * cfg.k                                   # north_star: counts sum to T*k
    assert idx.min() >= 0 and idx.max() < cfg.E
    for t in range(cfg.T):
        sel = idx[t]
        assert len(set(sel.tolist())) == cfg.k
        assert all(z[t, sel[j]] >= z[t, sel[j + 1]] for j in range(cfg.k - 1))   # descending
        rest = np.setdiff1d(np.arange(cfg.E), sel)
        assert z[t, rest].max() <= z[t, sel].min()
    assert (np.bincount(idx.reshape(-1), minlength=cfg.E) == cg).all()
    assert (gates > 0).all()
    if mode in (0, 1):
        np.testing.assert_allclose(gates.sum(1), 1.0, rtol=0, atol=1e-14)


def test_route_closed_forms():
    cfg = small_cfg(T=5, E=8, k=3)
    z = np.full((cfg.T, cfg.E), 0.37, np.float32)
    for mode in (0, 1):
        idx, gates, _ = O.route_topk(dataclasses.replace(cfg, gate_mode=mode), z)
        assert (idx == np.arange(3)[None, :]).all()                    # ties -> lowest index
        assert (gates == 1.0 / 3.0).all()                              # exactly 1/k
    cfg1 = small_cfg(T=7, E=5, k=1)
    z1 = np.random.default_rng(2).normal(size=(7, 5)).astype(np.float32)
    for mode in (0, 1):
        idx, gates, _ = O.route_topk(dataclasses.replace(cfg1, gate_mode=mode), z1)
        assert (gates == 1.0).all() and (idx[:, 0] == z1.argmax(1)).all()
    # k = E, mode 0: ordinary softmax
    cfgE = small_cfg(T=9, E=6, k=6)
    zE = np.random.default_rng(3).normal(size=(9, 6)).astype(np.float32)
    idx, gates, _ = O.route_topk(cfgE, zE)
    sm = torch.softmax(torch.from_numpy(zE).double(), dim=1).numpy()
    np.testing.assert_allclose(gates, np.take_along_axis(sm, idx.astype(np.int64), 1), rtol=1e-13)


def test_route_tie_rule():
    cfg = small_cfg(T=3, E=6, k=3)
    z = np.array([[1.0, 2.0, 2.0, 0.5, 2.0, 1.0],      # three equal maxima -> 1,2,4
                  [0.0, -0.0, 0.0, -0.0, -1.0, -1.0],  # -0.0 == +0.0 is a tie -> 0,1,2
                  [3.0, 1.0, 1.0, 3.0, 1.0, 0.0]], np.float32)  # 0,3 then tie among 1,2,4 -> 1
    idx, _, _ = O.route_topk(cfg, z)
    assert idx.tolist() == [[1, 2, 4], [0, 1, 2], [0, 3, 1]]


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_route_matches_torch_on_tie_free_rows(mode):
    cfg = small_cfg(T=200, E=32, k=8, gate_mode=mode)
    z = spread_logits(cfg, np.random.default_rng(4))
    idx, gates, _ = O.route_topk(cfg, z)
    zt = torch.from_numpy(z).double()
    v, i = torch.topk(zt, cfg.k, dim=1)
    assert (i.numpy() == idx).all()
    if mode == 0:
        ref = torch.softmax(v, dim=1)
    elif mode == 1:
        s = torch.sigmoid(v)
        ref = s / s.sum(1, keepdim=True)
    else:
        ref = torch.softmax(zt, dim=1).gather(1, i)
    np.testing.assert_allclose(gates, ref.numpy(), rtol=1e-12)


def test_route_neg_inf_and_preconditions():
    cfg = small_cfg(T=2, E=5, k=2)
    z = np.array([[-np.inf, 0.1, -np.inf, 0.3, 0.2], [1, 2, 3, 4, -np.inf]], np.float32)
    idx, gates, cg = O.route_topk(cfg, z)
    assert idx.tolist() == [[3, 4], [3, 2]] and cg[0] == 0
    bad = z.copy(); bad[0, 1] = np.nan
    with pytest.raises(ValueError):
        O.route_topk(cfg, bad)
    few = np.full((2, 5), -np.inf, np.float32); few[:, 0] = 1
    with pytest.raises(ValueError):
        O.route_topk(cfg, few)


# -------------------------------------------------------------------------------- permutation
@pytest.mark.parametrize("align", [1, 4, 16])
@pytest.mark.parametrize("local", [(0, 6), (2, 3)])
def test_permutation_invariants_and_literal_definition(align, local):
    e_lo, e_loc = local
    cfg = small_cfg(T=97, E=6, k=3, e_lo=e_lo, E_loc=e_loc, row_align=align)
    z = np.random.default_rng(5).normal(size=(cfg.T, cfg.E)).astype(np.float32)
    idx, gates, _ = O.route_topk(cfg, z)
    counts, offsets, row_of, src_of = O.permute(cfg, idx)
    local_mask = (idx >= e_lo) & (idx < e_lo + e_loc)
    assert counts.sum() == local_mask.sum()
    assert (np.diff(offsets) >= counts).all() and offsets[0] == 0
    assert (np.diff(offsets) == (counts + align - 1) // align * align).all()
    if align == 1:
        assert offsets[-1] == local_mask.sum()
    rows = row_of[local_mask]
    assert (row_of[~local_mask] == -1).all()
    assert len(np.unique(rows)) == len(rows)                            # bijection onto non-pad rows
    flat = row_of.reshape(-1)
    a_ids = np.nonzero(flat >= 0)[0]
    assert (src_of[flat[a_ids]] == a_ids).all()                         # src_of o row_of = id
    assert (src_of >= 0).sum() == len(a_ids)                            # everything else is -1
    # literal statement of the rule: offsets[i] + #{t' < t : e in topk_idx[t']}
    for t in range(cfg.T):
        for j in range(cfg.k):
            e = idx[t, j]
            if not (e_lo <= e < e_lo + e_loc):
                continue
            earlier = sum(1 for tp in range(t) if e in idx[tp])
            assert row_of[t, j] == offsets[e - e_lo] + earlier
    # ascending token ids inside each segment
    for i in range(e_loc):
        seg = src_of[offsets[i]: offsets[i] + counts[i]]
        assert (np.diff(seg // cfg.k) > 0).all()
        assert (src_of[offsets[i] + counts[i]: offsets[i + 1]] == -1).all()


def test_identity_experts_return_input():
    """unpermute o permute = identity: O := Xp, all experts local, renormalised gates -> Y = x."""
    for mode in (0, 1):
        cfg = small_cfg(T=50, E=8, k=4, gate_mode=mode)
        rng = np.random.default_rng(6)
        z = rng.normal(size=(cfg.T, cfg.E)).astype(np.float32)
        x = rng.normal(size=(cfg.T, cfg.d)).astype(np.float32)
        idx, gates, _ = O.route_topk(cfg, z)
        _, _, row_of, src_of = O.permute(cfg, idx)
        xp, gate_rows = O.pack(cfg, x, src_of, gates)
        assert (xp[row_of.reshape(-1)] == np.repeat(x.astype(np.float64), cfg.k, 0)).all()   # exact copies
        assert (gate_rows[row_of.reshape(-1)] == gates.reshape(-1)).all()
        y = O.combine(cfg, xp, row_of, gates)
        np.testing.assert_allclose(y, x.astype(np.float64), rtol=1e-14, atol=1e-15)


# ---------------------------------------------------------------------------------------- FFN
def test_single_expert_is_textbook_swiglu():
    cfg = small_cfg(T=17, E=1, k=1, d=10, I=14)
    inp = C.make_inputs(cfg)
    f = O.forward(cfg, inp)
    x, wg, wu, wd = (torch.from_numpy(inp[n].astype(np.float64)) for n in ("x", "w_gate", "w_up", "w_down"))
    ref = (torch.nn.functional.silu(x @ wg[0]) * (x @ wu[0])) @ wd[0]
    np.testing.assert_allclose(f["y"], ref.numpy(), rtol=1e-12, atol=1e-14)
    assert (f["gates"] == 1.0).all()


def dense_reference(cfg, inp, topk_idx, detach_gates=True):
    """Dense formulation in torch fp64: every local expert runs every token; results masked by the
    routing decision and weighted by the gates (recomputed from the logits with torch ops)."""
    x = torch.from_numpy(C.as_f64(inp["x"])).requires_grad_(True)
    z = torch.from_numpy(inp["logits"].astype(np.float64)).requires_grad_(True)
    W = {n: torch.from_numpy(C.as_f64(inp[n])).requires_grad_(True) for n in ("w_gate", "w_up", "w_down")}
    idx = torch.from_numpy(topk_idx.astype(np.int64))
    zsel = z.gather(1, idx)
    if cfg.gate_mode == 0:
        g = torch.softmax(zsel, dim=1)
    elif cfg.gate_mode == 1:
        s = torch.sigmoid(zsel)
        g = s / s.sum(1, keepdim=True)
    else:
        g = torch.softmax(z, dim=1).gather(1, idx)
    g.retain_grad()
    dense_gate = torch.zeros(cfg.T, cfg.E).scatter(1, idx, g)                      # [T, E], zero if unrouted
    y = torch.zeros(cfg.T, cfg.d)
    for i in range(cfg.e_loc):
        out_e = (torch.nn.functional.silu(x @ W["w_gate"][i]) * (x @ W["w_up"][i])) @ W["w_down"][i]
        y = y + dense_gate[:, cfg.e_lo + i: cfg.e_lo + i + 1] * out_e
    Ws = {}
    if cfg.I_shared:
        Ws = {n: torch.from_numpy(C.as_f64(inp[n])).requires_grad_(True) for n in ("ws_gate", "ws_up", "ws_down")}
        y = y + (torch.nn.functional.silu(x @ Ws["ws_gate"][0]) * (x @ Ws["ws_up"][0])) @ Ws["ws_down"][0]
    return x, z, g, W, Ws, y


@pytest.mark.parametrize("name", ["plain", "ep_slice_shared", "full_softmax"])
def test_dense_brute_force_forward_and_autograd_backward(name):
    cfg = {"plain": small_cfg(T=16, E=4, k=2),
           "ep_slice_shared": small_cfg(T=16, E=8, k=3, e_lo=2, E_loc=4, I_shared=10, gate_mode=1, bias="normal0.5"),
           "full_softmax": small_cfg(T=12, E=5, k=2, gate_mode=2)}[name]
    inp = C.make_inputs(cfg)
    inp["logits"] = spread_logits(cfg, np.random.default_rng(8))
    f = O.forward(cfg, inp)
    b = O.backward(cfg, inp, f)
    x, z, g, W, Ws, y = dense_reference(cfg, inp, f["topk_idx"])
    np.testing.assert_allclose(f["y"], y.detach().numpy(), rtol=1e-11, atol=1e-13)
    dy = torch.from_numpy(C.as_f64(inp["dy"]))
    (y * dy).sum().backward()
    tol = dict(rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(b["dw_gate"], W["w_gate"].grad.numpy(), **tol)
    np.testing.assert_allclose(b["dw_up"], W["w_up"].grad.numpy(), **tol)
    np.testing.assert_allclose(b["dw_down"], W["w_down"].grad.numpy(), **tol)
    np.testing.assert_allclose(b["dgates"], g.grad.numpy(), **tol)
    if cfg.I_shared:
        np.testing.assert_allclose(b["dws_gate"], Ws["ws_gate"].grad.numpy(), **tol)
        np.testing.assert_allclose(b["dws_up"], Ws["ws_up"].grad.numpy(), **tol)
        np.testing.assert_allclose(b["dws_down"], Ws["ws_down"].grad.numpy(), **tol)
    # x enters only through the experts here (logits are an independent input): expert-path dX
    np.testing.assert_allclose(b["dx"], x.grad.numpy(), **tol)
    # gradient w.r.t. the logits
    zg = z.grad.numpy()
    if cfg.gate_mode == 2:
        np.testing.assert_allclose(b["dz"], zg, **tol)
    else:
        np.testing.assert_allclose(b["dz"], np.take_along_axis(zg, f["topk_idx"].astype(np.int64), 1), **tol)
        mask = np.ones_like(zg, bool)
        np.put_along_axis(mask, f["topk_idx"].astype(np.int64), False, 1)
        assert (zg[mask] == 0).all()                                            # unselected logits get 0


def test_backward_finite_differences():
    """Central differences of L = <dY, Y> through the oracle's own forward, on exactly
    representable perturbations (fp32 inputs pre-rounded to 12 mantissa bits, h = 2^-9)."""
    cfg = small_cfg(T=6, E=4, k=2, d=8, I=10, I_shared=6)
    inp = C.make_inputs(cfg)
    q = lambda a: (np.round(a.astype(np.float64) * 4096) / 4096).astype(np.float32)
    for n in ("x", "w_gate", "w_up", "w_down", "ws_gate", "ws_up", "ws_down", "dy"):
        inp[n] = q(inp[n])
    inp["logits"] = q(spread_logits(cfg, np.random.default_rng(9), gap=0.25))
    f = O.forward(cfg, inp)
    b = O.backward(cfg, inp, f)
    dy = inp["dy"].astype(np.float64)
    h = 2.0 ** -9
    rng = np.random.default_rng(10)

    def loss(mod):
        return float((O.forward(cfg, mod)["y"] * dy).sum())

    def fd(name, index):
        plus = dict(inp); minus = dict(inp)
        plus[name] = inp[name].copy(); minus[name] = inp[name].copy()
        plus[name][index] += h; minus[name][index] -= h
        return (loss(plus) - loss(minus)) / (2 * h)

    grads = {"x": b["dx"], "w_gate": b["dw_gate"], "w_up": b["dw_up"], "w_down": b["dw_down"],
             "ws_gate": b["dws_gate"], "ws_up": b["dws_up"], "ws_down": b["dws_down"]}
    for name, gr in grads.items():
        for _ in range(4):
            index = tuple(int(rng.integers(0, s)) for s in gr.shape)
            np.testing.assert_allclose(gr[index], fd(name, index), rtol=2e-4, atol=2e-5)
    for _ in range(6):
        t, j = int(rng.integers(0, cfg.T)), int(rng.integers(0, cfg.k))
        np.testing.assert_allclose(b["dz"][t, j], fd("logits", (t, int(f["topk_idx"][t, j]))), rtol=2e-4, atol=2e-5)


def test_gate_backward_identities():
    for mode in (0, 1):
        cfg = small_cfg(T=40, E=10, k=4, gate_mode=mode)
        rng = np.random.default_rng(11)
        z = rng.normal(size=(cfg.T, cfg.E)).astype(np.float32)
        idx, gates, _ = O.route_topk(cfg, z)
        dg = rng.normal(size=(cfg.T, cfg.k))
        dz = O.route_bwd(cfg, z, idx, dg)
        if mode == 0:   # gates invariant to a common shift of the selected logits
            np.testing.assert_allclose(dz.sum(1), 0, atol=1e-14)
        else:           # gates invariant to a common scaling of the selected sigmoids: sum s_j ds_j = 0
            s = 1 / (1 + np.exp(-np.take_along_axis(z.astype(np.float64), idx.astype(np.int64), 1)))
            np.testing.assert_allclose((dz / (1 - s)).sum(1), 0, atol=1e-13)


def test_empty_experts_and_row_align_independence():
    cfg = small_cfg(T=30, E=6, k=2, bias="zipf1.2", n_dead=2)
    inp = C.make_inputs(cfg)
    f1 = O.forward(cfg, inp)
    b1 = O.backward(cfg, inp, f1)
    assert (f1["counts"][-2:] == 0).all()
    assert (b1["dw_gate"][-2:] == 0).all() and (b1["dw_up"][-2:] == 0).all() and (b1["dw_down"][-2:] == 0).all()
    cfg8 = dataclasses.replace(cfg, row_align=8)
    f8 = O.forward(cfg8, inp)
    b8 = O.backward(cfg8, inp, f8)
    assert f8["offsets"][-1] > f1["offsets"][-1]
    np.testing.assert_allclose(f8["y"], f1["y"], rtol=1e-13, atol=1e-15)
    for n in ("dx", "dw_gate", "dw_up", "dw_down", "dgates", "dz"):
        np.testing.assert_allclose(b8[n], b1[n], rtol=1e-12, atol=1e-14)
    pad = f8["src_of"] < 0
    assert (f8["xp"][pad] == 0).all() and (f8["o"][pad] == 0).all() and (b8["dxp"][pad] == 0).all()


def test_sampled_forms_equal_full_tensors():
    cfg = dataclasses.replace(C.C1S, T=60)
    inp = C.make_inputs(cfg)
    f = O.forward(cfg, inp)
    b = O.backward(cfg, inp, f)
    rt = O.routing(cfg, inp)
    for n in ("topk_idx", "row_of", "src_of", "counts", "offsets"):
        assert (rt[n] == f[n]).all()
    toks = [0, 7, 33, 59]
    s = O.sample_tokens(cfg, inp, rt, toks)
    tol = dict(rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(s["y"], f["y"][toks], **tol)
    np.testing.assert_allclose(s["dx"], b["dx"][toks], **tol)
    np.testing.assert_allclose(s["dgates"], b["dgates"][toks], **tol)
    np.testing.assert_allclose(s["o_rows"], f["o"][s["rows"]], **tol)
    np.testing.assert_allclose(s["dxp_rows"], b["dxp"][s["rows"]], **tol)
    np.testing.assert_allclose(O.sample_route_bwd(cfg, inp, rt, toks, s["dgates"]), b["dz"][toks], **tol)
    rows = np.nonzero(rt["src_of"] >= 0)[0][::3]
    sr = O.sample_rows(cfg, inp, rt, rows)
    np.testing.assert_allclose(sr["o"], f["o"][rows], **tol)
    np.testing.assert_allclose(sr["h"], f["h"][rows], **tol)
    np.testing.assert_allclose(sr["dxp"], b["dxp"][rows], **tol)
    np.testing.assert_allclose(sr["dg"], b["dg"][rows], **tol)
    np.testing.assert_allclose(sr["du"], b["du"][rows], **tol)
    J = np.array([0, 5, cfg.I - 1], np.int32)
    for e in range(cfg.e_loc):
        dwg, dwu, dwd = O.sample_wgrad(cfg, inp, rt, e, J)
        np.testing.assert_allclose(dwg, b["dw_gate"][e][:, J], **tol)
        np.testing.assert_allclose(dwu, b["dw_up"][e][:, J], **tol)
        np.testing.assert_allclose(dwd, b["dw_down"][e][J, :], **tol)
    Js = np.array([1, cfg.I_shared - 1], np.int32)
    dwg, dwu, dwd = O.sample_wgrad_shared(cfg, inp, Js)
    np.testing.assert_allclose(dwg, b["dws_gate"][0][:, Js], **tol)
    np.testing.assert_allclose(dwu, b["dws_up"][0][:, Js], **tol)
    np.testing.assert_allclose(dwd, b["dws_down"][0][Js, :], **tol)


def test_bf16_inputs_are_read_exactly():
    cfg = small_cfg(T=10, E=4, k=2, dtype=C.DT_BF16)
    inp = C.make_inputs(cfg)
    assert inp["x"].dtype == np.uint16
    f = O.forward(cfg, inp)
    cfg32 = dataclasses.replace(cfg, dtype=C.DT_F32)
    inp32 = {k_: (C.as_f64(v).astype(np.float32) if isinstance(v, np.ndarray) and v.dtype == np.uint16 else v)
             for k_, v in inp.items()}
    f32 = O.forward(cfg32, inp32)
    assert (f["y"] == f32["y"]).all()


# ---------------------------------------------------------------------------------- scheduler
def test_list_scheduler_golden_order():
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "pair_dag.json")))
    n = len(g["nodes"])
    order, n_desc, waits, records = O.list_schedule(n, g["edges"], g["stream_of"], g["prio"])
    assert n_desc.tolist() == g["n_desc"]
    assert order.tolist() == g["order"]
    so = g["stream_of"]
    assert [v for v in order if so[v] == 0] == g["q_comm"]
    assert [v for v in order if so[v] == 1] == g["q_gemm"]
    assert {tuple(w) for w in waits.tolist()} == {tuple(w) for w in g["waits"]}
    assert np.nonzero(records)[0].tolist() == g["records"]
    # every dependency is either same-queue-earlier or has a record/wait pair
    pos = {int(v): i for i, v in enumerate(order)}
    for s, t in g["edges"]:
        assert pos[s] < pos[t]
        if so[s] != so[t]:
            assert (s, t) in {tuple(w) for w in waits.tolist()} and records[s] == 1


# ------------------------------------------------------------------------------------ input recipe of the microbenchmark
@pytest.mark.parametrize("rows", [16, 64, 200])
def test_uniform_logits_give_every_expert_the_same_rows(rows):
    """bench.py --uniform-rows: the crafted logits must route exactly `rows` rows to each of the 32 experts, token t to
    experts (t k + j) mod E in that order (checked with the oracle's routing, the definition of SURVEY.md §8c-1)."""
    cfg = C.uniform_config(rows)
    z = C.uniform_logits(cfg)
    idx, gates, cg = O.route_topk(cfg, z)
    assert (cg == rows).all() and cg.sum() == cfg.T * cfg.k
    t = np.arange(cfg.T)[:, None]
    assert (idx == (t * cfg.k + np.arange(cfg.k)[None, :]) % cfg.E).all()
    assert (np.diff(gates, axis=1) < 0).all()  # descending preference -> descending gates
