"""GPU parity of the router GEMMs (Listing 1 `self.router(x)`) against the CPU oracle:
z = x W_r + bias feeding F1, dW_r = x^T dz, dX += dz W_r^T, as step calls and inside the chunk calls.

Routing parity on GPU-computed logits (reading c-18): the fp32 logits differ from the exactly rounded
sum by fp32 accumulation error, so a token's selection may differ from the oracle's only where the gap between its k-th and
(k+1)-th largest logit is below EPS_GAP; such rows are counted and must be rare."""
import dataclasses
import os

import numpy as np
import pytest
import torch

import paper_2606_11169_b200 as piper
from inputs import configs
from oracle import oracle
import piper_testutil as util

pytestmark = pytest.mark.gpu

# fp32 accumulation of K = d <= 7168 exact products of magnitude ~0.02: error ~ sqrt(d) * 2^-24 * |z| ~ 1e-5 at most
EPS_GAP = 1e-4
LOGIT_TOL = 1e-5  # north_star's fp32 bar; measured 4.5e-6 at d = 4096 (sequential fp32 accumulation: sqrt(d) * 2^-24)


def _router_inputs(cfg):
    inp = configs.make_inputs(cfg)
    dev = util.upload_inputs(inp)
    dev["w_r"] = util.to_dev(inp["w_r"])
    dev["router_bias"] = torch.from_numpy(inp["bias"]).cuda()
    return inp, dev


def _routing_agrees(cfg, z_ref64, idx_gpu):
    """Rows whose selection differs from the oracle's must have a k / (k+1) gap below EPS_GAP; returns their count."""
    idx_ref, _, _ = oracle.route_topk(cfg, z_ref64.astype(np.float32))
    bad = np.nonzero((idx_ref != idx_gpu).any(axis=1))[0]
    srt = -np.sort(-z_ref64[bad], axis=1)
    for r, t in enumerate(bad):
        # the two selections differ by experts whose logits are within EPS_GAP of each other
        a, b = set(idx_ref[t].tolist()), set(idx_gpu[t].tolist())
        diff = sorted(a ^ b)
        if diff:
            vals = z_ref64[t, diff]
            assert vals.max() - vals.min() < EPS_GAP, (t, diff, vals)
        else:  # same set, different order: two selected logits within EPS_GAP
            assert np.min(np.abs(np.diff(srt[r, : cfg.k]))) < EPS_GAP, t
    return len(bad)


@pytest.mark.parametrize("name", ["C1", "C1s", "C2s", "C3s", "C4s", "C6s"])
def test_router_step_calls_against_the_oracle(name):
    base = configs.BY_NAME[name]
    cfg = dataclasses.replace(base, row_align=128 if base.dtype == configs.DT_BF16 else 1)
    inp, dev = _router_inputs(cfg)
    ctx = piper.Context(util.desc_of(cfg))
    rb = piper.alloc_router_buffers(ctx)
    piper.piper_router_fwd(ctx, dev["x"], dev["w_r"], dev["router_bias"], rb["logits"])
    torch.cuda.synchronize()
    z_ref = oracle.router_fwd(cfg, inp["x"], inp["w_r"], inp["bias"])
    got = util.to_np(rb["logits"])
    finite = np.isfinite(z_ref)  # dead experts carry a -inf bias (variant C4z / n_dead)
    assert np.array_equal(np.isfinite(got), finite)
    frob, _ = util.errs(got[finite], z_ref[finite])
    assert frob <= (1e-5 if cfg.dtype == configs.DT_F32 else LOGIT_TOL), frob
    # F1 on the GPU's own logits
    b = piper.alloc_buffers(ctx)
    piper.piper_route_topk(ctx, rb["logits"], b["topk_idx"], b["gates"], b["counts_global"])
    torch.cuda.synchronize()
    n_bad = _routing_agrees(cfg, z_ref, util.to_np(b["topk_idx"]))
    assert n_bad <= max(1, cfg.T // 200), n_bad
    # backward from the oracle's dz on the generator's logits (the same routing on both sides)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    dz_dev = torch.from_numpy(g["dz"].astype(np.float32)).cuda()
    idx_dev = torch.from_numpy(f["topk_idx"]).cuda()
    piper.piper_router_bwd(ctx, dev["x"], dev["w_r"], idx_dev, dz_dev, rb["dz_scratch"], rb["dw_r"], rb["dx_router"])
    torch.cuda.synchronize()
    dw_ref, dx_ref = oracle.router_bwd(cfg, inp["x"], inp["w_r"], oracle.dense_dz(cfg, f["topk_idx"], g["dz"]))
    # dW_r is an fp32 output of exact products with a 2^-17 split of dz: fp32-level; dX_r is rounded to the layer dtype
    util.check_close("dw_r", util.to_np(rb["dw_r"]), dw_ref, configs.DT_F32, scale=20.0 if cfg.dtype == configs.DT_BF16 else 1.0)
    util.check_close("dx_router", util.to_np(rb["dx_router"]), dx_ref, cfg.dtype)
    ctx.close()


@pytest.mark.parametrize("name", ["C1", "C3s", "C4s"])
def test_chunk_calls_with_the_router_on_the_path(name):
    """piper_chunk_args.w_r != NULL: the forward chunk computes the logits itself, the backward chunk adds dW_r and the
    router's term of dX.  With the GPU's routing equal to the oracle's (checked), Y / dX (both paths) / dW match."""
    base = configs.BY_NAME[name]
    cfg = dataclasses.replace(base, row_align=128 if base.dtype == configs.DT_BF16 else 1)
    inp, dev = _router_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx = piper.Context(util.desc_of(cfg))
    b = piper.alloc_buffers(ctx)
    b.update(dev)
    b.update(piper.alloc_router_buffers(ctx))  # logits becomes an output
    b["logits"].fill_(float("nan"))
    args = piper.chunk_args(b)
    piper.piper_run_chunk_fwd(ctx, args)
    piper.piper_run_chunk_bwd(ctx, args)
    torch.cuda.synchronize()
    if not np.array_equal(util.to_np(b["topk_idx"]), f["topk_idx"]):
        z_ref = oracle.router_fwd(cfg, inp["x"], inp["w_r"], inp["bias"])
        _routing_agrees(cfg, z_ref, util.to_np(b["topk_idx"]))
        pytest.skip("a near-tie flipped a selection on this seed: covered by the routing-agreement rule")
    dt = cfg.dtype
    util.check_close("y", util.to_np(b["y"]), f["y"], dt)
    dw_ref, dx_ref = oracle.router_bwd(cfg, inp["x"], inp["w_r"], oracle.dense_dz(cfg, f["topk_idx"], g["dz"]))
    util.check_close("dx (expert + router path)", util.to_np(b["dx"]), g["dx"] + dx_ref, dt)
    util.check_close("dz_sel", util.to_np(b["dz_sel"]), g["dz"], dt)
    # dz on the GPU comes from bf16 O rows (dgates): dW_r carries the layer's tolerance, not fp32's
    util.check_close("dw_r", util.to_np(b["dw_r"]), dw_ref, dt)
    for n in ("dw_gate", "dw_up", "dw_down"):
        util.check_close(n, util.to_np(b[n]), g[n], dt)
    # Bi + Bw and the pair take the same path (B.route_bwd precedes B.unpack)
    ref_dx = b["dx"].clone()
    b["dx"].zero_()
    piper.piper_run_chunk_bwd_input(ctx, args)
    torch.cuda.synchronize()
    assert torch.equal(ref_dx, b["dx"])
    b["dx"].zero_()
    b2 = piper.alloc_buffers(ctx)  # a second microbatch (same inputs) for the forward side of the pair
    b2.update(dev)
    b2.update(piper.alloc_router_buffers(ctx))
    piper.piper_set_pair_policy(ctx, piper.ORDER_LIST, piper.PART_SHARED)
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    piper.piper_run_chunk_pair(ctx, piper.chunk_args(b2), args, n_sm, 32)
    torch.cuda.synchronize()
    assert torch.equal(ref_dx, b["dx"]) and torch.equal(b2["y"], b["y"]) and torch.equal(b2["logits"], b["logits"])
    ctx.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_full_size_router_logits_and_selection(name):
    """BASELINE.json full sizes: logits of 256 sampled tokens against the oracle, selections on all tokens against the
    oracle's on the generator's logits under the near-tie rule."""
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=128)
    inp = configs.make_inputs(cfg, weights=False, with_dy=False)
    ctx = piper.Context(util.desc_of(cfg))
    x, w_r = util.to_dev(inp["x"]), util.to_dev(inp["w_r"])
    bias = torch.from_numpy(inp["bias"]).cuda()
    rb = piper.alloc_router_buffers(ctx)
    piper.piper_router_fwd(ctx, x, w_r, bias, rb["logits"])
    b = piper.alloc_buffers(ctx, backward=False)
    piper.piper_route_topk(ctx, rb["logits"], b["topk_idx"], b["gates"], b["counts_global"])
    torch.cuda.synchronize()
    rng = np.random.default_rng(cfg.seed)
    tok = np.sort(np.concatenate([[0, 127, 128, cfg.T - 1], rng.choice(cfg.T, 252, replace=False)])).astype(np.int64)
    sub = dataclasses.replace(cfg, T=len(tok))
    oracle.set_threads(os.cpu_count() or 1)
    z_ref = oracle.router_fwd(sub, np.ascontiguousarray(inp["x"][tok]), inp["w_r"], inp["bias"])
    got = util.to_np(rb["logits"])[tok]
    frob, _ = util.errs(got, z_ref)
    assert frob <= LOGIT_TOL, frob
    # every token: the generator's logits are the exactly rounded sums (pinned on CPU against oracle.router_fwd)
    n_bad = _routing_agrees(cfg, inp["logits"].astype(np.float64), util.to_np(b["topk_idx"]))
    assert n_bad <= cfg.T // 500, n_bad
    ctx.close()
