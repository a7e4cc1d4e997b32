"""GPU parity tests: the CUDA path through the C-ABI (paper_2606_11169_b200.binding) against the CPU
oracle (oracle/) on the same seeded inputs (inputs/).  Integer / index outputs bit-exact; floating
point within the north_star tolerances (tests/piper_testutil.py: TOL)."""
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

SMALL = ["C1", "C1s", "C2s", "C3s", "C4s", "C6s"]


def _run_steps(cfg, inp, gemm_impl=piper.GEMM_AUTO, use_chunk_calls=False, backward=True, overlap=False, options=()):
    """Runs the whole path; returns (ctx, dict of device tensors)."""
    ctx = piper.Context(util.desc_of(cfg, gemm_impl))
    for opt, val in options:
        piper.piper_set_option(ctx, opt, val)
    if overlap:
        piper.piper_set_chunk_overlap(ctx, 1)
    dev = util.upload_inputs(inp)
    b = piper.alloc_buffers(ctx, backward=True)
    b.update(dev)
    if use_chunk_calls:
        args = piper.chunk_args(b)
        piper.piper_run_chunk_fwd(ctx, args)
        if backward:
            piper.piper_run_chunk_bwd(ctx, args)
        if piper.piper_chunk_gathers(ctx):
            # N2 fusion: the chunk's GEMMs gathered x / dY rows themselves and xp was not materialised; the all-to-all
            # payload comes from the pack task (= piper_dispatch_pack's second half)
            piper.piper_run_task(ctx, "F_PACK", args)
    else:
        piper.piper_route_topk(ctx, b["logits"], b["topk_idx"], b["gates"], b["counts_global"])
        piper.piper_dispatch_pack(ctx, b["x"], b["topk_idx"], b["gates"], b["counts"], b["offsets"], b["row_of"],
                                  b["src_of"], b["gate_rows"], b["xp"])
        piper.piper_expert_ffn_fwd(ctx, b["xp"], b["offsets"], b["w_gate"], b["w_up"], b["w_down"], b["g_save"],
                                   b["u_save"], b["h_save"], b["o"])
        if cfg.I_shared:
            piper.piper_shared_ffn_fwd(ctx, b["x"], b["ws_gate"], b["ws_up"], b["ws_down"], b["gs_save"], b["us_save"],
                                       b["hs_save"], b["s"])
        piper.piper_combine(ctx, b["o"], b["row_of"], b["gates"], b.get("s"), b["y"])
        if backward:
            piper.piper_combine_bwd(ctx, b["dy"], b["o"], b["src_of"], b["row_of"], b["gates"], b["offsets"], b["d_o"],
                                    b["dgates"])
            piper.piper_expert_ffn_bwd(ctx, b["d_o"], b["xp"], b["g_save"], b["u_save"], b["h_save"], b["offsets"],
                                       b["w_gate"], b["w_up"], b["w_down"], b["dg"], b["du"], b["dxp"], b["dw_gate"],
                                       b["dw_up"], b["dw_down"])
            if cfg.I_shared:
                piper.piper_shared_ffn_bwd(ctx, b["dy"], b["x"], b["gs_save"], b["us_save"], b["hs_save"], b["ws_gate"],
                                           b["ws_up"], b["ws_down"], b["dgs"], b["dus"], b["dxs"], b["dws_gate"],
                                           b["dws_up"], b["dws_down"])
            piper.piper_dispatch_unpack(ctx, b["dxp"], b["row_of"], b.get("dxs"), b["dx"])
            piper.piper_route_bwd(ctx, b["logits"], b["topk_idx"], b["gates"], b["dgates"], b["dz_sel"])
    torch.cuda.synchronize()
    return ctx, b


def _check_routing(cfg, b, ref):
    A = int(ref["offsets"][-1])
    for name in ("topk_idx", "counts_global", "counts", "row_of"):
        assert np.array_equal(util.to_np(b[name]).reshape(-1), ref[name].reshape(-1)), name
    assert np.array_equal(util.to_np(b["offsets"])[: cfg.e_loc + 1], ref["offsets"])
    assert np.array_equal(util.to_np(b["src_of"]), ref["src_of"])
    util.check_close("gates", util.to_np(b["gates"]), ref["gates"], configs.DT_F32)
    util.check_close("gate_rows", util.to_np(b["gate_rows"])[:A], ref["gate_rows"][:A], configs.DT_F32)
    return A


def _check_all(cfg, b, f, g, label=""):
    A = _check_routing(cfg, b, f)
    dt = cfg.dtype
    assert np.array_equal(util.to_np(b["xp"])[:A], f["xp"][:A]), "xp must be a bit-exact copy"
    out = {}
    out["o"] = util.check_close(label + "o", util.to_np(b["o"])[:A], f["o"][:A], dt)
    out["y"] = util.check_close(label + "y", util.to_np(b["y"]), f["y"], dt)
    if g is None:
        return out
    out["dgates"] = util.check_close(label + "dgates", util.to_np(b["dgates"]), g["dgates"], dt)
    out["dz"] = util.check_close(label + "dz_sel", util.to_np(b["dz_sel"]), g["dz"], dt)
    out["dxp"] = util.check_close(label + "dxp", util.to_np(b["dxp"])[:A], g["dxp"][:A], dt)
    out["dx"] = util.check_close(label + "dx", util.to_np(b["dx"]), g["dx"], dt)
    for n in ("dw_gate", "dw_up", "dw_down"):
        out[n] = util.check_close(label + n, util.to_np(b[n]), g[n], dt)
    if cfg.I_shared:
        for n in ("dws_gate", "dws_up", "dws_down"):
            out[n] = util.check_close(label + n, util.to_np(b[n]), g[n][0], dt)
    # exact zeros for empty experts (Definition 5)
    for i in np.nonzero(f["counts"] == 0)[0]:
        for n in ("dw_gate", "dw_up", "dw_down"):
            assert not util.to_np(b[n][int(i)]).any(), f"{n}[{i}] must be exactly zero for an empty expert"
    return out


@pytest.mark.parametrize("name", SMALL)
@pytest.mark.parametrize("impl", [piper.GEMM_AUTO, piper.GEMM_SIMT])
@pytest.mark.parametrize("align", [1, 16, 128])  # 16 / 128: the tcgen05 kernels; 1: dense packing, FP32-ALU GEMMs only
def test_small_configs_full_tensor_parity(name, impl, align):
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=align)
    if cfg.dtype == configs.DT_F32 and impl == piper.GEMM_SIMT:
        pytest.skip("fp32 already runs the FP32-ALU kernels under GEMM_AUTO")
    if cfg.dtype == configs.DT_BF16 and impl == piper.GEMM_AUTO and align % 16:
        # no silent ~100x slower path: a bf16 layer the tcgen05 kernels cannot take is refused at creation
        with pytest.raises(piper.PiperError):
            piper.Context(util.desc_of(cfg, impl))
        return
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp, gemm_impl=impl)
    _check_all(cfg, b, f, g)
    assert piper.piper_gemm_path(ctx) == (1 if cfg.dtype == configs.DT_BF16 and impl == piper.GEMM_AUTO else 0)
    ctx.close()


def _random_config(i):
    """Seeded random layer shapes: every dimension a multiple of 8 only, experts from empty to several row chunks,
    local slices, shared expert or not, all three gate modes."""
    rng = np.random.default_rng(1000 + i)
    E = int(rng.choice([2, 5, 8, 24]))
    k = int(rng.integers(1, min(E, 6) + 1))
    e_loc = int(rng.integers(1, E + 1))
    e_lo = int(rng.integers(0, E - e_loc + 1))
    return configs.MoeConfig(f"R{i}", T=int(rng.integers(1, 1400)), d=8 * int(rng.integers(8, 70)), E=E, k=k,
                             I=8 * int(rng.integers(8, 70)), seed=2000 + i, e_lo=e_lo, E_loc=e_loc,
                             I_shared=int(rng.choice([0, 8 * int(rng.integers(8, 40))])),
                             gate_mode=int(rng.integers(0, 3)), bias=str(rng.choice(["none", "normal0.5", "zipf1.2"])),
                             n_dead=int(rng.integers(0, 2)) if E > k + 1 else 0, row_align=int(rng.choice([16, 32, 128])))


@pytest.mark.parametrize("i", range(8))
def test_random_shapes_full_tensor_parity(i):
    cfg = _random_config(i)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp, use_chunk_calls=True)
    _check_all(cfg, b, f, g, label=f"{cfg} ")
    assert piper.piper_gemm_path(ctx) == 1
    ctx.close()


@pytest.mark.parametrize("name", ["C3s", "C4s"])
def test_chunk_calls_capture_into_a_cuda_graph(name):
    """The chunk calls only enqueue work on the caller's stream (no host read-back, no allocation), so a step can be
    captured in a CUDA graph; the replay is bit-identical to the eager run (the tile counters of the persistent
    kernels re-arm themselves)."""
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=128)
    inp = configs.make_inputs(cfg)
    ctx, b = _run_steps(cfg, inp, use_chunk_calls=True)
    names = ("y", "dx", "dz_sel", "dw_gate", "dw_up", "dw_down", "row_of")
    ref = {n: b[n].clone() for n in names}
    args = piper.chunk_args(b)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        piper.piper_run_chunk_fwd(ctx, args)
        piper.piper_run_chunk_bwd(ctx, args)
    for rep in range(2):
        for n in names:
            b[n].fill_(-1 if b[n].dtype == torch.int32 else 7.0)
        graph.replay()
        torch.cuda.synchronize()
        for n in names:
            assert torch.equal(ref[n], b[n]), (n, rep)
    ctx.close()


def test_more_local_experts_than_the_cta_pair_kernels_index():
    """256 local experts (> 192, the group bound of the CTA-pair kernels' tile-prefix arrays): every GEMM takes the
    1-CTA tcgen05 kernels without any switch; many experts are short or empty."""
    cfg = configs.MoeConfig("many", T=1500, d=128, E=256, k=4, I=192, seed=31, bias="zipf1.2", row_align=128)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp, use_chunk_calls=True)
    _check_all(cfg, b, f, g)
    assert piper.piper_gemm_path(ctx) == 1
    ctx.close()


@pytest.mark.parametrize("name", ["C3s", "C4s", "C6s"])
@pytest.mark.parametrize("family", ["rows_on_m", "one_cta", "dual_tiles", "wgrad_store_warp", "wgrad_warp_stores",
                                    "greedy_chunks", "equal_chunks"])
def test_fallback_kernel_families(name, family):
    """The rows-on-M CTA-pair kernels and the 1-CTA kernels (DESIGN.md section 5.1 b, c) stay correct: they serve
    layers with more than 192 local experts; so do the two-chunk tiles of the plain-store rows-on-N kernels (a measured
    variant).  piper_set_option selects them (host state of the context)."""
    if family in ("dual_tiles", "wgrad_store_warp", "wgrad_warp_stores", "greedy_chunks", "equal_chunks"):
        # wgrad: both ways of storing dW (the default picks one by the expected group length); rows-on-N kernels: both
        # ways of cutting an expert's rows into chunks (256-row chunks and a short last one / equal chunks)
        opt = {"dual_tiles": (piper.OPT_T_DUAL, 1), "wgrad_store_warp": (piper.OPT_WGRAD_STORE_WARP, 1),
               "wgrad_warp_stores": (piper.OPT_WGRAD_STORE_WARP, 0), "greedy_chunks": (piper.OPT_T_GREEDY, 1),
               "equal_chunks": (piper.OPT_T_GREEDY, 0)}[family]
        cfg = dataclasses.replace(configs.BY_NAME[name], row_align=16)
        inp = configs.make_inputs(cfg)
        f = oracle.forward(cfg, inp)
        ctx, b = _run_steps(cfg, inp, use_chunk_calls=True, options=[opt])
        _check_all(cfg, b, f, oracle.backward(cfg, inp, f))
        ctx.close()
        return
    opts = [(piper.OPT_TC_ROWS_ON_N, 0)] + ([(piper.OPT_TC_2CTA, 0)] if family == "one_cta" else [])
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=128)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp, use_chunk_calls=True, options=opts)
    _check_all(cfg, b, f, g)
    assert piper.piper_gemm_path(ctx) == 1
    ctx.close()
    # these families need whole 128-row tiles: at row_align 16 the switch is refused and the context keeps its kernels
    ctx = piper.Context(util.desc_of(dataclasses.replace(cfg, row_align=16)))
    with pytest.raises(piper.PiperError):
        piper.piper_set_option(ctx, piper.OPT_TC_ROWS_ON_N, 0)
    assert piper.piper_get_option(ctx, piper.OPT_TC_ROWS_ON_N) == 1
    ctx.close()


@pytest.mark.parametrize("name", ["C3s", "C4s"])
@pytest.mark.parametrize("items,cap", [(1, 1), (3, 5), (64, 64)])
def test_row_mover_grid_options(name, items, cap):
    """PIPER_OPT_MOVE_ITEMS / PIPER_OPT_MOVE_CAP only size the row movers' grids and column splits: any value gives the
    same bits as the defaults (and therefore the oracle's results)."""
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=16)
    inp = configs.make_inputs(cfg)
    ctx0, ref = _run_steps(cfg, inp, use_chunk_calls=True)
    ctx0.close()
    ctx, b = _run_steps(cfg, inp, use_chunk_calls=True, options=[(piper.OPT_MOVE_ITEMS, items), (piper.OPT_MOVE_CAP, cap)])
    A = int(ref["offsets"][cfg.e_loc].item())
    for n in ("xp", "y", "d_o", "dgates", "dx"):
        x, y = (ref[n][:A], b[n][:A]) if n in ("xp", "d_o") else (ref[n], b[n])
        assert torch.equal(x.view(torch.uint8), y.view(torch.uint8)), n
    ctx.close()


@pytest.mark.parametrize("name", ["C2s", "C3s", "C4s", "C6s"])
def test_poisoned_buffers_and_untouched_capacity(name):
    """No result may depend on what a buffer held before (pad rows are written, never assumed), and no kernel may
    write past the used rows: every output / scratch buffer starts as NaN (0x7FC1 / int 0x7FC17FC1 patterns), the
    chunk calls run, the results match the oracle, dW is finite, and the rows of the row buffers beyond
    offsets[E_loc] still hold the poison.  (compute-sanitizer is closed on this pool; this is the bounds check.)"""
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=128)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx = piper.Context(util.desc_of(cfg))
    b = piper.alloc_buffers(ctx, backward=True)
    for t in b.values():
        t.view(torch.int16).fill_(0x7FC1)
    b.update(util.upload_inputs(inp))
    args = piper.chunk_args(b)
    piper.piper_run_chunk_fwd(ctx, args)
    piper.piper_run_chunk_bwd(ctx, args)
    piper.piper_run_task(ctx, "F_PACK", args)  # the fused chunk calls do not materialise xp
    torch.cuda.synchronize()
    A = _check_all(cfg, b, f, g) and int(f["offsets"][-1])
    poison = torch.tensor(0x7FC1, dtype=torch.int16, device=b["xp"].device)
    for n in ("xp", "g_save", "u_save", "h_save", "o", "d_o", "dg", "du", "dxp"):
        assert bool((b[n][A:].view(torch.int16) == poison).all()), f"{n}: rows beyond offsets[E_loc] were written"
        assert bool(torch.isfinite(b[n][:A].float()).all()), f"{n}: non-finite value inside the used rows"
    for n in ("dw_gate", "dw_up", "dw_down", "y", "dx"):
        assert bool(torch.isfinite(b[n].float()).all()), n
    ctx.close()


@pytest.mark.parametrize("name", ["C2s", "C3s", "C4s", "C6s"])
def test_fp32_dw_and_accumulate(name):
    """Reading c-17: dW accumulated in fp32 over the whole ragged K; with dw_dtype = F32 it is written unrounded, and
    accumulate = 1 adds it into dW (main-grad style).  Two backward passes over the same microbatch, the second
    accumulating, must give twice the oracle's dW; empty experts stay exactly zero."""
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=128)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx = piper.Context(util.desc_of(cfg, dw_dtype=piper.DT_F32))
    b = piper.alloc_buffers(ctx, backward=True)
    assert b["dw_gate"].dtype == torch.float32
    b.update(util.upload_inputs(inp))
    args = piper.chunk_args(b)
    piper.piper_run_chunk_fwd(ctx, args)
    piper.piper_run_chunk_bwd(ctx, args)
    torch.cuda.synchronize()
    names = ["dw_gate", "dw_up", "dw_down"] + (["dws_gate", "dws_up", "dws_down"] if cfg.I_shared else [])
    ref = {n: (g[n] if n.startswith("dw_") else g[n][0]) for n in names}
    for n in names:
        util.check_close(n + " fp32", util.to_np(b[n]), ref[n], cfg.dtype)
    first = {n: b[n].clone() for n in names}
    piper.piper_set_wgrad_accumulate(ctx, 1)
    piper.piper_run_chunk_bwd(ctx, args)
    torch.cuda.synchronize()
    for n in names:
        assert torch.equal(b[n], first[n] + first[n]), n + ": accumulate must add the same fp32 sums"
        util.check_close(n + " accumulated", util.to_np(b[n]), 2.0 * ref[n], cfg.dtype)
    for i in np.nonzero(f["counts"] == 0)[0]:
        assert not util.to_np(b["dw_gate"][int(i)]).any()
    # the step call takes the flag as an argument
    piper.piper_set_wgrad_accumulate(ctx, 0)
    piper.piper_expert_ffn_bwd(ctx, b["d_o"], b["xp"], b["g_save"], b["u_save"], b["h_save"], b["offsets"], b["w_gate"],
                               b["w_up"], b["w_down"], b["dg"], b["du"], b["dxp"], b["dw_gate"], b["dw_up"], b["dw_down"],
                               accumulate=1)
    torch.cuda.synchronize()
    assert torch.equal(b["dw_down"], first["dw_down"] * 3.0)
    ctx.close()
    # bf16 dW cannot accumulate
    ctx2 = piper.Context(util.desc_of(cfg))
    with pytest.raises(piper.PiperError):
        piper.piper_set_wgrad_accumulate(ctx2, 1)
    ctx2.close()


@pytest.mark.parametrize("name", ["C1", "C3s", "C4s"])
def test_chunk_calls_equal_step_calls_bitwise(name):
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=128 if name != "C1" else 1)
    inp = configs.make_inputs(cfg)
    ctx1, b1 = _run_steps(cfg, inp)
    A = int(b1["offsets"][cfg.e_loc])
    for overlap in (False, True):  # piper_set_chunk_overlap: row movers on the library's side stream
        ctx2, b2 = _run_steps(cfg, inp, use_chunk_calls=True, overlap=overlap)
        for n in ("topk_idx", "gates", "counts", "row_of", "src_of", "y", "dgates", "dz_sel", "dx", "dw_gate", "dw_up",
                  "dw_down") + (("dws_gate", "dws_up", "dws_down") if cfg.I_shared else ()):
            assert torch.equal(b1[n], b2[n]), (n, overlap)
        for n in ("xp", "o", "dxp"):
            assert torch.equal(b1[n][:A], b2[n][:A]), (n, overlap)
        ctx2.close()
    ctx1.close()


@pytest.mark.parametrize("name", ["C2s", "C3s", "C4s", "C6s"])
@pytest.mark.parametrize("align,level", [(16, 1), (128, 1), (16, 2), (128, 2)])
def test_fused_gather_chunk_against_the_oracle_and_the_unfused_chunk(name, align, level):
    """N2 fusion: with PIPER_OPT_FUSED_GATHER the chunk calls run no pack kernel,
    F_GEMM1 and the gate|up wgrad gather the rows of x through src_of, DGRAD1 gathers the rows of dY and applies the gate
    to dH in its fp32 epilogue.  Both modes match the oracle; the forward (exact copies of the same rows) is bit-identical
    between them, the backward differs by one bf16 rounding less; xp is never written by the fused chunk calls."""
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=align)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx0, b0 = _run_steps(cfg, inp, use_chunk_calls=True, options=[(piper.OPT_FUSED_GATHER, 0)])
    assert not piper.piper_chunk_gathers(ctx0)
    _check_all(cfg, b0, f, g, label="unfused ")
    ctx = piper.Context(util.desc_of(cfg))
    piper.piper_set_option(ctx, piper.OPT_FUSED_GATHER, level)
    assert piper.piper_chunk_gathers(ctx)
    b = piper.alloc_buffers(ctx)
    b["xp"].view(torch.int16).fill_(0x7FC1)
    b.update(util.upload_inputs(inp))
    args = piper.chunk_args(b)
    launches0 = piper.piper_kernel_launches(ctx)
    piper.piper_run_chunk_fwd(ctx, args)
    n_fwd = piper.piper_kernel_launches(ctx) - launches0
    piper.piper_run_chunk_bwd(ctx, args)
    torch.cuda.synchronize()
    poison = torch.tensor(0x7FC1, dtype=torch.int16, device="cuda")
    assert bool((b["xp"].view(torch.int16) == poison).all()), "the fused chunk calls must not write xp"
    assert n_fwd == 6 + (2 if cfg.I_shared else 0), n_fwd  # route, hist, scan+rank, gemm1, gemm2, combine (+ shared 2): no pack
    piper.piper_run_task(ctx, "F_PACK", args)
    torch.cuda.synchronize()
    err = _check_all(cfg, b, f, g, label="fused ")
    A = int(f["offsets"][-1])
    for n in ("y", "src_of", "row_of"):
        assert torch.equal(b0[n], b[n]), n
    for n in ("o", "g_save", "u_save", "h_save", "gate_rows"):
        assert torch.equal(b0[n][:A], b[n][:A]), n
    if level == 1:  # the same rows, bit for bit, reach the same kernels' tensor cores
        for n in ("dx", "dw_gate", "dw_up", "dw_down", "dgates"):
            assert torch.equal(b0[n], b[n]), n
    else:  # one rounding less on the way to dG / dU: the fused backward is at least as close to the oracle
        err0 = util.errs(util.to_np(b0["dxp"])[:A], g["dxp"][:A])[0]
        assert err["dxp"][0] <= err0 * 1.05, (err["dxp"][0], err0)
    ctx0.close(), ctx.close()


@pytest.mark.parametrize("name", ["C3s", "C4s", "C1s"])
@pytest.mark.parametrize("split,policy", [((132, 16), "list/exclusive"), ((100, 48), "list/exclusive"),
                                          ((116, 32), "profile/exclusive"), ((148, 16), "list/shared"),
                                          ((148, 48), "profile/shared"), ((148, 16), "list/chunks"),
                                          ((132, 16), "list/exclusive/bi"), ((148, 32), "profile/shared/bi")])
def test_pair_matches_the_oracle_and_equals_serial_bitwise(name, split, policy):
    """the overlapped, out-of-order plan must respect every dependency.  The pair's outputs are checked
    against the CPU oracle (both microbatches) and must equal the serial chunks bit for bit, for the paper's list order
    and the profile-guided one, on disjoint (green contexts) and on shared SM partitions, and for F || Bi followed by Bw
    (PASS = Bi, Bw)."""
    base = configs.BY_NAME[name]
    align = 128 if base.dtype == configs.DT_BF16 else 1
    cfg_a = dataclasses.replace(base, row_align=align, seed=base.seed + 100)
    cfg_b = dataclasses.replace(base, row_align=align, seed=base.seed + 200)
    inp_a, inp_b = configs.make_inputs(cfg_a), configs.make_inputs(cfg_b)
    # serial: fwd(A) ; fwd(B) (untimed producer of B's saved activations) ; bwd(B)
    ctx, ba = _run_steps(cfg_a, inp_a, use_chunk_calls=True, backward=False)
    ctx_b, bb = _run_steps(cfg_b, inp_b, use_chunk_calls=True, backward=True)
    ctx_b.close()
    # pair on fresh buffers: B's forward first, then [F(A), B(B)] co-scheduled
    pa, pb = piper.alloc_buffers(ctx), piper.alloc_buffers(ctx)
    pa.update(util.upload_inputs(inp_a)), pb.update(util.upload_inputs(inp_b))
    args_a, args_b = piper.chunk_args(pa), piper.chunk_args(pb)
    piper.piper_run_chunk_fwd(ctx, args_b)
    parts = policy.split("/")
    order, part, bi = parts[0], parts[1], len(parts) > 2
    piper.piper_set_pair_policy(ctx, piper.ORDER_PROFILE if order == "profile" else piper.ORDER_LIST,
                                {"shared": piper.PART_SHARED, "chunks": piper.PART_CHUNK_STREAMS}.get(part, piper.PART_EXCLUSIVE))
    piper.piper_set_pair_bwd_pass(ctx, piper.PASS_BI if bi else piper.PASS_B)
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    sg = min(split[0], n_sm) if part != "exclusive" else min(split[0], n_sm - split[1])
    picked = piper.piper_pair_order(ctx, sg, split[1])
    want = [t for t in piper.TASKS if (base.I_shared or t not in ("F_SHARED", "B_SHARED")) and not (bi and t == "B_WGRAD")]
    assert sorted(picked) == sorted(want)
    piper.piper_pair_prepare(ctx, sg, split[1])  # partitions, streams and the plan exist before the run
    piper.piper_run_chunk_pair(ctx, args_a, args_b, sg, split[1])
    if bi:
        piper.piper_run_chunk_bwd_weight(ctx, args_b)
    torch.cuda.synchronize()
    # disjoint partitions are green contexts or an error, never a silent fallback (piper.h)
    assert piper.piper_pair_partition_mode(ctx) == {"shared": 2, "chunks": 3}.get(part, 1)
    if part == "exclusive":  # sm_gemm + sm_comm beyond the device, and a GEMM side that is neither a multiple of 8 nor
        with pytest.raises(piper.PiperError):  # the remainder, are refused on disjoint partitions
            piper.piper_run_chunk_pair(ctx, args_a, args_b, n_sm, 16)
        with pytest.raises(piper.PiperError):
            piper.piper_run_chunk_pair(ctx, args_a, args_b, 60, 16)
    for n in ("topk_idx", "gates", "counts", "row_of", "src_of", "y"):
        assert torch.equal(ba[n], pa[n]), "fwd " + n
    nofs = base.e_loc + 1  # the offsets buffers are over-allocated; entries past E_loc+1 are never written
    assert torch.equal(ba["offsets"][:nofs], pa["offsets"][:nofs]), "fwd offsets"
    for n in ("dgates", "dz_sel", "dx", "dw_gate", "dw_up", "dw_down") + (("dws_gate", "dws_up", "dws_down") if base.I_shared else ()):
        assert torch.equal(bb[n], pb[n]), "bwd " + n
    # against the oracle: microbatch A's forward, microbatch B's forward + backward
    if piper.piper_chunk_gathers(ctx):  # the all-to-all payload of a fused chunk comes from the pack task
        piper.piper_run_task(ctx, "F_PACK", args_a), piper.piper_run_task(ctx, "F_PACK", args_b)
        torch.cuda.synchronize()
    fa = oracle.forward(cfg_a, inp_a)
    _check_all(cfg_a, pa, fa, None, label="pair A ")
    fb = oracle.forward(cfg_b, inp_b)
    _check_all(cfg_b, pb, fb, oracle.backward(cfg_b, inp_b, fb), label="pair B ")
    ctx.close()


@pytest.mark.parametrize("name", ["C1", "C3s", "C4s", "C6s"])
def test_bwd_input_then_weight_equals_bwd_bitwise(name):
    """PASS = Bi, Bw: piper_run_chunk_bwd_input leaves dX, dgates, dz_sel complete and writes no dW;
    piper_run_chunk_bwd_weight then produces the dW of piper_run_chunk_bwd bit for bit."""
    base = configs.BY_NAME[name]
    cfg = dataclasses.replace(base, row_align=128 if base.dtype == configs.DT_BF16 else 1)
    inp = configs.make_inputs(cfg)
    ctx, ref = _run_steps(cfg, inp, use_chunk_calls=True)
    b = piper.alloc_buffers(ctx)
    b.update(util.upload_inputs(inp))
    dws = ["dw_gate", "dw_up", "dw_down"] + (["dws_gate", "dws_up", "dws_down"] if cfg.I_shared else [])
    for n in dws:
        b[n].fill_(3.0)
    args = piper.chunk_args(b)
    piper.piper_run_chunk_fwd(ctx, args)
    piper.piper_run_chunk_bwd_input(ctx, args)
    torch.cuda.synchronize()
    for n in ("dgates", "dz_sel", "dx"):
        assert torch.equal(ref[n], b[n]), n
    for n in dws:
        assert bool((b[n] == 3.0).all()), n + " written by the input pass"
    piper.piper_run_chunk_bwd_weight(ctx, args)
    torch.cuda.synchronize()
    for n in dws:
        assert torch.equal(ref[n], b[n]), n
    f = oracle.forward(cfg, inp)
    _check_all(cfg, b, f, oracle.backward(cfg, inp, f))
    ctx.close()


def test_two_streams_of_one_context_run_concurrently():
    """Calls of one context on different streams may overlap on the device: every GEMM launch draws its tiles from the
    counters of its own stream (piper.h conventions).  Two microbatches, one stream each, several steps deep with no
    host synchronisation in between, against the single-stream results; then a captured graph of stream 1 replayed on
    stream 2 while stream 1 runs eager launches."""
    cfg = dataclasses.replace(configs.C4S, row_align=128)
    cfgs = [dataclasses.replace(cfg, seed=cfg.seed + 7 * i) for i in range(2)]
    inps = [configs.make_inputs(c) for c in cfgs]
    ctx, ref0 = _run_steps(cfgs[0], inps[0], use_chunk_calls=True)
    ctx1, ref1 = _run_steps(cfgs[1], inps[1], use_chunk_calls=True)
    ctx1.close()
    refs = [ref0, ref1]
    names = ("y", "dx", "dz_sel", "dw_gate", "dw_up", "dw_down")
    bufs = []
    for inp in inps:
        b = piper.alloc_buffers(ctx)
        b.update(util.upload_inputs(inp))
        bufs.append(b)
    args = [piper.chunk_args(b) for b in bufs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for step in range(12):  # 5 dynamic-feed GEMM launches per chunk call and stream
        for i in (0, 1):
            piper.piper_run_chunk_fwd(ctx, args[i], stream=streams[i])
            piper.piper_run_chunk_bwd(ctx, args[i], stream=streams[i])
    torch.cuda.synchronize()
    for i in (0, 1):
        for n in names:
            assert torch.equal(refs[i][n], bufs[i][n]), (i, n)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(streams[0]):
        with torch.cuda.graph(graph, stream=streams[0]):
            piper.piper_run_chunk_fwd(ctx, args[0], stream=streams[0])
            piper.piper_run_chunk_bwd(ctx, args[0], stream=streams[0])
    for n in names:
        bufs[0][n].zero_(), bufs[1][n].zero_()
    torch.cuda.synchronize()
    for rep in range(4):
        with torch.cuda.stream(streams[1]):
            graph.replay()
        piper.piper_run_chunk_fwd(ctx, args[1], stream=streams[0])
        piper.piper_run_chunk_bwd(ctx, args[1], stream=streams[0])
    torch.cuda.synchronize()
    for i in (0, 1):
        for n in names:
            assert torch.equal(refs[i][n], bufs[i][n]), ("graph + eager", i, n)
    ctx.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C4z"])
def test_full_size_routing_and_permutation_bit_exact(name):
    cfg = configs.BY_NAME[name]
    inp = configs.make_inputs(cfg, weights=False, with_dy=False)
    ref = oracle.routing(cfg, inp)
    # dense packing (row_align 1, the survey's default): routing / permutation / pack do not depend on the GEMM family
    ctx = piper.Context(util.desc_of(cfg, piper.GEMM_SIMT))
    x = util.to_dev(inp["x"])
    logits = util.to_dev(inp["logits"])
    A_cap = ctx.a_cap
    i32 = dict(dtype=torch.int32, device="cuda")
    topk_idx, row_of = torch.empty((cfg.T, cfg.k), **i32), torch.empty((cfg.T, cfg.k), **i32)
    cg, counts, offsets = torch.empty(cfg.E, **i32), torch.empty(cfg.e_loc, **i32), torch.empty(cfg.e_loc + 4, **i32)
    src_of = torch.empty(A_cap, **i32)
    gates = torch.empty((cfg.T, cfg.k), dtype=torch.float32, device="cuda")
    gate_rows = torch.empty(A_cap, dtype=torch.float32, device="cuda")
    xp = torch.empty((A_cap, cfg.d), dtype=ctx.torch_dtype, device="cuda")
    piper.piper_route_topk(ctx, logits, topk_idx, gates, cg)
    piper.piper_dispatch_pack(ctx, x, topk_idx, gates, counts, offsets, row_of, src_of, gate_rows, xp)
    torch.cuda.synchronize()
    b = dict(topk_idx=topk_idx, counts_global=cg, counts=counts, offsets=offsets, row_of=row_of, src_of=src_of,
             gates=gates, gate_rows=gate_rows)
    ref["gate_rows"] = np.where(ref["src_of"] >= 0, ref["gates"].reshape(-1)[np.maximum(ref["src_of"], 0)], 0.0)
    A = _check_routing(cfg, b, ref)
    assert int(ref["counts_global"].sum()) == cfg.T * cfg.k
    # xp is the all-to-all payload: bit-exact rows
    src = torch.from_numpy(ref["src_of"][:A].astype(np.int64)).cuda()
    assert torch.equal(xp[:A].view(torch.int16), x[src // cfg.k].view(torch.int16))
    ctx.close()


def test_empty_input_edge_cases():
    """One token, k = E (every expert selected once), and a local slice that receives nothing."""
    cfg = configs.MoeConfig("edge1", T=1, d=64, E=4, k=4, I=64, seed=21, dtype=configs.DT_F32)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp)
    _check_all(cfg, b, f, g)
    ctx.close()
    cfg = configs.MoeConfig("edge2", T=40, d=64, E=8, k=1, I=64, seed=22, e_lo=6, E_loc=2, n_dead=2, bias="zipf1.2",
                            row_align=16)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    assert int(f["offsets"][-1]) == 0  # nothing is routed to the dead local experts
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp)
    _check_all(cfg, b, f, g)
    assert not util.to_np(b["y"]).any() and not util.to_np(b["dx"]).any()
    ctx.close()


def _boundary_rows(cfg, rt, rng, max_chunk_edges=3):
    """Packed rows aimed at tile edges: for every non-empty local expert its first row, its last real row, and rows
    255 / 256 of up to `max_chunk_edges` of its 256-row chunks (the rows-on-N kernels cut an expert's rows into
    256-row chunks and a last one rounded up to 16 rows; a CTA of the pair holds half a chunk, so 127 / 128 too)."""
    rows = []
    for e in range(cfg.e_loc):
        lo, cnt = int(rt["offsets"][e]), int(rt["counts"][e])
        if cnt == 0:
            continue
        rows += [lo, lo + cnt - 1]
        edges = list(range(256, cnt, 256))
        if len(edges) > max_chunk_edges:
            edges = [edges[0], edges[-1]] + list(rng.choice(edges[1:-1], max_chunk_edges - 2, replace=False))
        for c in edges:
            rows += [lo + c - 1, lo + c]
        if cnt > 128:
            rows += [lo + 127, lo + 128]
    return np.unique(np.asarray(rows, np.int64))


def _feature_columns(n):
    """Columns at the edges of the 128- / 256-wide feature tiles, including the last (possibly half-empty) tile."""
    return np.unique(np.asarray([c for c in (0, 127, 128, 255, 256, n - 129, n - 128, n - 1) if 0 <= c < n], np.int64))


def _sampled_check(cfg, inp, rt, b, fwd=True, bwd=True, n_tokens=64, experts=None, label=""):
    """Full-size outputs against the oracle on a deliberate sample: packed rows at chunk / tile edges
    of every expert (O, dXp), tokens owning such rows plus random ones, the first / last token and tokens without a
    local slot (Y, dgates, dz_sel, dX), pad rows (exact zeros in xp), and dW columns at the feature-tile edges of
    every local expert (all d rows of dW_gate / dW_up, all d columns of dW_down)."""
    dt = cfg.dtype
    rng = np.random.default_rng(cfg.seed)
    experts = list(range(cfg.e_loc)) if experts is None else list(experts)
    A = int(rt["offsets"][-1])
    rows = _boundary_rows(cfg, rt, rng)
    if experts is not None:
        ex_of_row = np.searchsorted(rt["offsets"], rows, side="right") - 1
        rows = rows[np.isin(ex_of_row, experts)]
    sr = oracle.sample_rows(cfg, inp, rt, rows, backward_too=bwd)
    rows_d = torch.from_numpy(rows).cuda()
    if fwd:
        util.check_close(label + "o rows at chunk edges", util.to_np(b["o"][rows_d]), sr["o"], dt)
        # xp is the all-to-all payload: pad rows are exact zeros, every other row below offsets[E_loc] a token's row
        pad = np.nonzero(rt["src_of"][:A] < 0)[0]
        if len(pad):
            pick = torch.from_numpy(np.unique(np.concatenate([pad[:4], pad[-4:], rng.choice(pad, min(16, len(pad)))]))).cuda()
            assert not bool(b["xp"][pick].any()), "xp pad rows must be zero"
            assert not bool(b["gate_rows"][pick].any()), "gate_rows of pad rows must be zero"
    if bwd:
        util.check_close(label + "dxp rows at chunk edges", util.to_np(b["dxp"][rows_d]), sr["dxp"], dt)
    # tokens: owners of boundary rows, random local ones, the first / last token, tokens with no local slot
    local = (rt["row_of"] >= 0).any(axis=1)
    owners = np.unique(sr["tokens"])
    want = [owners[:: max(1, len(owners) // (n_tokens // 2))][: n_tokens // 2], [0, cfg.T - 1],
            np.nonzero(~local)[0][:3]]
    have = set(np.concatenate(want).tolist())
    pool = np.setdiff1d(np.nonzero(local)[0], np.fromiter(have, np.int64))
    want.append(rng.choice(pool, max(0, n_tokens - len(have)), replace=False))
    tokens = np.unique(np.concatenate(want).astype(np.int64))
    assert len(tokens) >= min(n_tokens, cfg.T)
    s = oracle.sample_tokens(cfg, inp, rt, tokens, backward_too=bwd)
    tk = torch.from_numpy(tokens).cuda()
    if fwd:
        util.check_close(label + "y", util.to_np(b["y"][tk]), s["y"], dt)
    if bwd:
        util.check_close(label + "dgates", util.to_np(b["dgates"][tk]), s["dgates"], dt)
        util.check_close(label + "dz_sel", util.to_np(b["dz_sel"][tk]), oracle.sample_route_bwd(cfg, inp, rt, tokens, s["dgates"]), dt)
        util.check_close(label + "dx", util.to_np(b["dx"][tk]), s["dx"], dt)
        J = _feature_columns(cfg.I)
        Jc = torch.from_numpy(J).cuda()
        pooled = {n: ([], []) for n in ("dw_gate", "dw_up", "dw_down")}
        for e in experts:
            if rt["counts"][e] == 0:
                for n in ("dw_gate", "dw_up", "dw_down"):
                    assert not bool(b[n][int(e)].any()), f"{n}[{e}] must be exactly zero for an empty expert"
                continue
            rg, ru, rd = oracle.sample_wgrad(cfg, inp, rt, e, J)
            got = {"dw_gate": util.to_np(b["dw_gate"][e][:, Jc]), "dw_up": util.to_np(b["dw_up"][e][:, Jc]),
                   "dw_down": util.to_np(b["dw_down"][e][Jc, :])}
            for n, ref in (("dw_gate", rg), ("dw_up", ru), ("dw_down", rd)):
                # reading c-23: the tolerance is per OUTPUT TENSOR.  A single expert's slice (a few thousand values, as few
                # as 2 rows of K) scatters around the tensor's error, so it gets twice the bound (a wrong tile, expert or
                # row range is an error of order 1); the pooled sample of all experts gets the bound itself.
                util.check_close(f"{label}{n}[{e}] sample", got[n], ref, dt, scale=2.0)
                pooled[n][0].append(got[n].reshape(-1)), pooled[n][1].append(ref.reshape(-1))
        for n, (gs, rs) in pooled.items():
            if gs:
                util.check_close(f"{label}{n} (all experts' samples)", np.concatenate(gs), np.concatenate(rs), dt)
        if cfg.I_shared:
            Js = _feature_columns(cfg.I_shared)
            Jsc = torch.from_numpy(Js).cuda()
            rg, ru, rd = oracle.sample_wgrad_shared(cfg, inp, Js)
            util.check_close(label + "dws_gate[:,J]", util.to_np(b["dws_gate"][:, Jsc]), rg, dt)
            util.check_close(label + "dws_up[:,J]", util.to_np(b["dws_up"][:, Jsc]), ru, dt)
            util.check_close(label + "dws_down[J,:]", util.to_np(b["dws_down"][Jsc, :]), rd, dt)
    return len(rows), len(tokens)


def _check_full_size_routing(cfg, b, rt):
    for n in ("topk_idx", "counts_global", "counts", "row_of", "src_of"):
        assert np.array_equal(util.to_np(b[n]).reshape(-1), rt[n].reshape(-1)), n
    assert np.array_equal(util.to_np(b["offsets"])[: cfg.e_loc + 1], rt["offsets"])
    util.check_close("gates", util.to_np(b["gates"]), rt["gates"], configs.DT_F32)


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C4z"])
def test_full_size_sampled_parity_in_bench_configuration(name):
    """BASELINE.json full sizes in the launch configuration bench.py times (row_align 128, whole-chunk calls,
    tcgen05 GEMMs): routing / permutation bit-exact on the whole tensors; everything else on the deliberate sample of
    _sampled_check, each value computed by the oracle one by one from the definition."""
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=128)
    inp = configs.make_inputs(cfg)
    oracle.set_threads(os.cpu_count() or 1)
    rt = oracle.routing(cfg, inp)
    ctx = piper.Context(util.desc_of(cfg))
    assert piper.piper_gemm_path(ctx) == 1
    b = piper.alloc_buffers(ctx)
    b.update(util.upload_inputs(inp))
    args = piper.chunk_args(b)
    piper.piper_run_chunk_fwd(ctx, args)
    piper.piper_run_chunk_bwd(ctx, args)
    piper.piper_run_task(ctx, "F_PACK", args)  # the all-to-all payload (the fused chunk calls do not materialise xp)
    torch.cuda.synchronize()
    _check_full_size_routing(cfg, b, rt)
    n_rows, n_tok = _sampled_check(cfg, inp, rt, b)
    assert n_tok >= 64 and n_rows >= 2 * int((rt["counts"] > 0).sum())
    if name == "C4z":
        assert (rt["counts"] == 0).sum() >= 4
    ctx.close()


def test_full_size_c5_pair_against_the_oracle_and_the_serial_chunks():
    """BASELINE.json configs[4] (reading c-20): microbatch A (seed 4) forward co-scheduled with microbatch B (seed 5, own
    weights) backward at full size.  The pair's outputs equal the serial chunks bit for bit on disjoint green-context
    partitions (132:16, list order) and on shared SMs (148:32, profile order), and match the oracle on the deliberate
    sample of _sampled_check: Y(A), dX(B), dgates(B), dz_sel(B), dW(B) columns, O / dXp rows at chunk edges."""
    cfg_a = dataclasses.replace(configs.C5A, row_align=128)
    cfg_b = dataclasses.replace(configs.C5B, row_align=128)
    inp_a, inp_b = configs.make_inputs(cfg_a), configs.make_inputs(cfg_b)
    oracle.set_threads(os.cpu_count() or 1)
    rt_a, rt_b = oracle.routing(cfg_a, inp_a), oracle.routing(cfg_b, inp_b)
    ctx = piper.Context(util.desc_of(cfg_a))
    ba, bb = piper.alloc_buffers(ctx, backward=False), piper.alloc_buffers(ctx)
    ba.update(util.upload_inputs(inp_a)), bb.update(util.upload_inputs(inp_b))
    args_a, args_b = piper.chunk_args(ba), piper.chunk_args(bb)
    fwd_names = ("topk_idx", "gates", "counts", "row_of", "src_of", "y")
    bwd_names = ("dgates", "dz_sel", "dx", "dw_gate", "dw_up", "dw_down", "dws_gate", "dws_up", "dws_down")
    # serial chunks: fwd(B) untimed producer, then fwd(A), bwd(B) on one stream with all SMs
    piper.piper_run_chunk_fwd(ctx, args_b)
    piper.piper_run_chunk_fwd(ctx, args_a)
    piper.piper_run_chunk_bwd(ctx, args_b)
    torch.cuda.synchronize()
    serial = {n: ba[n].clone() for n in fwd_names}
    serial.update({n: bb[n].clone() for n in bwd_names})
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    for split, order, part in (((n_sm - 16, 16), piper.ORDER_LIST, piper.PART_EXCLUSIVE),
                               ((n_sm, 32), piper.ORDER_PROFILE, piper.PART_SHARED)):
        for n in fwd_names:
            ba[n].zero_()
        for n in bwd_names:
            bb[n].zero_()
        piper.piper_set_pair_policy(ctx, order, part)
        piper.piper_run_chunk_pair(ctx, args_a, args_b, split[0], split[1])
        torch.cuda.synchronize()
        assert piper.piper_pair_partition_mode(ctx) == (1 if part == piper.PART_EXCLUSIVE else 2)
        for n in fwd_names:
            assert torch.equal(serial[n], ba[n]), (split, "fwd", n)
        for n in bwd_names:
            assert torch.equal(serial[n], bb[n]), (split, "bwd", n)
    # the pair's outputs (last run) against the oracle
    piper.piper_run_task(ctx, "F_PACK", args_a)
    torch.cuda.synchronize()
    _check_full_size_routing(cfg_a, ba, rt_a)
    _check_full_size_routing(cfg_b, bb, rt_b)
    _sampled_check(cfg_a, inp_a, rt_a, ba, fwd=True, bwd=False, n_tokens=32, label="C5a ")
    _sampled_check(cfg_b, inp_b, rt_b, bb, fwd=False, bwd=True, n_tokens=32, label="C5b ")
    ctx.close()
