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


def _run_steps(cfg, inp, gemm_impl=piper.GEMM_AUTO, use_chunk_calls=False, backward=True, overlap=False):
    """Runs the whole path; returns (ctx, dict of device tensors)."""
    ctx = piper.Context(util.desc_of(cfg, gemm_impl))
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
@pytest.mark.parametrize("align", [1, 128])  # 128: the tcgen05 kernels; 1: dense packing, FP32-ALU GEMMs
def test_small_configs_full_tensor_parity(name, impl, align):
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=align)
    if cfg.dtype == configs.DT_F32 and impl == piper.GEMM_SIMT:
        pytest.skip("fp32 already runs the FP32-ALU kernels under GEMM_AUTO")
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp, gemm_impl=impl)
    _check_all(cfg, b, f, g)
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
                             n_dead=int(rng.integers(0, 2)) if E > k + 1 else 0, row_align=128)


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
@pytest.mark.parametrize("env", [{"PIPER_TC_ROWS_ON_N": "0"}, {"PIPER_TC_ROWS_ON_N": "0", "PIPER_TC_2CTA": "0"}])
def test_fallback_kernel_families(name, env, monkeypatch):
    """The rows-on-M CTA-pair kernels and the 1-CTA kernels (DESIGN.md section 5.1 b, c) stay correct: they serve
    layers with more than 192 local experts.  The switches are read when a context is created."""
    for k_, v_ in env.items():
        monkeypatch.setenv(k_, v_)
    cfg = dataclasses.replace(configs.BY_NAME[name], row_align=128)
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp, use_chunk_calls=True)
    _check_all(cfg, b, f, g)
    assert piper.piper_gemm_path(ctx) == 1
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


@pytest.mark.parametrize("name", ["C3s", "C4s", "C1s"])
@pytest.mark.parametrize("split,policy", [((132, 16), "list/exclusive"), ((100, 48), "list/exclusive"),
                                          ((116, 32), "profile/exclusive"), ((148, 16), "list/shared"),
                                          ((148, 48), "profile/shared"), ((148, 16), "list/chunks")])
def test_pair_is_bitwise_equal_to_serial(name, split, policy):
    """the overlapped, out-of-order plan must respect every dependency -> identical results,
    for the paper's list order and the profile-guided one, on disjoint and on shared SM partitions."""
    base = configs.BY_NAME[name]
    cfg_a = dataclasses.replace(base, row_align=128, seed=base.seed + 100)
    cfg_b = dataclasses.replace(base, row_align=128, seed=base.seed + 200)
    inp_a, inp_b = configs.make_inputs(cfg_a), configs.make_inputs(cfg_b)
    # serial: fwd(A) ; fwd(B) (untimed producer of B's saved activations) ; bwd(B)
    ctx, ba = _run_steps(cfg_a, inp_a, use_chunk_calls=True, backward=False)
    _, bb = _run_steps(cfg_b, inp_b, use_chunk_calls=True, backward=True)
    # pair on fresh buffers: B's forward first, then [F(A), B(B)] co-scheduled
    pa, pb = piper.alloc_buffers(ctx), piper.alloc_buffers(ctx)
    pa.update(util.upload_inputs(inp_a)), pb.update(util.upload_inputs(inp_b))
    args_a, args_b = piper.chunk_args(pa), piper.chunk_args(pb)
    piper.piper_run_chunk_fwd(ctx, args_b)
    order, part = policy.split("/")
    piper.piper_set_pair_policy(ctx, piper.ORDER_PROFILE if order == "profile" else piper.ORDER_LIST,
                                {"shared": piper.PART_SHARED, "chunks": piper.PART_CHUNK_STREAMS}.get(part, piper.PART_EXCLUSIVE))
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    sg = min(split[0], n_sm) if part != "exclusive" else min(split[0], n_sm - split[1])
    picked = piper.piper_pair_order(ctx, sg, split[1])
    assert sorted(picked) == sorted(t for t in piper.TASKS if base.I_shared or t not in ("F_SHARED", "B_SHARED"))
    piper.piper_run_chunk_pair(ctx, args_a, args_b, sg, split[1])
    torch.cuda.synchronize()
    mode = piper.piper_pair_partition_mode(ctx)
    assert mode == {"shared": 2, "chunks": 3}.get(part, mode) and mode in (1, 2, 3)
    if part == "exclusive":  # sm_gemm + sm_comm beyond the device is refused on disjoint partitions
        with pytest.raises(piper.PiperError):
            piper.piper_run_chunk_pair(ctx, args_a, args_b, n_sm, 16)
    for n in ("topk_idx", "gates", "counts", "row_of", "src_of", "y"):
        assert torch.equal(ba[n], pa[n]), "fwd " + n
    nofs = base.e_loc + 1  # the offsets buffers are over-allocated; entries past E_loc+1 are never written
    assert torch.equal(ba["offsets"][:nofs], pa["offsets"][:nofs]), "fwd offsets"
    for n in ("dgates", "dz_sel", "dx", "dw_gate", "dw_up", "dw_down"):
        assert torch.equal(bb[n], pb[n]), "bwd " + n
    ctx.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C4z"])
def test_full_size_routing_and_permutation_bit_exact(name):
    cfg = configs.BY_NAME[name]
    inp = configs.make_inputs(cfg, weights=False, with_dy=False)
    ref = oracle.routing(cfg, inp)
    ctx = piper.Context(util.desc_of(cfg))
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
    cfg = configs.MoeConfig("edge2", T=40, d=64, E=8, k=1, I=64, seed=22, e_lo=6, E_loc=2, n_dead=2, bias="zipf1.2")
    inp = configs.make_inputs(cfg)
    f = oracle.forward(cfg, inp)
    assert int(f["offsets"][-1]) == 0  # nothing is routed to the dead local experts
    g = oracle.backward(cfg, inp, f)
    ctx, b = _run_steps(cfg, inp)
    _check_all(cfg, b, f, g)
    assert not util.to_np(b["y"]).any() and not util.to_np(b["dx"]).any()
    ctx.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4z"])
def test_full_size_sampled_parity_in_bench_configuration(name):
    """BASELINE.json full sizes in the launch configuration bench.py times (row_align 128, whole-chunk calls,
    tcgen05 GEMMs): routing / permutation bit-exact on the whole tensors; Y, dX, dgates on sampled tokens and
    dW on sampled columns of sampled experts, each computed by the oracle one by one from the definition."""
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
    torch.cuda.synchronize()
    for n in ("topk_idx", "counts_global", "counts", "row_of", "src_of"):
        assert np.array_equal(util.to_np(b[n]).reshape(-1), rt[n].reshape(-1)), n
    assert np.array_equal(util.to_np(b["offsets"])[: cfg.e_loc + 1], rt["offsets"])
    rng = np.random.default_rng(cfg.seed)
    local_tokens = np.nonzero((rt["row_of"] >= 0).any(axis=1))[0]
    tokens = np.sort(np.concatenate([rng.choice(local_tokens, 5, replace=False), [0, cfg.T - 1]]))
    s = oracle.sample_tokens(cfg, inp, rt, tokens)
    tk = torch.from_numpy(tokens).cuda()
    rows = torch.from_numpy(s["rows"]).cuda()
    dt = cfg.dtype
    util.check_close("o rows", util.to_np(b["o"][rows]), s["o_rows"], dt)
    util.check_close("y", util.to_np(b["y"][tk]), s["y"], dt)
    util.check_close("dgates", util.to_np(b["dgates"][tk]), s["dgates"], dt)
    util.check_close("dxp rows", util.to_np(b["dxp"][rows]), s["dxp_rows"], dt)
    util.check_close("dx", util.to_np(b["dx"][tk]), s["dx"], dt)
    # wgrad: the fullest expert, a small one and (C4z) an empty one
    order = np.argsort(rt["counts"])
    picks = {int(order[-1]), int(order[len(order) // 4])}
    J = np.sort(rng.choice(cfg.I, 3, replace=False)).astype(np.int64)
    Jc = torch.from_numpy(J).cuda()
    for e in sorted(picks):
        rg, ru, rd = oracle.sample_wgrad(cfg, inp, rt, e, J)
        util.check_close(f"dw_gate[{e}][:,J]", util.to_np(b["dw_gate"][e][:, Jc]), rg, dt)
        util.check_close(f"dw_up[{e}][:,J]", util.to_np(b["dw_up"][e][:, Jc]), ru, dt)
        util.check_close(f"dw_down[{e}][J,:]", util.to_np(b["dw_down"][e][Jc, :]), rd, dt)
    for e in np.nonzero(rt["counts"] == 0)[0][:2]:
        for n in ("dw_gate", "dw_up", "dw_down"):
            assert not bool(b[n][int(e)].any()), f"{n}[{e}] must be exactly zero for an empty expert"
    if name == "C4z":
        assert (rt["counts"] == 0).sum() >= 4
    if cfg.I_shared:
        Js = np.sort(rng.choice(cfg.I_shared, 2, replace=False)).astype(np.int64)
        Jsc = torch.from_numpy(Js).cuda()
        rg, ru, rd = oracle.sample_wgrad_shared(cfg, inp, Js)
        util.check_close("dws_gate[:,J]", util.to_np(b["dws_gate"][:, Jsc]), rg, dt)
        util.check_close("dws_up[:,J]", util.to_np(b["dws_up"][:, Jsc]), ru, dt)
        util.check_close("dws_down[J,:]", util.to_np(b["dws_down"][Jsc, :]), rd, dt)
    ctx.close()
