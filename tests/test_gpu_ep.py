"""N4: expert parallelism with the pack / combine row movers fused with their
all-to-all over peer memory.  One B200 is all there is, so the n_ranks ranks live on one GPU: every rank has its own
context, tokens and buffers, the "peer" pointers are the other ranks' buffers, and no kernel waits on another rank's kernel
(the steps are ordered on one stream, as a collective would order them).  The oracle is the single-device definition on the
concatenated tokens: owner o's receive buffer must be, bit for bit, what piper_dispatch_pack builds for the local slice
[o * E_loc, (o + 1) * E_loc) of the T * n_ranks tokens, and Y / dX are the sums of the owners' partial results."""
import dataclasses

import numpy as np
import pytest
import torch

import paper_2606_11169_b200 as piper
from inputs import configs
from oracle import oracle
import piper_testutil as util

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_ranks,dtype,align", [(2, configs.DT_BF16, 16), (4, configs.DT_BF16, 128), (2, configs.DT_F32, 1)])
def test_expert_parallel_dispatch_and_combine_over_peer_pointers(n_ranks, dtype, align):
    R, Tr = n_ranks, 192
    E, k = 16, 4
    El = E // R
    base = configs.MoeConfig("ep", T=R * Tr, d=256, E=E, k=k, I=192, seed=41, bias="zipf1.2", gate_mode=1, dtype=dtype,
                             row_align=align)
    own = [dataclasses.replace(base, e_lo=o * El, E_loc=El) for o in range(R)]
    inps = [configs.make_inputs(c) for c in own]          # same tokens / logits, the owner's slice of the weights
    fo = [oracle.forward(c, i) for c, i in zip(own, inps)]
    go = [oracle.backward(c, i, f) for c, i, f in zip(own, inps, fo)]
    impl = piper.GEMM_AUTO
    tok_ctx = [piper.Context(util.desc_of(dataclasses.replace(own[r], T=Tr), impl)) for r in range(R)]
    exp_ctx = [piper.Context(util.desc_of(own[o], impl)) for o in range(R)]
    A = piper.piper_ep_a_cap(tok_ctx[0].desc, R)
    assert A == own[0].a_cap
    dt = tok_ctx[0].torch_dtype
    dev = "cuda"
    x_tot, dy_tot = util.to_dev(inps[0]["x"]), util.to_dev(inps[0]["dy"])
    logits_tot = util.to_dev(inps[0]["logits"])
    i32, f32 = torch.int32, torch.float32

    def e(shape, t):
        return torch.empty(shape, dtype=t, device=dev)

    # per-rank token-side state
    tk = [dict(x=x_tot[r * Tr:(r + 1) * Tr].contiguous(), dy=dy_tot[r * Tr:(r + 1) * Tr].contiguous(),
               logits=logits_tot[r * Tr:(r + 1) * Tr].contiguous(), topk_idx=e((Tr, k), i32), gates=e((Tr, k), f32),
               cg=e((E,), i32), counts=e((El,), i32), offsets=e((El + 4,), i32), send_base=e((E,), i32),
               dest_row=e((Tr, k), i32), y=e((Tr, base.d), dt), dx=e((Tr, base.d), dt), dgates=e((Tr, k), f32)) for r in range(R)]
    # per-owner expert-side buffers
    ow = [dict(xp=e((A, base.d), dt), src_of=e((A,), i32), gate_rows=e((A,), f32), g=e((A, base.I), dt), u=e((A, base.I), dt),
               h=e((A, base.I), dt), o=e((A, base.d), dt), d_o=e((A, base.d), dt), dg=e((A, base.I), dt), du=e((A, base.I), dt),
               dxp=e((A, base.d), dt), dw_gate=e((El, base.d, base.I), dt), dw_up=e((El, base.d, base.I), dt),
               dw_down=e((El, base.I, base.d), dt), w_gate=util.to_dev(inps[o]["w_gate"]), w_up=util.to_dev(inps[o]["w_up"]),
               w_down=util.to_dev(inps[o]["w_down"])) for o in range(R)]
    for b in ow:
        for n in ("xp", "o", "d_o", "dxp"):
            b[n].view(torch.int16 if dtype == configs.DT_BF16 else torch.int32).fill_(0x7FC1)  # poison: pads must be written
    tab = {n: piper.ptr_table([b[n] for b in ow]) for n in ("xp", "src_of", "gate_rows", "o", "d_o", "dxp")}

    # forward: route, exchange the split sizes, plan, dispatch into the owners' buffers
    for r in range(R):
        piper.piper_route_topk(tok_ctx[r], tk[r]["logits"], tk[r]["topk_idx"], tk[r]["gates"], tk[r]["cg"])
    all_counts = torch.stack([t["cg"] for t in tk]).contiguous()   # the all-gather of E integers per rank
    for r in range(R):
        piper.piper_ep_plan(tok_ctx[r], all_counts, r, R, tk[r]["counts"], tk[r]["offsets"], tk[r]["send_base"])
        piper.piper_ep_dispatch(tok_ctx[r], tk[r]["x"], tk[r]["topk_idx"], tk[r]["gates"], tk[r]["send_base"], r, R,
                                tab["xp"], tab["src_of"], tab["gate_rows"], tk[r]["dest_row"])
    for o in range(R):
        piper.piper_ep_finish_recv(tok_ctx[o], tk[o]["counts"], tk[o]["offsets"], R, ow[o]["src_of"], ow[o]["gate_rows"],
                                   ow[o]["xp"])
    torch.cuda.synchronize()
    for r in range(R):   # the device plan equals the host restatement
        hc, ho, hs = piper.piper_ep_plan_host(all_counts.cpu().numpy(), r, align)
        assert np.array_equal(util.to_np(tk[r]["counts"]), hc) and np.array_equal(util.to_np(tk[r]["offsets"])[: El + 1], ho)
        assert np.array_equal(util.to_np(tk[r]["send_base"]), hs)
    for o in range(R):   # the receive buffer is the packed buffer of the concatenated tokens, bit for bit
        f = fo[o]
        used = int(f["offsets"][-1])
        assert np.array_equal(util.to_np(tk[o]["counts"]), f["counts"])
        assert np.array_equal(util.to_np(tk[o]["offsets"])[: El + 1], f["offsets"])
        assert np.array_equal(util.to_np(ow[o]["src_of"]), f["src_of"])
        assert np.array_equal(util.to_np(ow[o]["xp"])[:used], f["xp"][:used]), "received rows must be exact copies"
        util.check_close("gate_rows", util.to_np(ow[o]["gate_rows"])[:used], f["gate_rows"][:used], configs.DT_F32)
    # owners: grouped expert FFN on what they received
    for o in range(R):
        b = ow[o]
        piper.piper_expert_ffn_fwd(exp_ctx[o], b["xp"], tk[o]["offsets"], b["w_gate"], b["w_up"], b["w_down"], b["g"], b["u"],
                                   b["h"], b["o"])
    for r in range(R):
        piper.piper_ep_combine(tok_ctx[r], tab["o"], tk[r]["topk_idx"], tk[r]["dest_row"], tk[r]["gates"], None, tk[r]["y"])
    torch.cuda.synchronize()
    y_ref = sum(f["y"] for f in fo)
    y = np.concatenate([util.to_np(t["y"]) for t in tk])
    util.check_close("y", y, y_ref, dtype)

    # backward: gate * dY to the owners + dgates, owners' dgrad / wgrad, dXp gathered back
    for r in range(R):
        piper.piper_ep_dispatch_bwd(tok_ctx[r], tk[r]["dy"], tk[r]["topk_idx"], tk[r]["dest_row"], tk[r]["gates"], tab["o"],
                                    tab["d_o"], tk[r]["dgates"])
    for o in range(R):
        b = ow[o]
        piper.piper_ep_finish_recv(tok_ctx[o], tk[o]["counts"], tk[o]["offsets"], R, b["src_of"], b["gate_rows"], b["d_o"])
        piper.piper_expert_ffn_bwd(exp_ctx[o], b["d_o"], b["xp"], b["g"], b["u"], b["h"], tk[o]["offsets"], b["w_gate"], b["w_up"],
                                   b["w_down"], b["dg"], b["du"], b["dxp"], b["dw_gate"], b["dw_up"], b["dw_down"])
    for r in range(R):
        piper.piper_ep_unpack(tok_ctx[r], tab["dxp"], tk[r]["topk_idx"], tk[r]["dest_row"], None, tk[r]["dx"])
    torch.cuda.synchronize()
    util.check_close("dgates", np.concatenate([util.to_np(t["dgates"]) for t in tk]), sum(g["dgates"] for g in go), dtype)
    util.check_close("dx", np.concatenate([util.to_np(t["dx"]) for t in tk]), sum(g["dx"] for g in go), dtype)
    for o in range(R):
        for n in ("dw_gate", "dw_up", "dw_down"):
            util.check_close(f"{n} of owner {o}", util.to_np(ow[o][n]), go[o][n], dtype)
    for c in tok_ctx + exp_ctx:
        c.close()
