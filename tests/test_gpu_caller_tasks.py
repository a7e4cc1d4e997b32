"""N3 (Fig. 3b, 161, 346): the rest of the overlapped block as caller tasks of the pair.
The "attention" of this test is whatever the caller enqueues (here: a delay kernel and a copy, through torch on the stream the
library hands over); what is checked is the scheduling contract: the producers of x / logits / dY run before every task
that reads them, the consumers of y / dX / dz_sel after every task that writes them, in every order / partition policy,
and the pair's results stay bit-identical to the serial chunks."""
import dataclasses

import pytest
import torch

import paper_2606_11169_b200 as piper
from inputs import configs
import piper_testutil as util

pytestmark = pytest.mark.gpu

_BEFORE = {"X_F_PRE": ["F_ROUTE", "F_PACK", "F_SHARED"], "F_COMBINE": ["X_F_POST"], "X_B_PRE": ["B_CGRAD", "B_SHARED"],
           "B_UNPACK": ["X_B_POST"], "B_ROUTE_BWD": ["X_B_POST"]}


@pytest.mark.parametrize("name", ["C3s", "C4s"])
@pytest.mark.parametrize("split,policy", [((132, 16), "list/exclusive"), ((116, 32), "profile/exclusive"),
                                          ((148, 48), "profile/shared"), ((148, 16), "list/chunks"),
                                          ((148, 32), "profile/shared/bi")])
def test_pair_schedules_caller_tasks_with_its_own(name, split, policy):
    base = configs.BY_NAME[name]
    cfg_a = dataclasses.replace(base, row_align=128, seed=base.seed + 300)
    cfg_b = dataclasses.replace(base, row_align=128, seed=base.seed + 400)
    inp_a, inp_b = configs.make_inputs(cfg_a), configs.make_inputs(cfg_b)
    # serial reference: fwd(A); fwd(B), bwd(B)
    ctx = piper.Context(util.desc_of(cfg_a))
    ra, rb = piper.alloc_buffers(ctx), piper.alloc_buffers(ctx)
    ra.update(util.upload_inputs(inp_a)), rb.update(util.upload_inputs(inp_b))
    piper.piper_run_chunk_fwd(ctx, piper.chunk_args(ra))
    piper.piper_run_chunk_fwd(ctx, piper.chunk_args(rb))
    piper.piper_run_chunk_bwd(ctx, piper.chunk_args(rb))
    torch.cuda.synchronize()

    pa, pb = piper.alloc_buffers(ctx), piper.alloc_buffers(ctx)
    pa.update(util.upload_inputs(inp_a)), pb.update(util.upload_inputs(inp_b))
    piper.piper_run_chunk_fwd(ctx, piper.chunk_args(pb))  # B's saved activations
    src = {"x": pa["x"].clone(), "logits": pa["logits"].clone(), "dy": pb["dy"].clone()}
    pa["x"].fill_(float("nan")), pa["logits"].fill_(float("nan")), pb["dy"].fill_(float("nan"))  # produced by the caller tasks
    big = torch.randn(4096, 4096, device="cuda")
    tmp = torch.empty_like(big)
    out = {"y2": torch.zeros_like(pa["y"]), "dx2": torch.zeros_like(pb["dx"]), "dz2": torch.zeros_like(pb["dz_sel"])}
    calls = []

    def on(stream_ptr, fn):
        with torch.cuda.stream(torch.cuda.ExternalStream(stream_ptr)):
            torch.mm(big, big, out=tmp)  # the producers are slow: a consumer that did not wait would read NaN
            fn()

    def f_pre(stream, sms):
        calls.append(("F_PRE", sms))
        on(stream, lambda: (pa["x"].copy_(src["x"]), pa["logits"].copy_(src["logits"])))

    def f_post(stream, sms):
        calls.append(("F_POST", sms))
        on(stream, lambda: torch.add(pa["y"], pa["y"], out=out["y2"]))

    def b_pre(stream, sms):
        calls.append(("B_PRE", sms))
        on(stream, lambda: pb["dy"].copy_(src["dy"]))

    def b_post(stream, sms):
        calls.append(("B_POST", sms))
        on(stream, lambda: (out["dx2"].copy_(pb["dx"]), out["dz2"].copy_(pb["dz_sel"])))

    parts = policy.split("/")
    order, part, bi = parts[0], parts[1], len(parts) > 2
    piper.piper_set_pair_policy(ctx, piper.ORDER_PROFILE if order == "profile" else piper.ORDER_LIST,
                                {"shared": piper.PART_SHARED, "chunks": piper.PART_CHUNK_STREAMS}.get(part, piper.PART_EXCLUSIVE))
    piper.piper_set_pair_bwd_pass(ctx, piper.PASS_BI if bi else piper.PASS_B)
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_F_PRE, f_pre, est_ms=0.3, side=1)   # "attention forward": GEMM side
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_F_POST, f_post, est_ms=0.05, side=0)
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_B_PRE, b_pre, est_ms=0.05, side=0)
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_B_POST, b_post, est_ms=0.6, side=1)  # "attention backward"
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    sg = min(split[0], n_sm) if part != "exclusive" else min(split[0], n_sm - split[1])
    picked = piper.piper_pair_order(ctx, sg, split[1])
    assert len(picked) == len(set(picked)) and {"X_F_PRE", "X_F_POST", "X_B_PRE", "X_B_POST"} <= set(picked)
    pos = {t: i for i, t in enumerate(picked)}
    for first, later in _BEFORE.items():
        for t in later:
            if t in pos:
                assert pos[first] < pos[t], (first, t, picked)
    piper.piper_run_chunk_pair(ctx, piper.chunk_args(pa), piper.chunk_args(pb), sg, split[1])
    if bi:
        piper.piper_run_chunk_bwd_weight(ctx, piper.chunk_args(pb))
    torch.cuda.synchronize()
    assert sorted(c[0] for c in calls) == ["B_POST", "B_PRE", "F_POST", "F_PRE"]
    if part != "chunks":  # each task is told its side's SM budget
        sides = {"F_PRE": sg, "B_POST": sg, "F_POST": split[1], "B_PRE": split[1]}
        assert all(sms == sides[n] for n, sms in calls), calls
    for n in ("topk_idx", "gates", "counts", "row_of", "src_of", "y"):
        assert torch.equal(ra[n], pa[n]), "fwd " + n
    for n in ("dgates", "dz_sel", "dx", "dw_gate", "dw_up", "dw_down") + (("dws_gate", "dws_up", "dws_down") if base.I_shared else ()):
        assert torch.equal(rb[n], pb[n]), "bwd " + n
    assert torch.equal(out["y2"], ra["y"] + ra["y"]) and torch.equal(out["dx2"], rb["dx"]) and torch.equal(out["dz2"], rb["dz_sel"])

    # a cleared slot leaves the DAG; a failing caller task fails the pair call loudly
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_F_POST, None)
    assert "X_F_POST" not in piper.piper_pair_order(ctx, sg, split[1])

    def broken(stream, sms):
        raise RuntimeError("caller task failed on purpose")

    piper.piper_pair_set_caller_task(ctx, piper.SLOT_B_POST, broken, side=1)
    with pytest.raises(piper.PiperError):
        piper.piper_run_chunk_pair(ctx, piper.chunk_args(pa), piper.chunk_args(pb), sg, split[1])
    torch.cuda.synchronize()
    ctx.close()
