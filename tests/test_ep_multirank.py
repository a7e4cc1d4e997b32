"""N4 host-side logic on CPU with two gloo ranks: every rank routes its own tokens (oracle), the ranks
all-gather the per-expert split sizes (counts_global, E integers per rank: the one exchange piper_ep_dispatch needs before it
can address the owners' buffers), and every rank derives the layout with piper_ep_plan_host.  The plans must agree: the rows
the ranks send for an expert tile the owner's segment exactly, in rank order, and the owner's counts / offsets are those of
the single-device permutation over the concatenated tokens."""
import dataclasses
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _cfg(world, tr):
    from inputs import configs
    return configs.MoeConfig("ep", T=world * tr, d=64, E=16, k=4, I=64, seed=43, bias="zipf1.2", row_align=16,
                             dtype=configs.DT_F32)


def _worker(rank, world, port, out):
    import paper_2606_11169_b200 as piper
    from inputs import configs
    from oracle import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    tr = 96
    cfg = _cfg(world, tr)
    inp = configs.make_inputs(cfg, weights=False, with_dy=False)
    mine = dataclasses.replace(cfg, T=tr)
    idx, _, cg = oracle.route_topk(mine, inp["logits"][rank * tr:(rank + 1) * tr])   # this rank's tokens only
    gathered = [torch.empty(cfg.E, dtype=torch.int32) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(cg.copy()))
    all_counts = torch.stack(gathered).numpy()
    counts, offsets, send_base = piper.piper_ep_plan_host(all_counts, rank, cfg.row_align)
    out[rank] = (all_counts, cg, counts, offsets, send_base)
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_agree_on_the_expert_parallel_layout():
    from inputs import configs
    from oracle import oracle
    world, tr = 2, 96
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    cfg = _cfg(world, tr)
    inp = configs.make_inputs(cfg, weights=False, with_dy=False)
    el = cfg.E // world
    assert np.array_equal(res[0][0], res[1][0]), "every rank must hold the same all_counts after the all-gather"
    for o in range(world):
        own = dataclasses.replace(cfg, e_lo=o * el, E_loc=el)
        rt = oracle.routing(own, inp)            # single-device definition over the concatenated tokens
        _, _, counts, offsets, _ = res[o]
        assert np.array_equal(counts, rt["counts"]) and np.array_equal(offsets, rt["offsets"])
        for i in range(el):                      # the ranks' rows of expert e tile the owner's segment in rank order
            e, at = o * el + i, int(offsets[i])
            for r in range(world):
                assert int(res[r][4][e]) == at, (o, e, r)
                at += int(res[r][1][e])
            assert at == int(offsets[i]) + int(counts[i])
