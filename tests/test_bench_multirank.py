"""N > 1 plumbing of bench.py on CPU: two gloo ranks shard the work as independent replicas, take the
max time over ranks and report the whole-job rate; the reference arm runs on rank 0 only."""
import os
import socket
import sys

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


def _worker(rank, world, port, out):
    import bench
    from inputs import configs
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = configs.C2S
    rcfg = bench.rank_config(cfg, rank)
    inp = configs.make_inputs(rcfg, weights=False, with_dy=False)
    my_ms = 10.0 * (rank + 1)  # rank 1 is the slow one
    worst = bench.max_over_ranks(my_ms, world, torch.device("cpu"))
    out[rank] = (rcfg.seed, float(inp["logits"].sum()), worst, bench.whole_job_tokens_per_s(cfg, world, worst))
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_are_independent_replicas_timed_by_the_slowest():
    from inputs import configs
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == configs.C2S.seed and res[1][0] == configs.C2S.seed + 1000
    assert res[0][1] != res[1][1], "ranks must draw different microbatches"
    for r in range(world):
        assert res[r][2] == 20.0  # max over ranks
        assert abs(res[r][3] - world * configs.C2S.T / 20e-3) < 1e-6


def test_reference_arm_runs_on_rank_zero_only(monkeypatch, capsys):
    import bench
    from inputs import configs
    monkeypatch.setenv("RANK", "1")
    args = type("A", (), dict(oracle_tokens=2, steps=1, warmup=0, gpus=2))()
    bench.run_reference(args, configs.C2S)
    assert capsys.readouterr().out == ""
