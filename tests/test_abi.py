"""CPU checks of the boundary: the library builds for sm_100a, loads, and exports every symbol that
include/piper.h declares; host-side argument validation; the host list scheduler against the golden
order of the pair DAG (SURVEY.md §8c c-sched).  No compute calls here."""
import ctypes
import json
import os
import re

import numpy as np
import pytest

import paper_2606_11169_b200 as piper

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "piper.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(piper_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = piper.lib()
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"libpiper.so does not export {n}"


def test_desc_validation_on_host():
    L = piper.lib()
    nbytes = ctypes.c_size_t(0)
    good = piper.make_desc(128, 64, 4, 2, 128, dtype=piper.DT_F32)
    assert L.piper_workspace_bytes(ctypes.byref(good), ctypes.byref(nbytes)) == 0 and nbytes.value > 0
    assert L.piper_a_cap(ctypes.byref(good)) == 128 * 2
    for bad in (piper.make_desc(128, 64, 4, 5, 128), piper.make_desc(128, 60, 4, 2, 128),
                piper.make_desc(128, 64, 4, 2, 100), piper.make_desc(128, 64, 4, 2, 128, e_lo=2, E_loc=3),
                piper.make_desc(128, 64, 600, 2, 128), piper.make_desc(128, 64, 4, 2, 128, row_align=0)):
        assert L.piper_workspace_bytes(ctypes.byref(bad), ctypes.byref(nbytes)) == -1
    al = piper.make_desc(100, 64, 8, 2, 128, e_lo=2, E_loc=4, row_align=16)
    assert L.piper_a_cap(ctypes.byref(al)) == 100 * 2 + 4 * 15


def test_context_needs_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(piper.PiperError):
        piper.Context(piper.make_desc(128, 64, 4, 2, 128, dtype=piper.DT_F32))


def test_list_scheduler_matches_golden_pair_dag():
    g = json.load(open(os.path.join(ROOT, "tests", "golden", "pair_dag.json")))
    order, waits, records = piper.piper_list_schedule(len(g["nodes"]), g["edges"], g["stream_of"], g["prio"])
    assert order.tolist() == g["order"]
    assert sorted(map(tuple, waits.tolist())) == sorted(map(tuple, g["waits"]))
    assert [i for i, r in enumerate(records) if r] == g["records"]
    # every edge is same-queue-earlier or has a wait; no other sync
    pos = {v: i for i, v in enumerate(order.tolist())}
    wait_set = set(map(tuple, waits.tolist()))
    for s, t in g["edges"]:
        assert pos[s] < pos[t]
        assert (g["stream_of"][s] == g["stream_of"][t]) != ((s, t) in wait_set)


def test_list_scheduler_rejects_cycles_and_bad_edges():
    with pytest.raises(piper.PiperError):
        piper.piper_list_schedule(3, [[0, 1], [1, 2], [2, 0]], [0, 0, 0], [0, 0, 0])
    with pytest.raises(piper.PiperError):
        piper.piper_list_schedule(2, [[0, 5]], [0, 0], [0, 0])


def test_list_scheduler_random_dags_agree_with_the_oracle():
    from oracle import oracle
    rng = np.random.default_rng(7)
    for _ in range(50):
        n = int(rng.integers(2, 24))
        edges = [[a, b] for a in range(n) for b in range(a + 1, n) if rng.random() < 0.2]
        stream_of = rng.integers(0, 3, n)
        prio = rng.integers(0, 2, n)
        o1, w1, r1 = piper.piper_list_schedule(n, edges, stream_of, prio)
        o2, _, w2, r2 = oracle.list_schedule(n, np.array(edges, np.int32).reshape(-1, 2), stream_of, prio)
        assert o1.tolist() == o2.tolist() and w1.tolist() == w2.tolist() and r1.tolist() == r2.tolist()
