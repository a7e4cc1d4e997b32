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


# ---- profile-guided schedule search (PIPER_ORDER_PROFILE) --------------------------------
def _simulate(n, edges, stream_of, dur, seq_by_stream):
    """Event-rule simulation written independently of sched.cpp: returns the makespan of the given
    per-stream sequences, or None on deadlock."""
    preds = {v: [s for s, t in edges if t == v] for v in range(n)}
    fin, head, free_at = {}, [0, 0], [0.0, 0.0]
    while any(head[s] < len(seq_by_stream[s]) for s in (0, 1)):
        progressed = False
        for s in (0, 1):
            if head[s] >= len(seq_by_stream[s]):
                continue
            v = seq_by_stream[s][head[s]]
            if all(p in fin for p in preds[v]):
                start = max([free_at[s]] + [fin[p] for p in preds[v]])
                fin[v] = start + dur[v]
                free_at[s] = fin[v]
                head[s] += 1
                progressed = True
        if not progressed:
            return None
    return max(free_at)


def _brute_force_makespan(n, edges, stream_of, dur):
    import itertools
    best = None
    per = [[v for v in range(n) if stream_of[v] == s] for s in (0, 1)]
    for a in itertools.permutations(per[0]):
        for b in itertools.permutations(per[1]):
            m = _simulate(n, edges, stream_of, dur, [list(a), list(b)])
            if m is not None and (best is None or m < best):
                best = m
    return best


def test_schedule_search_is_optimal_on_small_random_dags():
    rng = np.random.default_rng(11)
    for _ in range(25):
        n = int(rng.integers(2, 8))
        edges = [[a, b] for a in range(n) for b in range(a + 1, n) if rng.random() < 0.3]
        stream_of = rng.integers(0, 2, n).tolist()
        dur = rng.integers(1, 9, n).astype(np.float32)
        order, waits, records, mk = piper.piper_schedule_search(n, edges, stream_of, dur)
        pos = {v: i for i, v in enumerate(order.tolist())}
        assert sorted(pos) == list(range(n))
        wait_set = set(map(tuple, waits.tolist()))
        for s, t in edges:
            assert pos[s] < pos[t]
            assert (stream_of[s] == stream_of[t]) != ((s, t) in wait_set)
        assert [i for i in range(n) if records[i]] == sorted({s for s, t in wait_set})
        seqs = [[v for v in order.tolist() if stream_of[v] == s] for s in (0, 1)]
        assert _simulate(n, edges, stream_of, dur.tolist(), seqs) == pytest.approx(mk)
        assert mk == pytest.approx(_brute_force_makespan(n, edges, stream_of, dur.tolist()))


def test_schedule_search_on_the_pair_dag_beats_the_list_order():
    g = json.load(open(os.path.join(ROOT, "tests", "golden", "pair_dag.json")))
    n, edges, stream_of = len(g["nodes"]), g["edges"], g["stream_of"]
    # durations of the C3-shaped pair (ms): GEMM tasks on 132 SMs, movers on 16
    dur = np.array([.03, .03, .15, .58, .32, .56, .3, .3, .37, .58, 1.0, 1.2, .3, .02], np.float32)
    order, waits, records, mk = piper.piper_schedule_search(n, edges, stream_of, dur)
    seq_list = [g["q_comm"], g["q_gemm"]]
    m_list = _simulate(n, edges, stream_of, dur.tolist(), seq_list)
    assert mk <= m_list + 1e-6
    # lower bound: the GEMM stream's total work; the search must come within the last comm task of it
    gemm = float(sum(dur[v] for v in range(n) if stream_of[v] == 1))
    assert gemm <= mk <= gemm + 0.35
    again = piper.piper_schedule_search(n, edges, stream_of, dur)
    assert again[0].tolist() == order.tolist()  # deterministic
    with pytest.raises(piper.PiperError):
        piper.piper_schedule_search(3, [[0, 1], [1, 2], [2, 0]], [0, 1, 0], [1, 1, 1])


def test_schedule_search_with_the_four_caller_tasks_of_the_overlapped_block():
    """N3 (Fig. 3b): the pair DAG with attention forward / backward as caller tasks on the GEMM stream and the
    two residual slots on the pack/combine stream (piper_pair_set_caller_task): 18 tasks must still be searched in a time
    a first call can afford, every edge respected, and the makespan no worse than the list order's."""
    import time
    g = json.load(open(os.path.join(ROOT, "tests", "golden", "pair_dag.json")))
    n0, edges, stream_of = len(g["nodes"]), [list(e) for e in g["edges"]], list(g["stream_of"])
    idx = {name: i for i, name in enumerate(g["nodes"])}
    pre_f, post_f, pre_b, post_b = n0, n0 + 1, n0 + 2, n0 + 3
    edges += [[pre_f, idx["F.route"]], [pre_f, idx["F.pack"]], [pre_f, idx["F.shared"]], [idx["F.combine"], post_f],
              [pre_b, idx["B.cgrad"]], [pre_b, idx["B.shared_bwd"]], [idx["B.unpack"], post_b], [idx["B.route_bwd"], post_b]]
    stream_of += [1, 0, 0, 1]
    dur = np.array([.03, .03, .15, .58, .32, .56, .3, .3, .37, .58, 1.0, 1.2, .3, .02, .9, .05, .05, 1.8], np.float32)
    t0 = time.time()
    order, waits, records, mk = piper.piper_schedule_search(n0 + 4, edges, stream_of, dur)
    assert time.time() - t0 < 1.0  # branch and bound: about a millisecond (the product of all per-stream sequences took seconds)
    pos = {v: i for i, v in enumerate(order.tolist())}
    wait_set = set(map(tuple, waits.tolist()))
    for s, t in edges:
        assert pos[s] < pos[t]
        assert (stream_of[s] == stream_of[t]) != ((s, t) in wait_set)
    prio = list(g["prio"]) + [0, 0, 1, 1]
    lo, _, _ = piper.piper_list_schedule(n0 + 4, edges, stream_of, prio)
    seq_list = [[v for v in lo.tolist() if stream_of[v] == s] for s in (0, 1)]
    assert mk <= _simulate(n0 + 4, edges, stream_of, dur.tolist(), seq_list) + 1e-6


def test_schedule_search_stays_bounded_on_sparse_18_task_dags():
    """Almost independent tasks are the hard case for an exact search (every order of a stream's tasks is a schedule):
    the dominance rule folds them and a node budget caps the rest.  The result must be a valid schedule, no worse than
    the list order, found within a second."""
    import time
    rng = np.random.default_rng(3)
    for _ in range(40):
        n = 18
        p = float(rng.choice([0.03, 0.05, 0.1, 0.2]))
        edges = [[a, b] for a in range(n) for b in range(a + 1, n) if rng.random() < p]
        stream_of = rng.integers(0, 2, n).tolist()
        dur = (rng.random(n) * float(rng.choice([1, 10])) + 0.01).astype(np.float32)
        t0 = time.time()
        order, waits, records, mk = piper.piper_schedule_search(n, edges, stream_of, dur)
        assert time.time() - t0 < 3.0
        pos = {v: i for i, v in enumerate(order.tolist())}
        assert sorted(pos) == list(range(n))
        assert all(pos[s] < pos[t] for s, t in edges)
        seqs = [[v for v in order.tolist() if stream_of[v] == s] for s in (0, 1)]
        assert _simulate(n, edges, stream_of, dur.tolist(), seqs) == pytest.approx(mk, rel=1e-5)
        lo, _, _ = piper.piper_list_schedule(n, edges, stream_of, [0] * n)
        seq_list = [[v for v in lo.tolist() if stream_of[v] == s] for s in (0, 1)]
        assert mk <= _simulate(n, edges, stream_of, dur.tolist(), seq_list) + 1e-4


def test_schedule_search_with_dominance_is_optimal_on_sparse_dags():
    """The dominance rule of the search (a state is cut when one seen before with the same scheduled set is no later in
    every respect) must not lose the optimum: sparse DAGs of 8-9 tasks, where most of the pruning comes from it, against
    brute force over all pairs of per-stream orders."""
    rng = np.random.default_rng(23)
    for _ in range(12):
        n = int(rng.integers(8, 10))
        edges = [[a, b] for a in range(n) for b in range(a + 1, n) if rng.random() < 0.12]
        stream_of = [int(v % 2) for v in rng.permutation(n)]  # 4-5 tasks per stream: at most 5! x 4! orders
        dur = rng.integers(1, 9, n).astype(np.float32)
        order, waits, records, mk = piper.piper_schedule_search(n, edges, stream_of, dur)
        seqs = [[v for v in order.tolist() if stream_of[v] == s] for s in (0, 1)]
        assert _simulate(n, edges, stream_of, dur.tolist(), seqs) == pytest.approx(mk)
        assert mk == pytest.approx(_brute_force_makespan(n, edges, stream_of, dur.tolist()))
