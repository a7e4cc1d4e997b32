"""Thin ctypes binding over libpiper.so (include/piper.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; PyTorch is used for device memory and
streams.  There is no CPU fallback: loading fails loudly when the library is missing, and every
entry point raises on a non-zero status.  Function names equal the C-ABI names.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import build as _build

_i32, _vp = ctypes.c_int32, ctypes.c_void_p

PIPER_OK = 0
DT_F32, DT_BF16 = 0, 1
GEMM_AUTO, GEMM_SIMT = 0, 1


class PiperError(RuntimeError):
    pass


class MoeDesc(ctypes.Structure):
    """piper_moe_desc"""
    _fields_ = [(n, _i32) for n in ("T", "d", "E", "k", "e_lo", "E_loc", "I", "I_shared", "dtype", "gate_mode",
                                    "row_align", "dw_dtype", "gemm_impl")]


_CHUNK_FIELDS = ("logits", "x", "dy", "w_gate", "w_up", "w_down", "ws_gate", "ws_up", "ws_down",
                 "topk_idx", "counts_global", "counts", "offsets", "row_of", "src_of",
                 "gates", "gate_rows", "dgates", "dz_sel",
                 "xp", "g_save", "u_save", "h_save", "o",
                 "gs_save", "us_save", "hs_save", "s", "y",
                 "d_o", "dg", "du", "dxp", "dgs", "dus", "dxs", "dx",
                 "dw_gate", "dw_up", "dw_down", "dws_gate", "dws_up", "dws_down",
                 "w_r", "router_bias", "dw_r", "dx_router", "dz_scratch")


class ChunkArgs(ctypes.Structure):
    """piper_chunk_args (field order of include/piper.h)"""
    _fields_ = [(n, _vp) for n in _CHUNK_FIELDS]


_lib = None


def lib() -> ctypes.CDLL:
    """Loads libpiper.so (building it in-tree if the sources are newer).  Raises if that fails."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise PiperError(f"CUDA library missing: {path}")
        L = ctypes.CDLL(path)
        L.piper_a_cap.restype = ctypes.c_int64
        L.piper_ep_a_cap.restype = ctypes.c_int64
        L.piper_kernel_launches.restype = ctypes.c_int64
        L.piper_last_cuda_error.restype = ctypes.c_char_p
        L.piper_debug_tc_counters.restype = ctypes.c_void_p
        _lib = L
    return _lib


def _ptr(t):
    if t is None:
        return _vp(0)
    if not t.is_cuda or not t.is_contiguous():
        raise PiperError("tensor arguments must be contiguous CUDA tensors")
    return _vp(t.data_ptr())


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return _vp(s.cuda_stream)


def make_desc(T, d, E, k, I, e_lo=0, E_loc=-1, I_shared=0, dtype=DT_BF16, gate_mode=0, row_align=1,
              gemm_impl=GEMM_AUTO, dw_dtype=None) -> MoeDesc:
    """dw_dtype: element type of the dW outputs (default = dtype; DT_F32 on a bf16 layer = main-grad style fp32 dW)."""
    return MoeDesc(T, d, E, k, e_lo, E if E_loc < 0 else E_loc, I, I_shared, dtype, gate_mode, row_align,
                   dtype if dw_dtype is None else dw_dtype, gemm_impl)


class Context:
    """piper_ctx + the workspace tensor it lives on."""

    def __init__(self, desc: MoeDesc, device: int = 0):
        L = lib()
        if not torch.cuda.is_available():
            raise PiperError("no CUDA device: the piper library has no CPU path")
        self.desc = desc
        self.device = torch.device("cuda", device)
        nbytes = ctypes.c_size_t(0)
        rc = L.piper_workspace_bytes(ctypes.byref(desc), ctypes.byref(nbytes))
        if rc != PIPER_OK:
            raise PiperError(f"piper_workspace_bytes: status {rc} (invalid layer description)")
        self.workspace = torch.zeros(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) & ~255
        self._h = _vp(0)
        rc = L.piper_create(ctypes.byref(desc), device, _vp(base), ctypes.c_size_t(nbytes.value), ctypes.byref(self._h))
        if rc != PIPER_OK:
            raise PiperError(f"piper_create: status {rc}")

    def close(self):
        if self._h:
            lib().piper_destroy(self._h)
            self._h = _vp(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def a_cap(self) -> int:
        return int(lib().piper_a_cap(ctypes.byref(self.desc)))

    @property
    def torch_dtype(self):
        return torch.bfloat16 if self.desc.dtype == DT_BF16 else torch.float32

    def check(self, rc: int, what: str):
        if rc != PIPER_OK:
            msg = lib().piper_last_cuda_error(self._h).decode() if rc in (-4, -2) else ""
            raise PiperError(f"{what}: status {rc} {msg}")


def piper_kernel_launches(ctx: Context) -> int:
    return int(lib().piper_kernel_launches(ctx._h))


def piper_set_chunk_overlap(ctx: Context, on: int):
    ctx.check(lib().piper_set_chunk_overlap(ctx._h, int(on)), "piper_set_chunk_overlap")


def piper_set_wgrad_accumulate(ctx: Context, accumulate: int):
    ctx.check(lib().piper_set_wgrad_accumulate(ctx._h, int(accumulate)), "piper_set_wgrad_accumulate")


def piper_pair_partition_mode(ctx: Context) -> int:
    return int(lib().piper_pair_partition_mode(ctx._h))


def piper_route_topk(ctx, logits, topk_idx, gates, counts_global, stream=None):
    ctx.check(lib().piper_route_topk(ctx._h, _ptr(logits), _ptr(topk_idx), _ptr(gates), _ptr(counts_global),
                                     _stream(stream)), "piper_route_topk")


def piper_dispatch_pack(ctx, x, topk_idx, gates, counts, offsets, row_of, src_of, gate_rows, xp, stream=None):
    ctx.check(lib().piper_dispatch_pack(ctx._h, _ptr(x), _ptr(topk_idx), _ptr(gates), _ptr(counts), _ptr(offsets),
                                        _ptr(row_of), _ptr(src_of), _ptr(gate_rows), _ptr(xp), _stream(stream)),
              "piper_dispatch_pack")


def piper_expert_ffn_fwd(ctx, xp, offsets, w_gate, w_up, w_down, g_save, u_save, h_save, o, stream=None):
    ctx.check(lib().piper_expert_ffn_fwd(ctx._h, _ptr(xp), _ptr(offsets), _ptr(w_gate), _ptr(w_up), _ptr(w_down),
                                         _ptr(g_save), _ptr(u_save), _ptr(h_save), _ptr(o), _stream(stream)),
              "piper_expert_ffn_fwd")


def piper_shared_ffn_fwd(ctx, x, ws_gate, ws_up, ws_down, g_save, u_save, h_save, s, stream=None):
    ctx.check(lib().piper_shared_ffn_fwd(ctx._h, _ptr(x), _ptr(ws_gate), _ptr(ws_up), _ptr(ws_down), _ptr(g_save),
                                         _ptr(u_save), _ptr(h_save), _ptr(s), _stream(stream)), "piper_shared_ffn_fwd")


def piper_combine(ctx, o, row_of, gates, s, y, stream=None):
    ctx.check(lib().piper_combine(ctx._h, _ptr(o), _ptr(row_of), _ptr(gates), _ptr(s), _ptr(y), _stream(stream)),
              "piper_combine")


def piper_combine_bwd(ctx, dy, o, src_of, row_of, gates, offsets, d_o, dgates, stream=None):
    ctx.check(lib().piper_combine_bwd(ctx._h, _ptr(dy), _ptr(o), _ptr(src_of), _ptr(row_of), _ptr(gates),
                                      _ptr(offsets), _ptr(d_o), _ptr(dgates), _stream(stream)), "piper_combine_bwd")


def piper_expert_ffn_bwd(ctx, d_o, xp, g_save, u_save, h_save, offsets, w_gate, w_up, w_down, dg, du, dxp, dw_gate,
                         dw_up, dw_down, accumulate=0, stream=None):
    ctx.check(lib().piper_expert_ffn_bwd(ctx._h, _ptr(d_o), _ptr(xp), _ptr(g_save), _ptr(u_save), _ptr(h_save),
                                         _ptr(offsets), _ptr(w_gate), _ptr(w_up), _ptr(w_down), _ptr(dg), _ptr(du),
                                         _ptr(dxp), _ptr(dw_gate), _ptr(dw_up), _ptr(dw_down), int(accumulate),
                                         _stream(stream)), "piper_expert_ffn_bwd")


def piper_shared_ffn_bwd(ctx, dy, x, g_save, u_save, h_save, ws_gate, ws_up, ws_down, dgs, dus, dxs, dws_gate, dws_up,
                         dws_down, accumulate=0, stream=None):
    ctx.check(lib().piper_shared_ffn_bwd(ctx._h, _ptr(dy), _ptr(x), _ptr(g_save), _ptr(u_save), _ptr(h_save),
                                         _ptr(ws_gate), _ptr(ws_up), _ptr(ws_down), _ptr(dgs), _ptr(dus), _ptr(dxs),
                                         _ptr(dws_gate), _ptr(dws_up), _ptr(dws_down), int(accumulate),
                                         _stream(stream)), "piper_shared_ffn_bwd")


def piper_dispatch_unpack(ctx, dxp, row_of, dx_shared, dx, stream=None):
    ctx.check(lib().piper_dispatch_unpack(ctx._h, _ptr(dxp), _ptr(row_of), _ptr(dx_shared), _ptr(dx), _stream(stream)),
              "piper_dispatch_unpack")


def piper_router_fwd(ctx, x, w_r, bias, logits, stream=None):
    ctx.check(lib().piper_router_fwd(ctx._h, _ptr(x), _ptr(w_r), _ptr(bias), _ptr(logits), _stream(stream)),
              "piper_router_fwd")


def piper_router_bwd(ctx, x, w_r, topk_idx, dz_sel, dz_scratch, dw_r, dx_router, stream=None):
    ctx.check(lib().piper_router_bwd(ctx._h, _ptr(x), _ptr(w_r), _ptr(topk_idx), _ptr(dz_sel), _ptr(dz_scratch),
                                     _ptr(dw_r), _ptr(dx_router), _stream(stream)), "piper_router_bwd")


def piper_dispatch_unpack_router(ctx, dxp, row_of, dx_shared, dx_router, dx, stream=None):
    ctx.check(lib().piper_dispatch_unpack_router(ctx._h, _ptr(dxp), _ptr(row_of), _ptr(dx_shared), _ptr(dx_router),
                                                 _ptr(dx), _stream(stream)), "piper_dispatch_unpack_router")


# ---- N4: expert parallelism over peer memory (include/piper.h) ------------------------------------------------------
def ptr_table(tensors, device=None):
    """Device array of the tensors' data pointers (the peer_* arguments)."""
    dev = tensors[0].device if device is None else device
    return torch.tensor([t.data_ptr() for t in tensors], dtype=torch.int64, device=dev)


def piper_ep_a_cap(desc: MoeDesc, n_ranks: int) -> int:
    return int(lib().piper_ep_a_cap(ctypes.byref(desc), int(n_ranks)))


def piper_ep_plan_host(all_counts, rank: int, row_align: int = 1):
    """Host-only: all_counts [n_ranks, E] int32 numpy -> (counts [E_loc], offsets [E_loc + 1], send_base [E])."""
    import numpy as np
    ac = np.ascontiguousarray(all_counts, np.int32)
    R, E = ac.shape
    counts, offsets, send_base = np.empty(E // R, np.int32), np.empty(E // R + 1, np.int32), np.empty(E, np.int32)
    rc = lib().piper_ep_plan_host(_vp(ac.ctypes.data), _i32(E), _i32(R), _i32(rank), _i32(row_align), _vp(counts.ctypes.data),
                                  _vp(offsets.ctypes.data), _vp(send_base.ctypes.data))
    if rc != PIPER_OK:
        raise PiperError(f"piper_ep_plan_host: status {rc}")
    return counts, offsets, send_base


def piper_ep_plan(ctx, all_counts, rank, n_ranks, counts, offsets, send_base, stream=None):
    ctx.check(lib().piper_ep_plan(ctx._h, _ptr(all_counts), int(rank), int(n_ranks), _ptr(counts), _ptr(offsets),
                                  _ptr(send_base), _stream(stream)), "piper_ep_plan")


def piper_ep_dispatch(ctx, x, topk_idx, gates, send_base, rank, n_ranks, peer_xp, peer_src_of, peer_gate_rows, dest_row,
                      stream=None):
    ctx.check(lib().piper_ep_dispatch(ctx._h, _ptr(x), _ptr(topk_idx), _ptr(gates), _ptr(send_base), int(rank), int(n_ranks),
                                      _ptr(peer_xp), _ptr(peer_src_of), _ptr(peer_gate_rows), _ptr(dest_row), _stream(stream)),
              "piper_ep_dispatch")


def piper_ep_finish_recv(ctx, counts, offsets, n_ranks, src_of, gate_rows, rows, stream=None):
    ctx.check(lib().piper_ep_finish_recv(ctx._h, _ptr(counts), _ptr(offsets), int(n_ranks), _ptr(src_of), _ptr(gate_rows),
                                         _ptr(rows), _stream(stream)), "piper_ep_finish_recv")


def piper_ep_combine(ctx, peer_o, topk_idx, dest_row, gates, s, y, stream=None):
    ctx.check(lib().piper_ep_combine(ctx._h, _ptr(peer_o), _ptr(topk_idx), _ptr(dest_row), _ptr(gates), _ptr(s), _ptr(y),
                                     _stream(stream)), "piper_ep_combine")


def piper_ep_dispatch_bwd(ctx, dy, topk_idx, dest_row, gates, peer_o, peer_d_o, dgates, stream=None):
    ctx.check(lib().piper_ep_dispatch_bwd(ctx._h, _ptr(dy), _ptr(topk_idx), _ptr(dest_row), _ptr(gates), _ptr(peer_o),
                                          _ptr(peer_d_o), _ptr(dgates), _stream(stream)), "piper_ep_dispatch_bwd")


def piper_ep_unpack(ctx, peer_dxp, topk_idx, dest_row, dx_shared, dx, stream=None):
    ctx.check(lib().piper_ep_unpack(ctx._h, _ptr(peer_dxp), _ptr(topk_idx), _ptr(dest_row), _ptr(dx_shared), _ptr(dx),
                                    _stream(stream)), "piper_ep_unpack")


def piper_route_bwd(ctx, logits, topk_idx, gates, dgates, dz_sel, stream=None):
    ctx.check(lib().piper_route_bwd(ctx._h, _ptr(logits), _ptr(topk_idx), _ptr(gates), _ptr(dgates), _ptr(dz_sel),
                                    _stream(stream)), "piper_route_bwd")


def chunk_args(bufs: dict) -> ChunkArgs:
    """piper_chunk_args from a dict of tensors (missing / None entries become NULL)."""
    a = ChunkArgs()
    for n in _CHUNK_FIELDS:
        setattr(a, n, _ptr(bufs.get(n)))
    return a


def piper_run_chunk_fwd(ctx, args: ChunkArgs, stream=None):
    ctx.check(lib().piper_run_chunk_fwd(ctx._h, ctypes.byref(args), _stream(stream)), "piper_run_chunk_fwd")


def piper_run_chunk_bwd(ctx, args: ChunkArgs, stream=None):
    ctx.check(lib().piper_run_chunk_bwd(ctx._h, ctypes.byref(args), _stream(stream)), "piper_run_chunk_bwd")


def piper_run_chunk_bwd_input(ctx, args: ChunkArgs, stream=None):
    ctx.check(lib().piper_run_chunk_bwd_input(ctx._h, ctypes.byref(args), _stream(stream)), "piper_run_chunk_bwd_input")


def piper_run_chunk_bwd_weight(ctx, args: ChunkArgs, stream=None):
    ctx.check(lib().piper_run_chunk_bwd_weight(ctx._h, ctypes.byref(args), _stream(stream)), "piper_run_chunk_bwd_weight")


PASS_B, PASS_BI = 0, 1


def piper_dispatch_plan_static(desc, topk_idx, gates, counts, offsets, row_of, src_of, gate_rows, stream=None):
    """F2 on the current device without a context or any allocation (include/piper.h); raises PiperError with the
    library's message when the call is refused."""
    L = lib()
    L.piper_static_last_error.restype = ctypes.c_char_p
    rc = L.piper_dispatch_plan_static(ctypes.byref(desc), _ptr(topk_idx), _ptr(gates), _ptr(counts), _ptr(offsets), _ptr(row_of),
                                      _ptr(src_of), _ptr(gate_rows), _stream(stream))
    if rc != PIPER_OK:
        raise PiperError(f"piper_dispatch_plan_static: status {rc}: {L.piper_static_last_error().decode()}")


def piper_static_scratch_bytes() -> int:
    L = lib()
    L.piper_static_scratch_bytes.restype = ctypes.c_size_t
    return int(L.piper_static_scratch_bytes())


def piper_set_pair_bwd_pass(ctx, bwd_pass: int):
    ctx.check(lib().piper_set_pair_bwd_pass(ctx._h, int(bwd_pass)), "piper_set_pair_bwd_pass")


def piper_pair_prepare(ctx, sm_gemm: int, sm_comm: int):
    ctx.check(lib().piper_pair_prepare(ctx._h, int(sm_gemm), int(sm_comm)), "piper_pair_prepare")


OPT_TC_ROWS_ON_N, OPT_TC_2CTA, OPT_T_SMALL_ROWS, OPT_T_GREEDY, OPT_TC_PROFILE, OPT_FUSED_GATHER, OPT_T_DUAL, OPT_WGRAD_STORE_WARP, OPT_MOVE_ITEMS, OPT_MOVE_CAP = range(10)


def piper_set_option(ctx, option: int, value: int):
    ctx.check(lib().piper_set_option(ctx._h, int(option), int(value)), "piper_set_option")


def piper_chunk_gathers(ctx) -> bool:
    """True when the chunk calls of this context run the fused-gather GEMMs (N2) and do not materialise xp."""
    return bool(lib().piper_chunk_gathers(ctx._h))


def piper_get_option(ctx, option: int) -> int:
    v = _i32(0)
    ctx.check(lib().piper_get_option(ctx._h, int(option), ctypes.byref(v)), "piper_get_option")
    return int(v.value)


TASKS = ("F_ROUTE", "F_SCAN", "F_PACK", "F_GEMM1", "F_GEMM2", "F_SHARED", "F_COMBINE", "B_CGRAD", "B_DGRAD1",
         "B_DGRAD2", "B_WGRAD", "B_SHARED", "B_UNPACK", "B_ROUTE_BWD")  # PIPER_TASK_* of include/piper.h


def piper_run_task(ctx, task, args: ChunkArgs, stream=None):
    t = TASKS.index(task) if isinstance(task, str) else int(task)
    ctx.check(lib().piper_run_task(ctx._h, t, ctypes.byref(args), _stream(stream)), "piper_run_task")


def piper_run_chunk_pair(ctx, fwd_args: ChunkArgs, bwd_args: ChunkArgs, sm_gemm: int, sm_comm: int, stream=None):
    ctx.check(lib().piper_run_chunk_pair(ctx._h, ctypes.byref(fwd_args), ctypes.byref(bwd_args), int(sm_gemm),
                                         int(sm_comm), _stream(stream)), "piper_run_chunk_pair")


ORDER_LIST, ORDER_PROFILE = 0, 1
PART_EXCLUSIVE, PART_SHARED, PART_CHUNK_STREAMS = 0, 1, 2


def piper_set_pair_policy(ctx, order: int, partition: int, task_ms=None):
    """task_ms: 14 floats in TASKS order (ms on the whole device) or None for the library's own estimate."""
    arr = None
    if task_ms is not None:
        arr = (ctypes.c_float * 14)(*[float(v) for v in task_ms])
    ctx.check(lib().piper_set_pair_policy(ctx._h, int(order), int(partition), arr), "piper_set_pair_policy")


CALLER_SLOTS = ("F_PRE", "F_POST", "B_PRE", "B_POST")
SLOT_F_PRE, SLOT_F_POST, SLOT_B_PRE, SLOT_B_POST = range(4)
CALLER_TASK_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int)


def piper_pair_order(ctx, sm_gemm: int, sm_comm: int):
    """Task names in the pick sequence the current policy yields for this split (caller tasks: "X_F_PRE" ...)."""
    order = (ctypes.c_int32 * 18)()
    n = _i32(0)
    ctx.check(lib().piper_pair_order(ctx._h, int(sm_gemm), int(sm_comm), order, ctypes.byref(n)), "piper_pair_order")
    names = TASKS + tuple("X_" + s for s in CALLER_SLOTS)
    return [names[order[i]] for i in range(n.value)]


def piper_pair_set_caller_task(ctx, slot: int, fn, est_ms: float = 0.0, side: int = 1):
    """N3: `fn(stream_ptr: int, sm_count: int)` becomes a task of piper_run_chunk_pair (include/piper.h); it must only
    enqueue work on that stream.  fn = None clears the slot.  The ctypes thunk is kept alive on the context."""
    keep = ctx.__dict__.setdefault("_caller_thunks", {})
    if fn is None:
        ctx.check(lib().piper_pair_set_caller_task(ctx._h, int(slot), CALLER_TASK_FN(0), None, ctypes.c_float(0.0), int(side)),
                  "piper_pair_set_caller_task")
        keep.pop(slot, None)
        return

    def thunk(_user, stream, sms):
        try:
            fn(int(stream or 0), int(sms))
            return 0
        except Exception:  # an exception must not cross the C boundary: the pair call reports the failure
            import traceback
            traceback.print_exc()
            return 1

    cfn = CALLER_TASK_FN(thunk)
    ctx.check(lib().piper_pair_set_caller_task(ctx._h, int(slot), cfn, None, ctypes.c_float(float(est_ms)), int(side)),
              "piper_pair_set_caller_task")
    keep[slot] = cfn


def piper_schedule_search(n, edges, stream_of, dur):
    """Host-only: returns (order, waits[(producer, consumer)], records, makespan)."""
    import numpy as np
    edges = np.ascontiguousarray(edges, np.int32).reshape(-1, 2)
    stream_of = np.ascontiguousarray(stream_of, np.int32)
    dur = np.ascontiguousarray(dur, np.float32)
    order = np.empty(n, np.int32)
    waits = np.empty((max(1, len(edges)), 2), np.int32)
    records = np.empty(n, np.int32)
    nw = _i32(0)
    mk = ctypes.c_float(0)
    rc = lib().piper_schedule_search(_i32(n), _i32(len(edges)), _vp(edges.ctypes.data), _vp(stream_of.ctypes.data),
                                     _vp(dur.ctypes.data), _vp(order.ctypes.data), _vp(waits.ctypes.data),
                                     ctypes.byref(nw), _vp(records.ctypes.data), ctypes.byref(mk))
    if rc != PIPER_OK:
        raise PiperError(f"piper_schedule_search: status {rc}")
    return order, waits[: nw.value].copy(), records, float(mk.value)


def piper_list_schedule(n, edges, stream_of, prio):
    """Host-only: returns (order, waits[(producer, consumer)], records)."""
    import numpy as np
    edges = np.ascontiguousarray(edges, np.int32).reshape(-1, 2)
    stream_of = np.ascontiguousarray(stream_of, np.int32)
    prio = np.ascontiguousarray(prio, np.int32)
    order = np.empty(n, np.int32)
    waits = np.empty((max(1, len(edges)), 2), np.int32)
    records = np.empty(n, np.int32)
    nw = _i32(0)
    rc = lib().piper_list_schedule(_i32(n), _i32(len(edges)), _vp(edges.ctypes.data), _vp(stream_of.ctypes.data),
                                   _vp(prio.ctypes.data), _vp(order.ctypes.data), _vp(waits.ctypes.data),
                                   ctypes.byref(nw), _vp(records.ctypes.data))
    if rc != PIPER_OK:
        raise PiperError(f"piper_list_schedule: status {rc}")
    return order, waits[: nw.value].copy(), records


# ---------------------------------------------------------------------------------- memory plumbing
def to_tensor(a, device="cuda"):
    """Generated numpy tensor -> torch tensor on `device` (uint16 bit patterns are reinterpreted as bf16)."""
    import numpy as np
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16)).to(device).view(torch.bfloat16)
    return torch.from_numpy(a).to(device)


def piper_gemm_path(ctx: Context) -> int:
    """1 = the routed-expert GEMMs of this context run on the tcgen05 kernels, 0 = on the FP32 ALUs."""
    return int(lib().piper_gemm_path(ctx._h))


def alloc_router_buffers(ctx: Context) -> dict:
    """Outputs / scratch of the router GEMMs (N1): logits (an output once w_r is given), dw_r, dx_router, dz_scratch."""
    D, dev = ctx.desc, ctx.device
    return dict(logits=torch.empty((D.T, D.E), dtype=torch.float32, device=dev),
                dw_r=torch.empty((D.d, D.E), dtype=torch.float32, device=dev),
                dx_router=torch.empty((D.T, D.d), dtype=ctx.torch_dtype, device=dev),
                dz_scratch=torch.empty((D.T, D.E), dtype=torch.float32, device=dev))


def alloc_buffers(ctx: Context, backward: bool = True) -> dict:
    """Every output / scratch tensor of one microbatch, as torch CUDA tensors (no arithmetic here)."""
    D, dev, dt = ctx.desc, ctx.device, ctx.torch_dtype
    A = ctx.a_cap
    i32, f32 = torch.int32, torch.float32

    def e(shape, dtype):
        return torch.empty(shape, dtype=dtype, device=dev)

    b = dict(topk_idx=e((D.T, D.k), i32), counts_global=e((D.E,), i32), counts=e((D.E_loc,), i32),
             offsets=e((D.E_loc + 4,), i32), row_of=e((D.T, D.k), i32), src_of=e((A,), i32),
             gates=e((D.T, D.k), f32), gate_rows=e((A,), f32),
             xp=e((A, D.d), dt), g_save=e((A, D.I), dt), u_save=e((A, D.I), dt), h_save=e((A, D.I), dt),
             o=e((A, D.d), dt), y=e((D.T, D.d), dt))
    if D.I_shared:
        b.update(gs_save=e((D.T, D.I_shared), dt), us_save=e((D.T, D.I_shared), dt), hs_save=e((D.T, D.I_shared), dt),
                 s=e((D.T, D.d), dt))
    if backward:
        wt = torch.bfloat16 if D.dw_dtype == DT_BF16 else torch.float32
        b.update(dgates=e((D.T, D.k), f32), dz_sel=e((D.T, D.E if D.gate_mode == 2 else D.k), f32),
                 d_o=e((A, D.d), dt), dg=e((A, D.I), dt), du=e((A, D.I), dt), dxp=e((A, D.d), dt),
                 dx=e((D.T, D.d), dt), dw_gate=e((D.E_loc, D.d, D.I), wt), dw_up=e((D.E_loc, D.d, D.I), wt),
                 dw_down=e((D.E_loc, D.I, D.d), wt))
        if D.I_shared:
            b.update(dgs=e((D.T, D.I_shared), dt), dus=e((D.T, D.I_shared), dt), dxs=e((D.T, D.d), dt),
                     dws_gate=e((D.d, D.I_shared), wt), dws_up=e((D.d, D.I_shared), wt),
                     dws_down=e((D.I_shared, D.d), wt))
    return b
