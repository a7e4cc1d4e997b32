"""Python face of the CPU oracle — TEST INFRASTRUCTURE ONLY.

ctypes marshalling over oracle/liboracle.so plus the composition of the definition's steps
(SURVEY.md §8c Definition 1-5) into a full forward/backward and into the sampled forms used at
BASELINE.json's full sizes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the CUDA package.
All floating-point results are fp64 numpy arrays.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

_lib = None
_i32 = ctypes.c_int32
_vp = ctypes.c_void_p


class OracleDesc(ctypes.Structure):
    _fields_ = [(n, _i32) for n in ("T", "d", "E", "k", "e_lo", "E_loc", "I", "dtype", "gate_mode", "row_align")]


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        for name in ("oracle_router_fwd", "oracle_router_bwd", "oracle_route_topk", "oracle_permute", "oracle_pack", "oracle_ffn_fwd_rows", "oracle_combine",
                     "oracle_combine_bwd", "oracle_ffn_bwd_rows", "oracle_wgrad", "oracle_ffn_cols", "oracle_unpack",
                     "oracle_route_bwd", "oracle_list_schedule"):
            getattr(_lib, name).restype = ctypes.c_int
        _lib.oracle_set_threads.argtypes = [ctypes.c_int]
        _lib.oracle_get_threads.restype = ctypes.c_int
    return _lib


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def _p(a):
    if a is None:
        return _vp(0)
    assert a.flags.c_contiguous
    return _vp(a.ctypes.data)


def _desc(cfg, I=None, row_align=None) -> OracleDesc:
    return OracleDesc(cfg.T, cfg.d, cfg.E, cfg.k, cfg.e_lo, cfg.e_loc, cfg.I if I is None else I, cfg.dtype,
                      cfg.gate_mode, cfg.row_align if row_align is None else row_align)


def _chk(rc, what):
    if rc != 0:
        raise ValueError(f"oracle {what}: precondition violated (rc={rc})")


def _f64(a: np.ndarray) -> np.ndarray:
    """Exact widening of fp32 / bf16-bit arrays to fp64."""
    if a.dtype == np.uint16:
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return np.ascontiguousarray(a, dtype=np.float64)


# ----------------------------------------------------------------------------------------- steps
def router_fwd(cfg, x, w_r, bias=None):
    """z = x W_r + bias in fp64, unrounded (plain loops in oracle.cpp)."""
    z = np.empty((cfg.T, cfg.E), np.float64)
    b32 = None if bias is None else np.ascontiguousarray(bias, np.float32)
    D = _desc(cfg)
    _chk(lib().oracle_router_fwd(ctypes.byref(D), _p(np.ascontiguousarray(x)), _p(np.ascontiguousarray(w_r)), _p(b32), _p(z)),
         "router_fwd")
    return z


def dense_dz(cfg, topk_idx, dz):
    """dz_sel [T,k] scattered to the selected experts' columns of a dense [T,E] array (mode 2: dz is dense already)."""
    if cfg.gate_mode == 2:
        return np.ascontiguousarray(dz, np.float64)
    dense = np.zeros((cfg.T, cfg.E))
    np.put_along_axis(dense, topk_idx.astype(np.int64), dz, axis=1)
    return dense


def router_bwd(cfg, x, w_r, dz_dense):
    """dW_r = x^T dz and dX_r = dz W_r^T (plain loops in oracle.cpp)."""
    dw = np.empty((cfg.d, cfg.E), np.float64)
    dx = np.empty((cfg.T, cfg.d), np.float64)
    D = _desc(cfg)
    _chk(lib().oracle_router_bwd(ctypes.byref(D), _p(np.ascontiguousarray(x)), _p(np.ascontiguousarray(w_r)),
                                 _p(np.ascontiguousarray(dz_dense, np.float64)), _p(dw), _p(dx)), "router_bwd")
    return dw, dx


def route_topk(cfg, logits):
    logits = np.ascontiguousarray(logits, dtype=np.float32)
    idx = np.empty((cfg.T, cfg.k), np.int32)
    gates = np.empty((cfg.T, cfg.k), np.float64)
    cg = np.empty(cfg.E, np.int32)
    D = _desc(cfg)
    _chk(lib().oracle_route_topk(ctypes.byref(D), _p(logits), _p(idx), _p(gates), _p(cg)), "route_topk")
    return idx, gates, cg


def permute(cfg, topk_idx, a_cap=None, row_align=None):
    a_cap = cfg.a_cap if a_cap is None else a_cap
    counts = np.empty(cfg.e_loc, np.int32)
    offsets = np.empty(cfg.e_loc + 1, np.int32)
    row_of = np.empty((cfg.T, cfg.k), np.int32)
    src_of = np.empty(a_cap, np.int32)
    D = _desc(cfg, row_align=row_align)
    _chk(lib().oracle_permute(ctypes.byref(D), _p(np.ascontiguousarray(topk_idx, np.int32)), _i32(a_cap), _p(counts),
                              _p(offsets), _p(row_of), _p(src_of)), "permute")
    return counts, offsets, row_of, src_of


def pack(cfg, x, src_of, gates):
    a_cap = src_of.shape[0]
    xp = np.empty((a_cap, cfg.d), np.float64)
    gr = np.empty(a_cap, np.float64)
    D = _desc(cfg)
    _chk(lib().oracle_pack(ctypes.byref(D), _p(x), _p(src_of), _p(gates), _i32(a_cap), _p(xp), _p(gr)), "pack")
    return xp, gr


def ffn_fwd_rows(cfg, I, X, ex, wg, wu, wd, want=("G", "U", "H", "O")):
    X = np.ascontiguousarray(X, np.float64)
    ex = np.ascontiguousarray(ex, np.int32)
    n = X.shape[0]
    out = {"G": None, "U": None, "H": None, "O": None}
    for key in want:
        out[key] = np.empty((n, cfg.d if key == "O" else I), np.float64)
    D = _desc(cfg, I=I)
    _chk(lib().oracle_ffn_fwd_rows(ctypes.byref(D), _i32(I), _i32(n), _p(X), _p(ex), _p(wg), _p(wu), _p(wd),
                                   _p(out["G"]), _p(out["U"]), _p(out["H"]), _p(out["O"])), "ffn_fwd_rows")
    return out


def combine(cfg, O, row_of, gates, S=None):
    Y = np.empty((cfg.T, cfg.d), np.float64)
    D = _desc(cfg)
    _chk(lib().oracle_combine(ctypes.byref(D), _p(O), _p(row_of), _p(gates), _p(S), _p(Y)), "combine")
    return Y


def combine_bwd(cfg, dy, O, row_of, src_of, gate_rows):
    a_cap = src_of.shape[0]
    dO = np.empty((a_cap, cfg.d), np.float64)
    dgates = np.empty((cfg.T, cfg.k), np.float64)
    D = _desc(cfg)
    _chk(lib().oracle_combine_bwd(ctypes.byref(D), _p(dy), _p(O), _p(row_of), _p(src_of), _p(gate_rows), _i32(a_cap),
                                  _p(dO), _p(dgates)), "combine_bwd")
    return dO, dgates


def ffn_bwd_rows(cfg, I, X, ex, dO, wg, wu, wd):
    X = np.ascontiguousarray(X, np.float64)
    dO = np.ascontiguousarray(dO, np.float64)
    ex = np.ascontiguousarray(ex, np.int32)
    n = X.shape[0]
    dX = np.empty((n, cfg.d), np.float64)
    dG, dU, H = (np.empty((n, I), np.float64) for _ in range(3))
    D = _desc(cfg, I=I)
    _chk(lib().oracle_ffn_bwd_rows(ctypes.byref(D), _i32(I), _i32(n), _p(X), _p(ex), _p(dO), _p(wg), _p(wu), _p(wd),
                                   _p(dX), _p(dG), _p(dU), _p(H)), "ffn_bwd_rows")
    return dX, dG, dU, H


def wgrad(cfg, I, n_e, X, ex, dG, dU, H, dO):
    X, dG, dU, H, dO = (np.ascontiguousarray(a, np.float64) for a in (X, dG, dU, H, dO))
    ex = np.ascontiguousarray(ex, np.int32)
    dWg = np.empty((n_e, cfg.d, I), np.float64)
    dWu = np.empty((n_e, cfg.d, I), np.float64)
    dWd = np.empty((n_e, I, cfg.d), np.float64)
    D = _desc(cfg, I=I)
    _chk(lib().oracle_wgrad(ctypes.byref(D), _i32(I), _i32(n_e), _i32(X.shape[0]), _p(X), _p(ex), _p(dG), _p(dU),
                            _p(H), _p(dO), _p(dWg), _p(dWu), _p(dWd)), "wgrad")
    return dWg, dWu, dWd


def ffn_cols(cfg, I, e, X, dO, J, wg, wu, wd):
    X = np.ascontiguousarray(X, np.float64)
    dO = np.ascontiguousarray(dO, np.float64)
    J = np.ascontiguousarray(J, np.int32)
    n, nJ = X.shape[0], J.shape[0]
    Hc, dGc, dUc = (np.empty((n, nJ), np.float64) for _ in range(3))
    D = _desc(cfg, I=I)
    _chk(lib().oracle_ffn_cols(ctypes.byref(D), _i32(I), _i32(e), _i32(n), _p(X), _p(dO), _i32(nJ), _p(J), _p(wg),
                               _p(wu), _p(wd), _p(Hc), _p(dGc), _p(dUc)), "ffn_cols")
    return Hc, dGc, dUc


def unpack(cfg, dXp, row_of, dXs=None):
    dX = np.empty((cfg.T, cfg.d), np.float64)
    D = _desc(cfg)
    _chk(lib().oracle_unpack(ctypes.byref(D), _p(dXp), _p(row_of), _p(dXs), _p(dX)), "unpack")
    return dX


def route_bwd(cfg, logits, topk_idx, dgates):
    logits = np.ascontiguousarray(logits, np.float32)
    dgates = np.ascontiguousarray(dgates, np.float64)
    dz = np.empty((cfg.T, cfg.E if cfg.gate_mode == 2 else cfg.k), np.float64)
    D = _desc(cfg)
    _chk(lib().oracle_route_bwd(ctypes.byref(D), _p(logits), _p(topk_idx), _p(dgates), _p(dz)), "route_bwd")
    return dz


def list_schedule(n, edges, stream_of, prio):
    edges = np.ascontiguousarray(edges, np.int32).reshape(-1, 2)
    stream_of = np.ascontiguousarray(stream_of, np.int32)
    prio = np.ascontiguousarray(prio, np.int32)
    order = np.empty(n, np.int32)
    n_desc = np.empty(n, np.int32)
    waits = np.empty((max(1, edges.shape[0]), 2), np.int32)
    n_waits = _i32(0)
    records = np.empty(n, np.int32)
    _chk(lib().oracle_list_schedule(_i32(n), _i32(edges.shape[0]), _p(edges), _p(stream_of), _p(prio), _p(order),
                                    _p(n_desc), _p(waits), ctypes.byref(n_waits), _p(records)), "list_schedule")
    return order, n_desc, waits[: n_waits.value].copy(), records


# --------------------------------------------------------------------------- full-tensor chain
def expert_of_rows(cfg, topk_idx, src_of):
    """Local expert index of every packed row (-1 for pad/unused rows)."""
    flat = topk_idx.reshape(-1)
    return np.where(src_of >= 0, flat[np.maximum(src_of, 0)] - cfg.e_lo, -1).astype(np.int32)


def forward(cfg, inp, a_cap=None, row_align=None):
    """Definition steps 1-4 on full tensors.  Returns every intermediate (fp64 / int32)."""
    r = {}
    r["topk_idx"], r["gates"], r["counts_global"] = route_topk(cfg, inp["logits"])
    r["counts"], r["offsets"], r["row_of"], r["src_of"] = permute(cfg, r["topk_idx"], a_cap, row_align)
    r["xp"], r["gate_rows"] = pack(cfg, inp["x"], r["src_of"], r["gates"])
    r["ex"] = expert_of_rows(cfg, r["topk_idx"], r["src_of"])
    f = ffn_fwd_rows(cfg, cfg.I, r["xp"], r["ex"], inp["w_gate"], inp["w_up"], inp["w_down"])
    r.update(g=f["G"], u=f["U"], h=f["H"], o=f["O"])
    r["s"] = None
    if cfg.I_shared:
        xs = _f64(inp["x"])
        fs = ffn_fwd_rows(cfg, cfg.I_shared, xs, np.zeros(cfg.T, np.int32), inp["ws_gate"], inp["ws_up"], inp["ws_down"])
        r.update(s=fs["O"], gs=fs["G"], us=fs["U"], hs=fs["H"])
    r["y"] = combine(cfg, r["o"], r["row_of"], r["gates"], r["s"])
    return r


def backward(cfg, inp, fwd):
    """Definition step 5 on full tensors, from the forward's exact (unrounded) intermediates."""
    b = {}
    b["d_o"], b["dgates"] = combine_bwd(cfg, inp["dy"], fwd["o"], fwd["row_of"], fwd["src_of"], fwd["gate_rows"])
    b["dxp"], b["dg"], b["du"], h = ffn_bwd_rows(cfg, cfg.I, fwd["xp"], fwd["ex"], b["d_o"], inp["w_gate"], inp["w_up"],
                                                 inp["w_down"])
    b["dw_gate"], b["dw_up"], b["dw_down"] = wgrad(cfg, cfg.I, cfg.e_loc, fwd["xp"], fwd["ex"], b["dg"], b["du"], h,
                                                   b["d_o"])
    dxs = None
    if cfg.I_shared:
        xs, dys = _f64(inp["x"]), _f64(inp["dy"])
        z0 = np.zeros(cfg.T, np.int32)
        dxs, dgs, dus, hs = ffn_bwd_rows(cfg, cfg.I_shared, xs, z0, dys, inp["ws_gate"], inp["ws_up"], inp["ws_down"])
        b["dws_gate"], b["dws_up"], b["dws_down"] = wgrad(cfg, cfg.I_shared, 1, xs, z0, dgs, dus, hs, dys)
        b["dx_shared"] = dxs
    b["dx"] = unpack(cfg, b["dxp"], fwd["row_of"], dxs)
    b["dz"] = route_bwd(cfg, inp["logits"], fwd["topk_idx"], b["dgates"])
    return b


def router_terms(cfg, inp, fwd, bwd):
    """Outside the library boundary (reading c-16): dW_r = x^T dz and the router part of dX."""
    dz = bwd["dz"]
    if cfg.gate_mode != 2:
        dense = np.zeros((cfg.T, cfg.E))
        np.put_along_axis(dense, fwd["topk_idx"].astype(np.int64), dz, axis=1)
        dz = dense
    return _f64(inp["x"]).T @ dz, dz @ _f64(inp["w_r"]).T


# ------------------------------------------------------------- sampled forms (full-size configs)
def routing(cfg, inp, a_cap=None):
    """Steps 1-2 only (cheap at any size)."""
    r = {}
    r["topk_idx"], r["gates"], r["counts_global"] = route_topk(cfg, inp["logits"])
    r["counts"], r["offsets"], r["row_of"], r["src_of"] = permute(cfg, r["topk_idx"], a_cap)
    return r


def sample_tokens(cfg, inp, rt, tokens, backward_too=True):
    """Y[t], O rows, dgates[t], dX[t] for the listed tokens, each from the definition directly."""
    tokens = np.asarray(tokens, np.int64)
    k = cfg.k
    xs = _f64(inp["x"][tokens])
    slots = [(ti, j) for ti, t in enumerate(tokens) for j in range(k) if rt["row_of"][t, j] >= 0]
    X = np.stack([xs[ti] for ti, _ in slots]) if slots else np.zeros((0, cfg.d))
    ex = np.array([rt["topk_idx"][tokens[ti], j] - cfg.e_lo for ti, j in slots], np.int32)
    f = ffn_fwd_rows(cfg, cfg.I, X, ex, inp["w_gate"], inp["w_up"], inp["w_down"])
    out = {"tokens": tokens, "slots": slots, "o_rows": f["O"], "g_rows": f["G"], "u_rows": f["U"], "h_rows": f["H"],
           "rows": np.array([rt["row_of"][tokens[ti], j] for ti, j in slots], np.int64)}
    y = np.zeros((len(tokens), cfg.d))
    for q, (ti, j) in enumerate(slots):
        y[ti] += rt["gates"][tokens[ti], j] * f["O"][q]
    z0 = np.zeros(len(tokens), np.int32)
    if cfg.I_shared:
        fs = ffn_fwd_rows(cfg, cfg.I_shared, xs, z0, inp["ws_gate"], inp["ws_up"], inp["ws_down"], want=("O",))
        y += fs["O"]
    out["y"] = y
    if not backward_too:
        return out
    dys = _f64(inp["dy"][tokens])
    dgates = np.zeros((len(tokens), k))
    dO = np.zeros((len(slots), cfg.d))
    for q, (ti, j) in enumerate(slots):
        dgates[ti, j] = dys[ti] @ f["O"][q]
        dO[q] = rt["gates"][tokens[ti], j] * dys[ti]
    dXp, dG, dU, _ = ffn_bwd_rows(cfg, cfg.I, X, ex, dO, inp["w_gate"], inp["w_up"], inp["w_down"])
    dx = np.zeros((len(tokens), cfg.d))
    for q, (ti, j) in enumerate(slots):
        dx[ti] += dXp[q]
    if cfg.I_shared:
        dxs, _, _, _ = ffn_bwd_rows(cfg, cfg.I_shared, xs, z0, dys, inp["ws_gate"], inp["ws_up"], inp["ws_down"])
        dx += dxs
    out.update(dgates=dgates, dx=dx, dxp_rows=dXp, dg_rows=dG, du_rows=dU)
    return out


def sample_rows(cfg, inp, rt, rows, backward_too=True):
    """O[r] (and dXp[r], dG[r], dU[r]) for the listed non-pad packed rows, each from the definition directly:
    row r holds token src_of[r] // k at expert topk_idx[src_of[r]]; dO[r] = gates[src_of[r]] * dY[token]."""
    rows = np.asarray(rows, np.int64)
    a = rt["src_of"][rows].astype(np.int64)
    assert (a >= 0).all(), "sample_rows wants non-pad rows"
    tok = a // cfg.k
    ex = (rt["topk_idx"].reshape(-1)[a] - cfg.e_lo).astype(np.int32)
    X = _f64(inp["x"][tok])
    f = ffn_fwd_rows(cfg, cfg.I, X, ex, inp["w_gate"], inp["w_up"], inp["w_down"])
    out = {"rows": rows, "tokens": tok, "o": f["O"], "g": f["G"], "u": f["U"], "h": f["H"]}
    if backward_too:
        dO = rt["gates"].reshape(-1)[a][:, None] * _f64(inp["dy"][tok])
        dXp, dG, dU, _ = ffn_bwd_rows(cfg, cfg.I, X, ex, dO, inp["w_gate"], inp["w_up"], inp["w_down"])
        out.update(dxp=dXp, dg=dG, du=dU)
    return out


def sample_route_bwd(cfg, inp, rt, tokens, dgates):
    """dz_sel[t] for the listed tokens from the oracle's dgates[t] (gate backward is per token)."""
    import dataclasses
    tokens = np.asarray(tokens, np.int64)
    sub = dataclasses.replace(cfg, T=len(tokens))
    return route_bwd(sub, np.ascontiguousarray(inp["logits"][tokens]), np.ascontiguousarray(rt["topk_idx"][tokens]),
                     np.ascontiguousarray(dgates))


def sample_wgrad(cfg, inp, rt, e_local, J):
    """dW_gate[e][:, J], dW_up[e][:, J] ([d, nJ]) and dW_down[e][J, :] ([nJ, d]) for local expert e_local."""
    lo, cnt = int(rt["offsets"][e_local]), int(rt["counts"][e_local])
    rows = np.arange(lo, lo + cnt)
    a = rt["src_of"][rows].astype(np.int64)
    tok = a // cfg.k
    X = _f64(inp["x"][tok])
    gate_rows = rt["gates"].reshape(-1)[a]
    dO = gate_rows[:, None] * _f64(inp["dy"][tok])
    Hc, dGc, dUc = ffn_cols(cfg, cfg.I, e_local, X, dO, J, inp["w_gate"], inp["w_up"], inp["w_down"])
    return X.T @ dGc, X.T @ dUc, Hc.T @ dO


def sample_wgrad_shared(cfg, inp, J):
    X, dO = _f64(inp["x"]), _f64(inp["dy"])
    Hc, dGc, dUc = ffn_cols(cfg, cfg.I_shared, 0, X, dO, J, inp["ws_gate"], inp["ws_up"], inp["ws_down"])
    return X.T @ dGc, X.T @ dUc, Hc.T @ dO
