"""Helpers shared by the GPU parity tests: host<->device marshalling and the tolerance check."""
import numpy as np
import torch

import paper_2606_11169_b200 as piper
from inputs import configs

# north_star / reading c-23: bf16 rel. Frobenius <= 5e-3 and max|err| <= 2e-2 max|ref|; fp32 1e-5 both.
TOL = {configs.DT_BF16: (5e-3, 2e-2), configs.DT_F32: (1e-5, 1e-5)}


def desc_of(cfg, gemm_impl=piper.GEMM_AUTO, dw_dtype=None):
    return piper.make_desc(cfg.T, cfg.d, cfg.E, cfg.k, cfg.I, e_lo=cfg.e_lo, E_loc=cfg.e_loc, I_shared=cfg.I_shared,
                           dtype=cfg.dtype, gate_mode=cfg.gate_mode, row_align=cfg.row_align, gemm_impl=gemm_impl,
                           dw_dtype=dw_dtype)


def to_dev(a: np.ndarray, device="cuda"):
    """Generated tensor -> CUDA tensor (uint16 bit patterns become bf16)."""
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16)).to(device).view(torch.bfloat16)
    return torch.from_numpy(a).to(device)


def to_np(t: torch.Tensor) -> np.ndarray:
    """CUDA tensor -> host numpy (floating types widened exactly to fp64)."""
    if t.dtype in (torch.bfloat16, torch.float32):
        return t.detach().to("cpu", torch.float64).numpy()
    return t.detach().cpu().numpy()


def upload_inputs(inp: dict) -> dict:
    keys = ("logits", "x", "dy", "w_gate", "w_up", "w_down", "ws_gate", "ws_up", "ws_down")
    return {k: to_dev(inp[k]) for k in keys if k in inp}


def errs(got: np.ndarray, ref: np.ndarray):
    got, ref = np.asarray(got, np.float64), np.asarray(ref, np.float64)
    den = np.linalg.norm(ref)
    frob = np.linalg.norm(got - ref) / den if den > 0 else np.linalg.norm(got - ref)
    mx = np.abs(ref).max() if ref.size else 0.0
    rel_max = (np.abs(got - ref).max() / mx) if mx > 0 else (np.abs(got - ref).max() if ref.size else 0.0)
    return frob, rel_max


def check_close(name, got, ref, dtype, scale=1.0):
    tf, tm = TOL[dtype]
    assert np.all(np.isfinite(got)), f"{name}: non-finite values"
    frob, rel_max = errs(got, ref)
    assert frob <= tf * scale and rel_max <= tm * scale, f"{name}: frob {frob:.3e} (<= {tf * scale:.1e}) max {rel_max:.3e} (<= {tm * scale:.1e})"
    return frob, rel_max
