"""Config recipes C1..C5 (BASELINE.json:configs[0..4]) and reduced parity shapes.

Every tensor is seeded and synthetic (inputs/gen.c).  Readings c-2..c-5, c-13, c-15, c-18, c-19
of SURVEY.md §8(c) are implemented here and restated in DESIGN.md "Input recipe":
  x ~ N(0,1); W_r ~ N(0, std 0.02); W_gate/W_up ~ N(0, std d^-1/2); W_down ~ N(0, std I^-1/2);
  shared expert alike; dY ~ N(0,1); router bias folded into the logits in fp32;
  logits l = fl32(sum_i x[t,i] W_r[i,e]) with the sum in fp64, z = l (+) bias[e] (one fp32 add).
bf16 configs round x, W_*, dY to bf16 (RNE) in the generator; logits stay fp32.
No arithmetic of the method itself (routing, permutation, FFN, combine) lives here.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

from . import gen

# tensor ids of the counter-based generator
TID = dict(x=1, w_r=2, bias=3, w_gate=4, w_up=5, w_down=6, ws_gate=7, ws_up=8, ws_down=9, dy=10)

GATE_SOFTMAX_RENORM, GATE_SIGMOID_RENORM, GATE_SOFTMAX_FULL = 0, 1, 2
DT_F32, DT_BF16 = 0, 1


@dataclasses.dataclass(frozen=True)
class MoeConfig:
    name: str
    T: int
    d: int
    E: int
    k: int
    I: int
    seed: int
    e_lo: int = 0
    E_loc: int = -1            # -1: all experts local
    I_shared: int = 0
    dtype: int = DT_BF16
    gate_mode: int = GATE_SOFTMAX_RENORM
    bias: str = "none"         # none | normal0.5 | zipf1.2
    n_dead: int = 0            # last n_dead experts get bias -inf (variant C4z, reading c-15)
    row_align: int = 1

    @property
    def e_loc(self) -> int:
        return self.E if self.E_loc < 0 else self.E_loc

    @property
    def a_cap(self) -> int:
        return self.T * min(self.k, self.e_loc) + self.e_loc * (self.row_align - 1)


C1 = MoeConfig("C1", T=128, d=64, E=4, k=2, I=128, seed=0, dtype=DT_F32)
C2 = MoeConfig("C2", T=4096, d=4096, E=8, k=2, I=14336, seed=1)
C3 = MoeConfig("C3", T=8192, d=7168, E=256, k=8, I=2048, seed=2, e_lo=0, E_loc=32, I_shared=2048,
               gate_mode=GATE_SIGMOID_RENORM, bias="normal0.5")
C4 = MoeConfig("C4", T=16384, d=2048, E=64, k=6, I=1408, seed=3, bias="zipf1.2")
C4Z = dataclasses.replace(C4, name="C4z", n_dead=4)
C5A = dataclasses.replace(C3, name="C5a", seed=4)
C5B = dataclasses.replace(C3, name="C5b", seed=5)

# Reduced shapes for element-by-element parity: several tiles, ragged tails, empty groups.
C2S = MoeConfig("C2s", T=600, d=256, E=8, k=2, I=512, seed=11)
C3S = MoeConfig("C3s", T=500, d=512, E=64, k=8, I=256, seed=12, e_lo=8, E_loc=8, I_shared=384,
                gate_mode=GATE_SIGMOID_RENORM, bias="normal0.5")
C4S = MoeConfig("C4s", T=1000, d=256, E=16, k=6, I=448, seed=13, bias="zipf1.2", n_dead=2)
C1S = MoeConfig("C1s", T=200, d=72, E=6, k=3, I=88, seed=14, dtype=DT_F32, I_shared=40, e_lo=1, E_loc=4,
                gate_mode=GATE_SIGMOID_RENORM, bias="normal0.5")

# d, I, I_shared that are multiples of 8 only (ragged K blocks and feature tiles), experts of ~450 rows (two row chunks)
C6S = MoeConfig("C6s", T=900, d=328, E=4, k=2, I=296, seed=15, I_shared=200)

BY_NAME = {c.name: c for c in (C1, C2, C3, C4, C4Z, C5A, C5B, C2S, C3S, C4S, C1S, C6S)}


def router_bias(cfg: MoeConfig) -> np.ndarray:
    if cfg.bias == "none":
        b = np.zeros(cfg.E, dtype=np.float32)
    elif cfg.bias == "normal0.5":
        b = gen.normal(cfg.seed, TID["bias"], (cfg.E,), std=0.5)
    elif cfg.bias == "zipf1.2":
        p = np.arange(1, cfg.E + 1, dtype=np.float64) ** -1.2
        b = np.log(p / p.sum()).astype(np.float32)
    else:
        raise ValueError(cfg.bias)
    if cfg.n_dead:
        b = b.copy()
        b[cfg.E - cfg.n_dead:] = -np.inf
    return b


def as_f64(a: np.ndarray) -> np.ndarray:
    """Exact widening of a generated tensor (fp32, or bf16 bits as uint16) to fp64."""
    if a.dtype == np.uint16:
        return gen.bf16_to_f32(a).astype(np.float64)
    return a.astype(np.float64)


def make_inputs(cfg: MoeConfig, weights: bool = True, with_dy: bool = True) -> dict:
    """All inputs of one microbatch as host numpy arrays (bf16 tensors as uint16 bit patterns)."""
    bf = cfg.dtype == DT_BF16
    s = cfg.seed
    out: dict = {"cfg": cfg}
    out["x"] = gen.normal(s, TID["x"], (cfg.T, cfg.d), bf16=bf)
    out["w_r"] = gen.normal(s, TID["w_r"], (cfg.d, cfg.E), std=0.02, bf16=bf)
    out["bias"] = router_bias(cfg)
    # logits: fp64 sum rounded once to fp32, then one fp32 add of the bias (reading c-18)
    l32 = (as_f64(out["x"]) @ as_f64(out["w_r"])).astype(np.float32)
    out["logits"] = (l32 + out["bias"][None, :]).astype(np.float32)
    if weights:
        el = cfg.e_loc
        # Local experts only: expert (e_lo + i) of the global model is local index i.  The element
        # offset i0 makes the local slice identical to the slice of a full [E, ...] tensor.
        per = cfg.d * cfg.I
        out["w_gate"] = gen.normal(s, TID["w_gate"], (el, cfg.d, cfg.I), std=cfg.d ** -0.5, bf16=bf, i0=cfg.e_lo * per)
        out["w_up"] = gen.normal(s, TID["w_up"], (el, cfg.d, cfg.I), std=cfg.d ** -0.5, bf16=bf, i0=cfg.e_lo * per)
        out["w_down"] = gen.normal(s, TID["w_down"], (el, cfg.I, cfg.d), std=cfg.I ** -0.5, bf16=bf, i0=cfg.e_lo * per)
        if cfg.I_shared:
            Is = cfg.I_shared
            out["ws_gate"] = gen.normal(s, TID["ws_gate"], (1, cfg.d, Is), std=cfg.d ** -0.5, bf16=bf)
            out["ws_up"] = gen.normal(s, TID["ws_up"], (1, cfg.d, Is), std=cfg.d ** -0.5, bf16=bf)
            out["ws_down"] = gen.normal(s, TID["ws_down"], (1, Is, cfg.d), std=Is ** -0.5, bf16=bf)
    if with_dy:
        out["dy"] = gen.normal(s, TID["dy"], (cfg.T, cfg.d), bf16=bf)
    return out


def flops_fwd_bwd(cfg: MoeConfig, a_rows: int) -> float:
    """18*d*I per routed row + 18*d*I_sh per token."""
    return 18.0 * cfg.d * cfg.I * a_rows + 18.0 * cfg.d * cfg.I_shared * cfg.T


def uniform_config(rows_per_expert: int) -> MoeConfig:
    """Microbenchmark workload (bench.py --uniform-rows): C3's routed layer shape (d = 7168, I = 2048, 32 local
    experts, top-8, no shared expert) with exactly `rows_per_expert` rows in every expert, so that a GEMM's rate can be
    read as a function of the group length alone."""
    E, k = 32, 8
    return MoeConfig(f"U{rows_per_expert}", T=rows_per_expert * E // k, d=7168, E=E, k=k, I=2048, seed=7, row_align=128)


def uniform_logits(cfg: MoeConfig) -> np.ndarray:
    """Logits that send token t to experts (t k + j) mod E, j < k, in that order of preference."""
    lg = np.full((cfg.T, cfg.E), -10.0, dtype=np.float32)
    t = np.arange(cfg.T)
    for j in range(cfg.k):
        lg[t, (t * cfg.k + j) % cfg.E] = np.float32(1.0 - 0.01 * j)
    return lg
