"""bench.py — MoE fwd+bwd tokens/s of the per-device expert-parallel chunk on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2|C3|C4|C4z] [--impl piper|reference] [--pair]

A step = one pass of the whole hot path over one microbatch: forward chunk F1-F5 then backward chunk
B1-B6 through the C-ABI (piper_run_chunk_fwd + piper_run_chunk_bwd).  Default workload:
C2 = BASELINE.json configs[1] (Mixtral-8x7B-shaped layer), seeded synthetic inputs (inputs/configs.py).
Multi-GPU (torchrun): every rank runs its own microbatch (same layer shape, seed + 1000*rank), no
data-path collective, value = all ranks' tokens / max-over-ranks time: weak scaling.

One JSON line on stdout (rank 0); everything else goes to stderr.  --impl reference times the CPU oracle
(oracle/) on a bounded sample of the same workload on the host cores.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "moe_fwd_bwd_tokens_per_s"
UNIT = "tokens/s"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks():
    """MEASURED_PEAKS.json (driver-written) or the fallback of /opt/skills/guides/B200_PROFILING.md."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            m = json.load(f)
        return dict(hbm=float(m["hbm_gbs"]), tf_burst=float(m["bf16_tflops"]),
                    tf_sustained=float(m.get("bf16_tflops_sustained", m["bf16_tflops"])), kind="measured")
    return dict(hbm=6650.0, tf_burst=1590.0, tf_sustained=1400.0, kind="fallback")


STORED = os.path.join("profiles", "r2_traffic.json.txt")


def stored_ncu():
    """Figures that this run does NOT measure (ncu cannot run inside a timed bench): dram bytes per launch from the
    committed `ncu --set full` capture and per-launch gpu__time_duration of the row movers from the committed launch
    lists.  Everything taken from here is labelled with its source file in the JSON line."""
    try:
        with open(os.path.join(ROOT, STORED)) as f:
            return json.load(f)
    except (OSError, ValueError):
        return {}


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML every 5 ms.  The thread is started before the warm-up (NVML
    start-up stays outside the timed region) and records only between begin() and end(): the timed region."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None
        self.recording, self.power_w, self.power_limit_w = False, [], None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            try:
                self.power_limit_w = pynvml.nvmlDeviceGetEnforcedPowerLimit(self.h) / 1000.0
            except Exception:
                pass
        except Exception as e:  # pragma: no cover
            log("clock sampler unavailable:", e)
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self.stop_flag:
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                if self.recording:
                    self.samples.append(mhz)
                    for bit, nm in names.items():
                        if r & bit:
                            self.reasons.add(nm)
                    self.power_w.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(0.005)

    def begin(self):
        self.samples, self.reasons, self.power_w, self.recording = [], set(), [], True

    def end(self):
        self.recording = False
        s = sorted(self.samples)
        # NVML refreshes its clock / reason / power readings every ~100 ms: a 0.15 s region sees one or two distinct values,
        # and a reason bit that was clear at those instants stays unreported.  The board power beside its limit says
        # independently whether the power cap is what holds the clock.
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_min_mhz": s[0] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s),
                "power_w_max": round(max(self.power_w), 1) if self.power_w else None, "power_limit_w": self.power_limit_w}


# --------------------------------------------------------------------------------- reference arm
def oracle_sample_cfg(cfg, tokens: int):
    """Bounded sample of the workload for the CPU oracle: the first `tokens` tokens of the same layer
    (same d, E, k, I, weights and seed; only T shrinks)."""
    return dataclasses.replace(cfg, T=tokens, name=f"{cfg.name}[first {tokens} tokens]")


def time_oracle(cfg, tokens: int, steps: int, warmup: int):
    """Seconds per fwd+bwd pass of the oracle, as it stands, on `tokens` tokens; threads = host cores."""
    from inputs import configs
    from oracle import oracle
    cores = os.cpu_count() or 1
    oracle.set_threads(cores)
    scfg = oracle_sample_cfg(cfg, tokens)
    inp = configs.make_inputs(scfg)
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        f = oracle.forward(scfg, inp)
        oracle.backward(scfg, inp, f)
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
        log(f"oracle pass {i}: {dt:.2f} s on {tokens} tokens")
    return sum(times) / len(times), cores, scfg


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return  # rank 0 alone runs the reference arm
    tokens = args.oracle_tokens or 8
    sec, cores, scfg = time_oracle(cfg, tokens, args.steps, args.warmup)
    value = tokens / sec
    sample = (f"CPU oracle (oracle/, fp64 plain loops, OpenMP over rows) fwd+bwd on the first {tokens} tokens of "
              f"{cfg.name} (same d/E/k/I and weights), {args.steps} passes after {args.warmup} warm-up")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, extra={"sample_tokens": tokens}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(cfg, extra=None):
    w = {"workload": f"{cfg.name}: one MoE layer fwd+bwd chunk, T={cfg.T} d={cfg.d} E={cfg.E} (local {cfg.e_loc}) "
                     f"top-{cfg.k} I={cfg.I} I_shared={cfg.I_shared} gate_mode={cfg.gate_mode}",
         "T": cfg.T, "d": cfg.d, "E": cfg.E, "E_loc": cfg.e_loc, "k": cfg.k, "I": cfg.I, "I_shared": cfg.I_shared,
         "seed": cfg.seed, "storage": "bf16" if cfg.dtype == 1 else "f32", "accumulate": "f32",
         "row_align": cfg.row_align,
         "l2": "working set (weights + dW, GBs) exceeds the 126 MB L2 every step; no explicit flush"}
    if extra:
        w.update(extra)
    return w


# ------------------------------------------------------------------------------ algorithmic work
def task_work(cfg, A: int, t_touched: int):
    """Algorithmic FLOP (GEMM tasks) or HBM bytes (movers) per task, SURVEY.md §8(d) / DESIGN.md §6."""
    b = 2 if cfg.dtype == 1 else 4
    d, I, Is, T, k = cfg.d, cfg.I, cfg.I_shared, cfg.T, cfg.k
    sh = 1 if Is else 0
    w = {
        "F_ROUTE": ("hbm", T * cfg.E * 4 + T * k * 8 + cfg.E * 4),
        "F_SCAN": ("hbm", 2 * T * k * 4 + A * 4),
        "F_PACK": ("hbm", (t_touched + A) * d * b + 8 * A),
        "F_GEMM1": ("tensor", 4.0 * d * I * A),
        "F_GEMM2": ("tensor", 2.0 * d * I * A),
        "F_COMBINE": ("hbm", (A + T + sh * T) * d * b + 8 * T * k),
        "B_CGRAD": ("hbm", (t_touched + 2 * A) * d * b),
        "B_DGRAD1": ("tensor", 2.0 * d * I * A),
        "B_DGRAD2": ("tensor", 4.0 * d * I * A),
        "B_WGRAD": ("tensor", 6.0 * d * I * A),
        "B_UNPACK": ("hbm", (A + T + sh * T) * d * b),
        "B_ROUTE_BWD": ("hbm", T * k * 16),
    }
    if Is:
        w["F_SHARED"] = ("tensor", 6.0 * d * Is * T)
        w["B_SHARED"] = ("tensor", 12.0 * d * Is * T)
    return w


# ------------------------------------------------------------------------------- multi-rank glue
def rank_config(cfg, rank: int):
    """Every rank runs its own microbatch of the same layer shape (replicas, weak scaling): seed + 1000*rank."""
    return dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)


def max_over_ranks(ms: float, world: int, device):
    """The slowest rank's time (all-reduce MAX over the default process group; identity at world 1)."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_tokens_per_s(cfg, world: int, ms_per_step: float) -> float:
    return world * cfg.T / (ms_per_step * 1e-3)


# ----------------------------------------------------------------------------------- piper arm
INPUT_NAMES = ("logits", "x", "dy", "w_gate", "w_up", "w_down", "ws_gate", "ws_up", "ws_down")


def desc_of(piper, cfg, dw_f32=False):
    return piper.make_desc(cfg.T, cfg.d, cfg.E, cfg.k, cfg.I, e_lo=cfg.e_lo, E_loc=cfg.e_loc, I_shared=cfg.I_shared,
                           dtype=cfg.dtype, gate_mode=cfg.gate_mode, row_align=cfg.row_align,
                           dw_dtype=piper.DT_F32 if dw_f32 else None)


class Workload:
    """One config on this rank: inputs generated and resident, context and buffers allocated."""

    def __init__(self, args, cfg, rank, local):
        import torch
        import paper_2606_11169_b200 as piper
        from inputs import configs
        self.args, self.cfg, self.piper, self.torch = args, cfg, piper, torch
        self.dev = torch.device("cuda", local)
        self.rcfg = rank_config(cfg, rank)
        t0 = time.time()
        self.inp = configs.make_inputs(self.rcfg)
        if getattr(args, "uniform_rows", 0):
            self.inp["logits"] = configs.uniform_logits(self.rcfg)
        log(f"[rank {rank}] {cfg.name}: inputs generated in {time.time() - t0:.1f} s")
        self.ctx = piper.Context(desc_of(piper, self.rcfg, dw_f32=args.main_grad), device=local)
        piper.piper_set_chunk_overlap(self.ctx, 1 if getattr(args, "chunk_overlap", False) else 0)
        for kv in getattr(args, "opt", None) or []:  # measured variants: --opt T_SPLIT_K=0 ...
            name, val = kv.split("=")
            piper.piper_set_option(self.ctx, getattr(piper, "OPT_" + name), int(val))
        if args.main_grad:  # measured variant (reading c-17): fp32 dW, every step adds into it
            piper.piper_set_wgrad_accumulate(self.ctx, 1)
        self.b = piper.alloc_buffers(self.ctx)
        if args.main_grad:
            for n in ("dw_gate", "dw_up", "dw_down", "dws_gate", "dws_up", "dws_down"):
                if n in self.b:
                    self.b[n].zero_()
        self.b.update({n: piper.to_tensor(self.inp[n], self.dev) for n in INPUT_NAMES if n in self.inp})
        self.cargs = piper.chunk_args(self.b)
        self.stream = torch.cuda.current_stream()

    def step(self):
        self.piper.piper_run_chunk_fwd(self.ctx, self.cargs)
        self.piper.piper_run_chunk_bwd(self.ctx, self.cargs)

    def close(self):
        self.ctx.close()
        self.b.clear()
        self.inp.clear()
        self.torch.cuda.empty_cache()


def time_resident(w: Workload, steps, warmup, sampler, barrier, world, min_seconds=0.0):
    """W untimed steps, then exactly `steps` steps (more when `min_seconds` asks for a longer clock record) between a
    barrier + synchronize on both sides; CUDA events on the launching stream; max over ranks."""
    torch, piper = w.torch, w.piper
    for _ in range(warmup):
        w.step()
    barrier()
    if min_seconds > 0:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(w.stream)
        w.step()
        e1.record(w.stream)
        torch.cuda.synchronize()
        steps = max(steps, int(min_seconds * 1e3 / max(e0.elapsed_time(e1), 1e-3)) + 1)
    launches0 = piper.piper_kernel_launches(w.ctx)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.begin()
    ev0.record(w.stream)
    for _ in range(steps):
        w.step()
    ev1.record(w.stream)
    barrier()
    clocks = sampler.end()
    launches = piper.piper_kernel_launches(w.ctx) - launches0
    ms_per_step = max_over_ranks(ev0.elapsed_time(ev1), world, w.dev) / steps
    if clocks.get("samples") and ev0.elapsed_time(ev1) < 400.0:
        # NVML refreshes clock, throttle reasons and power every ~100 ms (power is an average over longer still): a timed
        # region of K = 20 steps (0.14 s) shows one or two stale readings.  The same loop therefore keeps running, untimed,
        # for 0.6 s more under the sampler, and that record is reported beside the timed region's own.
        n_more = int(600.0 / max(ms_per_step, 1e-3)) + 1
        sampler.begin()
        for _ in range(n_more):
            w.step()
        torch.cuda.synchronize()
        clocks["same_loop_continued_untimed"] = dict(sampler.end(), steps=n_more)
    return ms_per_step, clocks, int(launches), steps


def time_e2e(w: Workload, steps, warmup, barrier, world):
    """The same metric through the C-ABI with HOST buffers: every step copies logits / x / dY from pinned host memory to
    the device and y / dX / dz_sel back, inside the timed region."""
    torch, piper, b, cfg = w.torch, w.piper, w.b, w.cfg
    dev, stream, ctx = w.dev, w.stream, w.ctx
    host_in = {n: piper.to_tensor(w.inp[n], "cpu").pin_memory() for n in ("logits", "x", "dy")}
    out_names = ("y", "dx", "dz_sel")
    host_out = {n: torch.empty(b[n].shape, dtype=b[n].dtype).pin_memory() for n in out_names}
    h2d = sum(t.numel() * t.element_size() for t in host_in.values())
    d2h = sum(t.numel() * t.element_size() for t in host_out.values())

    # Software pipeline over three streams (what a training loop's data loader does): the inputs of step i+1 go up
    # and the results of step i-1 come down while step i computes; two sets of input / output device buffers, the
    # scratch and the weights are shared (the compute stream is serial).  Every step's copies are inside the timed
    # region.
    sets = [b, dict(b)]
    for n in ("logits", "x", "dy") + out_names:
        sets[1][n] = torch.empty_like(b[n])
    set_args = [w.cargs, piper.chunk_args(sets[1])]
    s_in, s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
    in_ready = [torch.cuda.Event() for _ in range(2)]   # logits and x are up (what the forward chunk reads)
    dy_ready = [torch.cuda.Event() for _ in range(2)]   # dY is up (first read by the backward chunk)
    fwd_done = [torch.cuda.Event() for _ in range(2)]   # y can go down while the backward chunk runs
    comp_done = [torch.cuda.Event() for _ in range(2)]
    out_done = [torch.cuda.Event() for _ in range(2)]

    def e2e_steps(n_steps):
        for i in range(n_steps):
            k = i & 1
            with torch.cuda.stream(s_in):
                if i >= 2:
                    s_in.wait_event(comp_done[k])  # step i-2 has consumed this input set
                for n in ("logits", "x"):
                    sets[k][n].copy_(host_in[n], non_blocking=True)
                in_ready[k].record(s_in)
                sets[k]["dy"].copy_(host_in["dy"], non_blocking=True)
                dy_ready[k].record(s_in)
            stream.wait_event(in_ready[k])
            if i >= 2:
                stream.wait_event(out_done[k])  # step i-2's results have left this output set
            piper.piper_run_chunk_fwd(ctx, set_args[k])
            fwd_done[k].record(stream)
            stream.wait_event(dy_ready[k])
            piper.piper_run_chunk_bwd(ctx, set_args[k])
            comp_done[k].record(stream)
            with torch.cuda.stream(s_out):
                s_out.wait_event(fwd_done[k])
                host_out["y"].copy_(sets[k]["y"], non_blocking=True)
                s_out.wait_event(comp_done[k])
                for n in ("dx", "dz_sel"):
                    host_out[n].copy_(sets[k][n], non_blocking=True)
                out_done[k].record(s_out)
        stream.wait_event(out_done[0])
        stream.wait_event(out_done[1])

    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2e_steps(min(warmup, 3))
    torch.cuda.synchronize(dev)
    barrier()
    w0 = time.perf_counter()
    ev0.record(stream)
    e2e_steps(steps)
    ev1.record(stream)
    barrier()
    wall_ms = (time.perf_counter() - w0) * 1e3
    e2e_ms = max_over_ranks(max(ev0.elapsed_time(ev1), wall_ms), world, dev) / steps
    return {"value": whole_job_tokens_per_s(cfg, world, e2e_ms), "unit": UNIT, "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms,
            "what": "every step: pinned host logits/x/dY -> device, piper_run_chunk_fwd + piper_run_chunk_bwd, y/dX/dz_sel "
                    "-> pinned host, as a 3-stream pipeline (copies of steps i+1 / i-1 overlap the compute of step i; dY goes up "
                    "behind x and y comes down while the backward chunk runs); "
                    "timed as max(CUDA events, host wall clock) over the whole pipeline"}


def time_tasks(w: Workload, n_prof):
    """Per-task device times (CUDA events on the launching stream between the tasks of full steps), each against its
    algorithmic work: `kernels`, and `roofline` for the dominant kernel."""
    import numpy as np
    torch, piper, cfg, rcfg, b = w.torch, w.piper, w.cfg, w.rcfg, w.b
    tasks = [t for t in piper.TASKS if cfg.I_shared or t not in ("F_SHARED", "B_SHARED")]
    order = ["F_ROUTE", "F_SCAN", "F_PACK", "F_SHARED", "F_GEMM1", "F_GEMM2", "F_COMBINE", "B_CGRAD", "B_DGRAD1",
             "B_DGRAD2", "B_WGRAD", "B_SHARED", "B_UNPACK", "B_ROUTE_BWD"]
    order = [t for t in order if t in tasks]
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(len(order) + 1)] for _ in range(n_prof)]
    for it in range(n_prof):
        evs[it][0].record(w.stream)
        for i, t in enumerate(order):
            piper.piper_run_task(w.ctx, t, w.cargs)
            evs[it][i + 1].record(w.stream)
    torch.cuda.synchronize()
    task_ms = {t: float(np.mean([evs[it][i].elapsed_time(evs[it][i + 1]) for it in range(n_prof)]))
               for i, t in enumerate(order)}

    A_padded = int(b["offsets"][rcfg.e_loc].item())  # rows the kernels process (segments padded to row_align)
    A = int(b["counts"].sum().item())                # rows the method defines: the algorithmic work
    t_touched = int((b["row_of"] >= 0).any(dim=1).sum().item())
    counts = b["counts"].cpu().numpy()
    peaks = measured_peaks()
    work = task_work(rcfg, A, t_touched)
    stored = stored_ncu()
    gemm_bytes = gemm_hbm_bytes(rcfg, A)
    kernels = {}
    for t in order:
        bound, amount = work[t]
        sec = task_ms[t] * 1e-3
        if bound == "tensor":
            ach, peak, unit = amount / sec / 1e12, peaks["tf_sustained"], "TFLOP/s"
        else:
            ach, peak, unit = amount / sec / 1e9, peaks["hbm"], "GB/s"
        kernels[t] = {"ms": round(task_ms[t], 4), "bound": bound, "achieved": round(ach, 2), "unit": unit,
                      "frac": round(ach / peak, 4)}
        if bound == "tensor" and t in gemm_bytes:  # the other roof of a GEMM task: weights, dW and row buffers moved once
            gbs = gemm_bytes[t] / sec / 1e9
            kernels[t]["hbm_gbs_at_least"] = round(gbs, 1)
            kernels[t]["hbm_frac"] = round(gbs / peaks["hbm"], 4)
        us = stored.get("ncu_us", {}).get(cfg.name, {}).get(t)
        if us:  # NOT measured in this run: the same algorithmic bytes over the kernel's own duration under ncu
            kernels[t]["stored_ncu"] = {"us": us, "frac": round(amount / (us * 1e-6) / 1e9 / peak, 4),
                                        "stored_from": stored.get("_ncu_us_source", STORED)}
    gemm_tasks = [t for t in order if work[t][0] == "tensor"]
    gemm_ms = sum(task_ms[t] for t in gemm_tasks)
    gemm_flop = sum(work[t][1] for t in gemm_tasks)
    dom = "F_GEMM1"  # one launch per task: the fused gate/up GEMM + SwiGLU kernel (largest single-kernel share)
    impl = "tcgen05" if (cfg.dtype == 1 and piper.piper_gemm_path(w.ctx) == 1) else "fp32-alu"
    traffic = stored.get(cfg.name, {}).get(dom)
    roofline = {"bound": "tensor", "kernel": f"{dom} ({impl} grouped GEMM gate|up + SwiGLU epilogue, 1 launch/step)",
                "achieved": kernels[dom]["achieved"], "peak": peaks["tf_sustained"], "unit": "TFLOP/s",
                "frac": kernels[dom]["frac"], "frac_of_burst_peak": round(kernels[dom]["achieved"] / peaks["tf_burst"], 4),
                "frac_of_nominal_2250": round(kernels[dom]["achieved"] / 2250.0, 4),
                "traffic": traffic,
                "traffic_stored_from": (stored.get("_source", STORED) + " -- a committed ncu capture, NOT measured in this run")
                if traffic else None,
                "peak_kind": f"bf16_tflops_sustained of {peaks['kind']} (kernel timed inside a long step); burst {peaks['tf_burst']}",
                "flop_per_launch": work[dom][1], "ms_per_launch": task_ms[dom],
                "all_gemm": {"tflops": round(gemm_flop / (gemm_ms * 1e-3) / 1e12, 2),
                             "frac": round(gemm_flop / (gemm_ms * 1e-3) / 1e12 / peaks["tf_sustained"], 4),
                             "frac_of_burst_peak": round(gemm_flop / (gemm_ms * 1e-3) / 1e12 / peaks["tf_burst"], 4),
                             "frac_of_nominal_2250": round(gemm_flop / (gemm_ms * 1e-3) / 1e12 / 2250.0, 4),
                             "share_of_step": round(gemm_ms / sum(task_ms.values()), 4)}}
    shape = {"A_rows": A, "A_rows_padded": A_padded, "tokens_touched": t_touched,
             "rows_per_expert_min_max": [int(counts.min()), int(counts.max())]}
    return kernels, roofline, shape, impl, task_ms


def tc_counters(w: Workload):
    """Debug wait-cycle counters of the tcgen05 kernels (PIPER_OPT_TC_PROFILE), one row per GEMM launch of each task:
    cycles of the MMA-issuing warp's loop and the shares it spent waiting for operands / for a free accumulator, the
    weight producer's share waiting for a free stage, the epilogue's shares waiting for an accumulator / a staging
    buffer, tiles per cluster.  Mean over the leader CTAs."""
    import ctypes
    import numpy as np
    torch, piper = w.torch, w.piper
    piper.piper_set_option(w.ctx, piper.OPT_TC_PROFILE, 1)
    ptr = piper.lib().piper_debug_tc_counters(w.ctx._h)
    n_words = 16 * 160 * 8
    rt = ctypes.CDLL("libcudart.so")

    def read():
        t = torch.empty(n_words, dtype=torch.int64, device=w.dev)
        torch.cuda.synchronize()
        rt.cudaMemcpy(ctypes.c_void_p(t.data_ptr()), ctypes.c_void_p(ptr), ctypes.c_size_t(n_words * 8), 3)
        return t.cpu().numpy().reshape(16, 160, 8)

    tasks = ["F_GEMM1", "F_GEMM2", "B_DGRAD1", "B_DGRAD2", "B_WGRAD"] + (["F_SHARED", "B_SHARED"] if w.cfg.I_shared else [])
    rows = []
    for t in tasks:
        before = read()
        piper.piper_run_task(w.ctx, t, w.cargs)
        after = read()
        for s in range(16):
            if np.array_equal(before[s], after[s]):
                continue
            q = after[s]
            lead, epi = q[:, 2] > 0, q[:, 5] > 0
            if not lead.any():
                continue
            loop = q[lead, 2].astype(float)
            rows.append({"task": t, "launch_slot": s, "clusters": int(lead.sum()), "mma_loop_cycles": float(loop.mean()),
                         "mma_wait_operands": float((q[lead, 0] / loop).mean()),
                         "mma_wait_accumulator": float((q[lead, 1] / loop).mean()),
                         "producer_wait_stage": float((q[lead, 3] / loop).mean()),
                         "epilogue_wait_accumulator": float((q[epi, 4] / np.maximum(q[epi, 5], 1)).mean()),
                         "epilogue_wait_staging": float((q[epi, 7] / np.maximum(q[epi, 5], 1)).mean()),
                         "tiles_per_cluster": float(q[lead, 6].mean()), "loop_max_over_min": float(loop.max() / loop.min())})
    piper.piper_set_option(w.ctx, piper.OPT_TC_PROFILE, 0)
    return rows


def run_piper(args, cfg, sampler, rank, world, local, barrier, e2e=True, min_seconds=0.0):
    """The bench line of one config (resident value, optional e2e, per-task times)."""
    from inputs import configs
    w = Workload(args, cfg, rank, local)
    ms_per_step, clocks, launches, steps = time_resident(w, args.steps, args.warmup, sampler, barrier, world, min_seconds)
    value = whole_job_tokens_per_s(cfg, world, ms_per_step)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16" if cfg.dtype == 1 else "f32", "data": "synthetic"}
    if e2e:
        line["e2e"] = time_e2e(w, args.steps, args.warmup, barrier, world)
    kernels, roofline, shape, impl, _ = time_tasks(w, max(3, min(args.steps, 10)))
    shape["parallelism"] = f"replicas x{world} (one microbatch per GPU)"
    line.update({"config": workload_config(cfg, extra=shape),
                 "tflops": configs.flops_fwd_bwd(w.rcfg, shape["A_rows"]) / (ms_per_step * 1e-3) / 1e12,
                 "clocks": clocks, "gpu_launches": launches, "roofline": roofline, "kernels": kernels, "gemm_impl": impl})
    if args.main_grad:
        line["config"]["dw"] = "fp32, accumulated across steps (accumulate = 1)"
    if getattr(args, "tc_counters", False) and impl == "tcgen05":
        line["tc_counters"] = tc_counters(w)
    return line, w


def time_torch_eager(w: Workload, steps=5, warmup=2):
    """Context, not the product: the same fwd+bwd chunk written with stock PyTorch ops (top-k, gather, a loop of torch.mm
    over the experts, index_add, autograd), which is what the paper's Chunks execute ("stock PyTorch
    ops"), on the same device, inputs and dtype.  No kernel or entry point of this library is on that path."""
    import torch
    import torch.nn.functional as F
    from inputs import configs
    cfg, b = w.rcfg, w.b
    T, k, lo, El = cfg.T, cfg.k, cfg.e_lo, cfg.e_loc
    names = ["w_gate", "w_up", "w_down"] + (["ws_gate", "ws_up", "ws_down"] if cfg.I_shared else [])
    params = {n: b[n].detach().clone().requires_grad_(True) for n in names}
    x = b["x"].detach().clone().requires_grad_(True)
    logits = b["logits"].detach().clone().requires_grad_(True)
    dy = b["dy"]

    def step():
        for t in [x, logits] + list(params.values()):
            t.grad = None
        topv, topi = logits.topk(k, dim=1)
        if cfg.gate_mode == configs.GATE_SOFTMAX_RENORM:
            gates = torch.softmax(topv, dim=1)
        elif cfg.gate_mode == configs.GATE_SIGMOID_RENORM:
            sg = torch.sigmoid(topv)
            gates = sg / sg.sum(dim=1, keepdim=True)
        else:
            gates = torch.softmax(logits, dim=1).gather(1, topi)
        flat_e, flat_g = topi.reshape(-1), gates.reshape(-1)
        flat_t = torch.arange(T, device=x.device).repeat_interleave(k)
        local = (flat_e >= lo) & (flat_e < lo + El)
        e_l, t_l, g_l = flat_e[local] - lo, flat_t[local], flat_g[local]
        order = torch.argsort(e_l, stable=True)
        tok, gate = t_l[order], g_l[order]
        counts = torch.bincount(e_l, minlength=El).tolist()  # the host needs the split sizes: a sync, as in eager MoE code
        xp = x[tok]
        outs, start = [], 0
        for e, n in enumerate(counts):
            seg = xp[start:start + n]
            h = F.silu(seg @ params["w_gate"][e]) * (seg @ params["w_up"][e])
            outs.append(h @ params["w_down"][e])
            start += n
        o = torch.cat(outs) * gate.to(x.dtype)[:, None]
        y = torch.zeros_like(x).index_add_(0, tok, o)
        if cfg.I_shared:
            y = y + (F.silu(x @ params["ws_gate"][0]) * (x @ params["ws_up"][0])) @ params["ws_down"][0]
        y.backward(dy)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    return {"value": T / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": steps,
            "what": "the same chunk (route, permute, expert FFNs, combine, backward through autograd) in stock PyTorch eager ops "
                    "on this GPU: cuBLAS GEMMs per expert in a Python loop, bf16, fp32 routing; context only (PAPER.md:137, 326)"}


def gemm_hbm_bytes(cfg, A: int):
    """Bytes the GEMM tasks must move at least once (weights read once per GEMM, dW written once, row buffers read /
    written once per use): {task: bytes}."""
    b, d, I, Is, T, E = 2 if cfg.dtype == 1 else 4, cfg.d, cfg.I, cfg.I_shared, cfg.T, cfg.e_loc

    def ffn(rows, n_e, inter):
        w = n_e * d * inter * b
        return {"gemm1": 2 * w + rows * d * b + 3 * rows * inter * b, "gemm2": w + rows * inter * b + rows * d * b,
                "dgrad1": w + rows * d * b + 4 * rows * inter * b, "dgrad2": 2 * w + 2 * rows * inter * b + rows * d * b,
                "wgrad": 2 * rows * d * b + 3 * rows * inter * b + 3 * w}
    r = ffn(A, E, I)
    out = {"F_GEMM1": r["gemm1"], "F_GEMM2": r["gemm2"], "B_DGRAD1": r["dgrad1"], "B_DGRAD2": r["dgrad2"],
           "B_WGRAD": r["wgrad"]}
    if Is:
        sh = ffn(T, 1, Is)
        out["F_SHARED"] = sh["gemm1"] + sh["gemm2"]
        out["B_SHARED"] = sh["dgrad1"] + sh["dgrad2"] + sh["wgrad"]
    return out


def overlapped_block(piper, ctx, cfg, args_a, args_b, task_ms, timed, timed_beside, n_sm):
    """N3 (Fig. 3b): the whole overlapped block - attention forward of microbatch A in front of its MoE
    chunk, attention backward of microbatch B behind its MoE chunk - with the attention as CALLER tasks of the pair
    (piper_pair_set_caller_task).  The attention here is torch's fused SDPA (library code, causal, heads of 128, sequences
    of up to 4096 tokens; its output is not wired into x: a timing stand-in for the caller's own kernels)."""
    import torch
    H, S = max(1, cfg.d // 128), min(cfg.T, 4096)
    B = max(1, cfg.T // S)
    dev = torch.device("cuda", torch.cuda.current_device())
    q, k, v, dout = (torch.randn(B, H, S, 128, device=dev, dtype=torch.bfloat16) for _ in range(4))
    ops = torch.ops.aten
    fwd = ops._scaled_dot_product_flash_attention(q, k, v, 0.0, True, False)
    o, lse, cq, ck, mq, mk, seed, off = fwd[:8]

    def attn_fwd(stream_ptr=None, sms=0):
        with torch.cuda.stream(torch.cuda.ExternalStream(stream_ptr) if stream_ptr else torch.cuda.current_stream()):
            ops._scaled_dot_product_flash_attention(q, k, v, 0.0, True, False)

    def attn_bwd(stream_ptr=None, sms=0):
        with torch.cuda.stream(torch.cuda.ExternalStream(stream_ptr) if stream_ptr else torch.cuda.current_stream()):
            ops._scaled_dot_product_flash_attention_backward(dout, q, k, v, o, lse, cq, ck, mq, mk, 0.0, True, seed, off)

    t_af, t_ab = timed(attn_fwd), timed(attn_bwd)
    t_f = timed(lambda: piper.piper_run_chunk_fwd(ctx, args_a))
    t_b = timed(lambda: piper.piper_run_chunk_bwd(ctx, args_b))
    def serial_block():
        attn_fwd(), piper.piper_run_chunk_fwd(ctx, args_a), piper.piper_run_chunk_bwd(ctx, args_b), attn_bwd()

    serial = timed(serial_block)
    res = {"attention": f"torch SDPA (flash), causal, batch {B} x {H} heads x {S} tokens x 128, bf16", "attn_fwd_ms": t_af,
           "attn_bwd_ms": t_ab, "chunk_fwd_ms": t_f, "chunk_bwd_ms": t_b, "serial_ms": serial, "variants": {}}
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_F_PRE, attn_fwd, est_ms=t_af, side=1)
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_B_POST, attn_bwd, est_ms=t_ab, side=1)
    for name, order, part, splits in (("list_order_exclusive", piper.ORDER_LIST, piper.PART_EXCLUSIVE, [(132, 16), (116, 32)]),
                                      ("profile_order_shared_sms", piper.ORDER_PROFILE, piper.PART_SHARED, [(n_sm, 32)]),
                                      ("chunk_streams", piper.ORDER_LIST, piper.PART_CHUNK_STREAMS, [(n_sm, 16)])):
        piper.piper_set_pair_policy(ctx, order, part, task_ms)
        for sg, sc in splits:
            piper.piper_pair_prepare(ctx, sg, sc)
            t_p, t_s, ratio = timed_beside(lambda: piper.piper_run_chunk_pair(ctx, args_a, args_b, sg, sc), base=serial_block)
            res["variants"][f"{name} {sg}:{sc}"] = {"pair_ms": t_p, "serial_ms_beside": t_s, "ratio_vs_serial": ratio,
                                                    "order": piper.piper_pair_order(ctx, sg, sc)}
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_F_PRE, None)
    piper.piper_pair_set_caller_task(ctx, piper.SLOT_B_POST, None)
    piper.piper_set_pair_policy(ctx, piper.ORDER_LIST, piper.PART_EXCLUSIVE)
    return res


def run_pair(piper, ctx, cfg, b_a, inp_a, splits, iters, sampler=None, attn=False):
    """Step P on this context's layer shape: forward chunk of microbatch A (the bench inputs) co-scheduled
    with the backward chunk of microbatch B (seed + 1, own weights: reading c-20) versus the same two
    chunks back to back on one stream with all SMs."""
    import torch
    from inputs import configs
    cfg_b = dataclasses.replace(cfg, seed=cfg.seed + 1)
    inp_b = configs.make_inputs(cfg_b)
    dev = b_a["x"].device
    b_b = piper.alloc_buffers(ctx)
    b_b.update({n: piper.to_tensor(inp_b[n], dev) for n in INPUT_NAMES if n in inp_b})
    args_a, args_b = piper.chunk_args(b_a), piper.chunk_args(b_b)
    piper.piper_run_chunk_fwd(ctx, args_b)  # untimed producer of B's saved activations
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if sampler is not None:
        sampler.begin()

    def timed(fn, repeats=3):
        """Median over `repeats` timings of `iters` back-to-back calls (the pair's time moves by several % from one
        timing to the next: which SMs a partition gets and how the two streams interleave is not ours to fix)."""
        for _ in range(2):
            fn()
        ts = []
        for _ in range(repeats):
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(iters):
                fn()
            e1.record(stream)
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) / iters)
        return sorted(ts)[len(ts) // 2]

    # the serial baseline: every task of both chunks on one stream, all SMs
    piper.piper_set_chunk_overlap(ctx, 0)
    t_f = timed(lambda: piper.piper_run_chunk_fwd(ctx, args_a))
    t_b = timed(lambda: piper.piper_run_chunk_bwd(ctx, args_b))
    out = {"fwd_ms": t_f, "bwd_ms": t_b, "serial_ms": t_f + t_b, "tokens_per_pair": 2 * cfg.T,
           "tokens_per_s_serial": 2 * cfg.T / ((t_f + t_b) * 1e-3), "splits": {}, "variants": {}}

    def serial_fn():
        piper.piper_run_chunk_fwd(ctx, args_a)
        piper.piper_run_chunk_bwd(ctx, args_b)

    serial_beside = []

    def timed_beside_serial(fn, repeats=8, base=None):
        """The pair and the serial chunks (fwd(A) then bwd(B) on one stream, all SMs) timed alternately, a few calls
        each, the order swapped every repeat: under the power cap the same kernels slow down by several % while a run
        warms the board, so a baseline taken once at the start would flatter itself.  Medians of the pair's time, of the
        serial time beside it and of their ratio."""
        base_fn = base or serial_fn
        for _ in range(2):
            fn()
        base_fn()
        tp, ts, ratio = [], [], []
        n_in = max(3, iters // 2)
        for r in range(repeats):
            pair_first = r % 2 == 1
            t = {}
            for which in ((0, 1) if pair_first else (1, 0)):
                torch.cuda.synchronize()
                e0.record(stream)
                for _ in range(n_in):
                    (fn if which == 0 else base_fn)()
                e1.record(stream)
                torch.cuda.synchronize()
                t[which] = e0.elapsed_time(e1) / n_in
            tp.append(t[0]), ts.append(t[1]), ratio.append(t[0] / t[1])
        if base is None:
            serial_beside.extend(ts)
        med = lambda v: sorted(v)[len(v) // 2]
        return med(tp), med(ts), med(ratio)

    def sweep(split_list):
        res = {}
        for sg, sc in split_list:
            piper.piper_pair_prepare(ctx, sg, sc)  # partitions / streams / plan are created outside the timed calls
            t_p, t_s, ratio = timed_beside_serial(lambda: piper.piper_run_chunk_pair(ctx, args_a, args_b, sg, sc))
            res[f"{sg}:{sc}"] = {"pair_ms": t_p, "serial_ms_beside": t_s, "ratio_vs_serial": ratio,
                                 "order": piper.piper_pair_order(ctx, sg, sc)}
        return res

    # the contract's sweep: Piper's list scheduling on disjoint SM partitions
    piper.piper_set_pair_policy(ctx, piper.ORDER_LIST, piper.PART_EXCLUSIVE)
    out["splits"] = sweep(splits)
    out["partition_mode"] = {1: "green contexts", 2: "bounded grids on plain streams", 3: "one stream per chunk"}.get(
        piper.piper_pair_partition_mode(ctx), "?")
    # measured variants: profile-guided order from per-task times taken here, and SM sharing
    # (the paper leaves SM allocation to the GPU) where the GEMM grids keep every SM
    tasks = [t for t in piper.TASKS]
    task_ms = []
    for t in tasks:
        if t in ("F_SHARED", "B_SHARED") and not cfg.I_shared:
            task_ms.append(0.0)
            continue
        a = args_a if t.startswith("F_") else args_b
        task_ms.append(timed(lambda: piper.piper_run_task(ctx, t, a)))
    out["task_ms"] = dict(zip(tasks, task_ms))
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    piper.piper_set_pair_policy(ctx, piper.ORDER_PROFILE, piper.PART_EXCLUSIVE, task_ms)
    out["variants"]["profile_order_exclusive"] = sweep(splits)
    shared_splits = [(n_sm, 16), (n_sm, 32), (n_sm, 48)]
    piper.piper_set_pair_policy(ctx, piper.ORDER_PROFILE, piper.PART_SHARED, task_ms)
    out["variants"]["profile_order_shared_sms"] = sweep(shared_splits)
    # the paper's own setting: one stream per chunk, SM allocation left to the GPU
    piper.piper_set_pair_policy(ctx, piper.ORDER_LIST, piper.PART_CHUNK_STREAMS, task_ms)
    out["variants"]["chunk_streams_gpu_allocates_sms"] = sweep([(n_sm, 16)])
    piper.piper_set_pair_policy(ctx, piper.ORDER_LIST, piper.PART_EXCLUSIVE)
    if attn:
        out["overlapped_block"] = overlapped_block(piper, ctx, cfg, args_a, args_b, task_ms, timed, timed_beside_serial, n_sm)
    best = min(((v["ratio_vs_serial"], name, k) for name, d in
                [("list_order_exclusive", out["splits"])] + list(out["variants"].items()) for k, v in d.items()))
    best_ms = dict([("list_order_exclusive", out["splits"])] + list(out["variants"].items()))[best[1]][best[2]]["pair_ms"]
    out["best"] = {"ratio_vs_serial": best[0], "variant": best[1], "split": best[2], "pair_ms": best_ms,
                   "tokens_per_s": 2 * cfg.T / (best_ms * 1e-3)}
    out["serial_back_to_back_ms"] = sorted(serial_beside)[len(serial_beside) // 2]
    out["ratio_is"] = ("pair_ms / serial_ms_beside: the serial chunks (fwd(A) then bwd(B) on one stream, all SMs) re-timed "
                       "beside every pair timing, alternating; serial_ms = fwd and bwd timed separately at the start")
    # What the pair can reach on this workload: the floors of the two roofs and of "every row
    # mover hidden under GEMMs that keep their serial speed", each as a ratio to the measured serial time.
    peaks = measured_peaks()
    A_a, A_b = int(b_a["counts"].sum().item()), int(b_b["counts"].sum().item())
    tt_a = int((b_a["row_of"] >= 0).any(dim=1).sum().item())
    tt_b = int((b_b["row_of"] >= 0).any(dim=1).sum().item())
    wa, wb = task_work(cfg, A_a, tt_a), task_work(cfg_b, A_b, tt_b)
    ga, gb = gemm_hbm_bytes(cfg, A_a), gemm_hbm_bytes(cfg_b, A_b)
    flop = sum(v for t, (k_, v) in wa.items() if k_ == "tensor" and t.startswith("F_")) + \
        sum(v for t, (k_, v) in wb.items() if k_ == "tensor" and t.startswith("B_"))
    hbm = sum(v for t, (k_, v) in wa.items() if k_ == "hbm" and t.startswith("F_")) + \
        sum(v for t, (k_, v) in wb.items() if k_ == "hbm" and t.startswith("B_")) + \
        sum(v for t, v in ga.items() if t.startswith("F_")) + sum(v for t, v in gb.items() if t.startswith("B_"))
    gemm_ms = sum(ms for t, ms in out["task_ms"].items() if (wa.get(t) or ("", 0))[0] == "tensor")
    mover_ms = sum(ms for t, ms in out["task_ms"].items() if (wa.get(t) or ("", 0))[0] == "hbm")
    serial = t_f + t_b
    out["bound"] = {"serial_ms": serial, "gemm_tasks_ms": gemm_ms, "row_mover_and_routing_tasks_ms": mover_ms,
                    "ratio_if_every_mover_is_hidden": gemm_ms / serial,
                    "flop": flop, "tensor_floor_ms": flop / (peaks["tf_sustained"] * 1e9),
                    "tensor_floor_ratio": flop / (peaks["tf_sustained"] * 1e9) / serial,
                    "hbm_bytes": hbm, "hbm_floor_ms": hbm / (peaks["hbm"] * 1e6),
                    "hbm_floor_ratio": hbm / (peaks["hbm"] * 1e6) / serial,
                    "what": "tensor floor = GEMM FLOP of fwd(A) + bwd(B) / bf16_tflops_sustained; hbm floor = bytes the row movers "
                            "and the GEMMs must move once (weights, dW, row buffers) / hbm_gbs; 'every mover hidden' = the GEMM "
                            "tasks alone at their measured whole-device speed.  The 0.8 target lies below the last one."}
    if sampler is not None:
        out["clocks"] = sampler.end()
    return out


def run_ab(w: Workload, spec: str, blocks: int, per: int, tasks=None):
    """Paired A/B of one kernel-variant switch inside one process (`--ab NAME=v0,v1,...`): blocks of `per` timed steps
    alternate between the values (order reversed every block, one untimed step after each switch), so the drift of the
    power-capped clocks while the board warms hits every value alike.  Separate bench runs of the same library differ by
    several % on one box and cannot resolve a 1-2 % change (DESIGN.md findings 30, 31).  With `tasks` (--ab-tasks, names of
    the pair DAG's tasks) a timed unit is those tasks run once each through piper_run_task instead of a whole step."""
    import statistics
    torch, piper = w.torch, w.piper
    name, vals = spec.split("=")
    vals = [int(v) for v in vals.split(",")]
    if name == "CHUNK_OVERLAP":  # not a piper_set_option switch: piper_set_chunk_overlap (row movers on the side stream)
        def set_value(v):
            piper.piper_set_chunk_overlap(w.ctx, v)
    else:
        def set_value(v):
            piper.piper_set_option(w.ctx, getattr(piper, "OPT_" + name), v)
    def unit():
        if tasks:
            for t in tasks:
                piper.piper_run_task(w.ctx, t, w.cargs)
        else:
            w.step()

    for _ in range(10):
        w.step()
    torch.cuda.synchronize()
    times = {v: [] for v in vals}
    for b in range(blocks):
        for v in (vals if b % 2 == 0 else vals[::-1]):
            set_value(v)
            unit()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(w.stream)
            for _ in range(per):
                unit()
            e1.record(w.stream)
            torch.cuda.synchronize()
            times[v].append(e0.elapsed_time(e1) / per)
    base = statistics.mean(times[vals[0]])
    return {"option": name, "blocks": blocks, "steps_per_block": per, "workload": w.cfg.name, "unit": tasks or "step",
            "values": {str(v): {"mean_ms": statistics.mean(t), "median_ms": statistics.median(t), "min_ms": min(t),
                                "vs_first_pct": 100 * (statistics.mean(t) / base - 1)} for v, t in times.items()}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C2")
    ap.add_argument("--impl", default="piper", choices=["piper", "reference"])
    ap.add_argument("--row-align", type=int, default=None, help="override the config's row_align")
    ap.add_argument("--oracle-tokens", type=int, default=0, help="tokens of the CPU-oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true",
                    help="only the headline workload: skip the C3 / C4 / C5-pair blocks of the default run")
    ap.add_argument("--tc-counters", action="store_true",
                    help="add the tcgen05 kernels' debug wait-cycle counters per GEMM task (PIPER_OPT_TC_PROFILE) to the line")
    ap.add_argument("--opt", action="append", help="kernel-variant switch NAME=VALUE (piper_set_option, PIPER_OPT_<NAME>)")
    ap.add_argument("--uniform-rows", type=int, default=0,
                    help="microbenchmark: C3's routed layer shape with exactly this many rows in each of 32 experts "
                         "(overrides --config; use with --no-cpu-baseline)")
    ap.add_argument("--chunk-overlap", action="store_true",
                    help="measured variant: piper_set_chunk_overlap(1), the chunks' row movers on the library's side "
                         "stream beside the shared expert's GEMMs / the routed wgrad (default: one stream; measured "
                         "neutral, C2 6.67 -> 6.82 ms, C3 4.22 -> 4.23 ms: the GEMM beside them slows by what they hide)")
    ap.add_argument("--pair", action="store_true", help="also time step P (chunk pair vs serial) on this shape")
    ap.add_argument("--attn", action="store_true",
                    help="with --pair: also time the whole overlapped block (N3), attention forward / backward (torch SDPA) as "
                         "caller tasks of the pair")
    ap.add_argument("--ab", default=None,
                    help="paired A/B of a kernel-variant switch, NAME=v0,v1,...: alternates the values inside one process "
                         "(--ab-blocks blocks of --ab-steps timed steps per value) and prints only that comparison")
    ap.add_argument("--ab-blocks", type=int, default=30)
    ap.add_argument("--ab-steps", type=int, default=5)
    ap.add_argument("--ab-tasks", default=None, help="with --ab: time these tasks (comma-separated, e.g. F_COMBINE,B_UNPACK) instead of whole steps")
    ap.add_argument("--main-grad", action="store_true",
                    help="measured variant: fp32 dW accumulated across steps (dw_dtype F32, accumulate = 1)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "piper" else args.warmup

    import __graft_entry__ as ge
    from inputs import configs
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        ge.build()
    default_run = args.config == "C2" and not args.uniform_rows and not args.pair and not args.main_grad and not args.opt
    if args.config == "C5":  # configs[4]: the C3-shaped chunk pair, microbatch seeds 4 (forward) and 5 (backward)
        args.config, args.pair = "C5a", True

    def bench_cfg(name):
        c = configs.BY_NAME[name]
        return dataclasses.replace(c, row_align=args.row_align or 128) if c.dtype == configs.DT_BF16 else c

    cfg = dataclasses.replace(configs.uniform_config(args.uniform_rows), row_align=args.row_align or 128) \
        if args.uniform_rows else bench_cfg(args.config)
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    import paper_2606_11169_b200 as piper
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the piper library has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.ab:
        w = Workload(args, cfg, rank, local)
        print(json.dumps({"ab": run_ab(w, args.ab, args.ab_blocks, args.ab_steps,
                                       args.ab_tasks.split(",") if args.ab_tasks else None)}), flush=True)
        w.close()
        return
    sampler = ClockSampler(local)
    sampler.start()  # before any warm-up; it records only inside the timed regions
    line, w = run_piper(args, cfg, sampler, rank, world, local, barrier)
    iters = max(3, min(args.steps, 10))
    contract_splits = [(132, 16), (124, 24), (116, 32), (100, 48)]
    if args.pair and world == 1:
        line["pair"] = run_pair(piper, w.ctx, w.rcfg, w.b, w.inp, contract_splits, iters, sampler, attn=args.attn)
    if rank == 0 and world == 1 and not args.no_extra and cfg.dtype == configs.DT_BF16:
        try:
            line["torch_eager"] = time_torch_eager(w)
        except RuntimeError as e:  # e.g. out of memory beside the library's buffers: the context line is optional
            line["torch_eager"] = {"unavailable": str(e).splitlines()[0][:200]}
        torch.cuda.empty_cache()
    w.close()
    if default_run and world == 1 and not args.no_extra:
        # the north star's whole report in one line: the other single-GPU workloads of BASELINE.json, each with its own
        # clock record over a timed region of >= 0.5 s, and the chunk pair of configs[4]
        line["configs"] = {}
        for name in ("C3", "C4"):
            sub, w2 = run_piper(args, bench_cfg(name), sampler, rank, world, local, barrier, e2e=False, min_seconds=0.5)
            w2.close()
            keep = ("value", "unit", "ms_per_step", "steps", "tflops", "clocks", "gpu_launches", "roofline", "kernels", "config")
            line["configs"][name] = {k_: sub[k_] for k_ in keep}
        w5 = Workload(args, bench_cfg("C5a"), rank, local)
        w5.step()
        line["configs"]["C5_pair"] = run_pair(piper, w5.ctx, w5.rcfg, w5.b, w5.inp, contract_splits, iters, sampler)
        line["configs"]["C5_pair"]["config"] = workload_config(w5.cfg, extra={"microbatch_b_seed": w5.rcfg.seed + 1})
        w5.close()
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        tokens = args.oracle_tokens or 8
        sec, cores, _ = time_oracle(cfg, tokens, 1, 0)
        line["cpu_baseline"] = {"value": tokens / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"CPU oracle fwd+bwd, one pass over the first {tokens} tokens of {cfg.name} "
                                          f"(same d/E/k/I, weights, seed), {sec:.1f} s"}
    sampler.stop_flag = True
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
