#!/usr/bin/env python
"""bench.py -- CARVE layer-operator fwd+bwd throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config cfg1]

A "step" is one pass of the whole hot path over one batch of synthetic input: carve_fwd (saving
for backward) + carve_bwd through the C ABI (paper_2606_27229_b200/csrc/libcarve.so).  The default
workload is BASELINE.json configs[1] (B=8,H=16,T=4096,L=64,dk=dv=128,r=16, bf16 tokens, fp32 state),
the shape the metric is quoted on.  Prints ONE JSON line (rank 0):
  value     tokens/s, inputs resident in HBM, CUDA events on the launching stream, max over ranks
  e2e       same metric through carve_fwd_bwd_host: pinned HOST buffers, H2D/D2H copies inside the timing
  roofline  dominant kernel: algorithmic bytes per launch / its event-timed duration vs measured HBM peak
  cpu_baseline  the fp64 oracle, as it stands, on the host cores, on a bounded sample of the same workload
With N > 1 (torchrun) every rank runs the same per-GPU workload on its own batch shard (weak scaling:
chains are independent); the only exchange is one NCCL all-reduce of the shared weight
gradients (tens of KB) per step.  `--impl reference` times the oracle (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_27229_b200 import synth  # noqa: E402

METRIC = "CARVE layer fwd+bwd tokens/sec"
PAPER_CONTEXT = ("paper: full-model training throughput 95.52K vs 94.21K tok/s, 1xH100, bf16, Table 3 "
                 "(captioned 125M/T=1024; not an operator timing, not comparable)")


def get_cfg(name: str) -> synth.Config:
    table = {"cfg0": synth.CFG0, "cfg1": synth.CFG1, "cfg3": synth.CFG3, "cfg4": synth.CFG4}
    table.update({f"cfg2_L{L}": c for L, c in synth.CFG2.items()})
    return table[name]


# ---- algorithmic bytes / flops -------------------------------
def algorithmic(cfg: synth.Config, scalar_write: bool = False):
    e = 2 if cfg.dtype == "bf16" else 4
    dk, dv, r, L = cfg.dk, cfg.dv, cfg.r, cfg.L
    tokh = cfg.B * cfg.T * cfg.H
    chains = cfg.B * cfg.H
    n_in = 2 * dk + dv + dk + dk + (0 if scalar_write else dv) + 1      # scalar-write variant: no wx in, no dwx out
    fwd_b = tokh * (e * n_in + e * dv) + chains * 4 * dv * dk * 2
    bwd_b = tokh * (e * n_in + e * dv + e * n_in) + chains * 4 * dv * dk * 2
    fwd_f = (4 * r * dv * dk + 4 * L * r * dk + 2 * L * r * (dk + dv) + L * (L - 1) * dk + L * (L + 1) * dk +
             L * (L - 1) * dv + 3 * 2 * L * dk * dv + L * (L + 1) * dv)
    fwd_f *= chains * (cfg.T // L)
    return dict(fwd_bytes=fwd_b, bwd_bytes=0 if cfg.fwd_only else bwd_b, fwd_flops=fwd_f,
                bwd_flops=0 if cfg.fwd_only else 2 * fwd_f)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d["bf16_tflops"]),
                    bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


class ClockSampler:
    """Samples SM clocks and throttle reasons every ~2 ms (NVML) from before the warm-up until after the timed loop;
    `mark()` brackets the timed region so that the summary is taken from the samples that fall inside it."""
    NAMES = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index: int):
        self.index, self.rows, self.stop_flag, self.thr, self.marks, self.err = index, [], False, None, [], None
        self.max_sm = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_sm = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # noqa: BLE001
            self.err = f"nvml unavailable: {e}"
            return

        def loop():
            while not self.stop_flag:
                try:
                    sm = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                    rs = int(pynvml.nvmlDeviceGetCurrentClocksEventReasons(h))
                    self.rows.append((time.perf_counter(), sm, rs))
                except Exception:  # noqa: BLE001
                    pass
                time.sleep(0.002)
        self.thr = threading.Thread(target=loop, daemon=True)
        self.thr.start()

    def mark(self):
        self.marks.append(time.perf_counter())

    def stop(self) -> dict:
        if self.thr is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": [self.err or "sampler not started"]}
        self.stop_flag = True
        self.thr.join(timeout=2)
        lo, hi = (self.marks[0], self.marks[1]) if len(self.marks) >= 2 else (0.0, float("inf"))
        inside = [r for r in self.rows if lo <= r[0] <= hi] or self.rows
        sm = [r[1] for r in inside]
        reasons = sorted(n for n, bit in self.NAMES.items() if any(r[2] & bit for r in inside))
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": self.max_sm, "samples": len(sm),
                "samples_total": len(self.rows), "reasons": reasons}


# ---- CPU oracle leg ------------------------------------------------------------------------------
def oracle_sample(cfg: synth.Config, x: dict, ct: dict, nchains: int):
    """The first `nchains` (batch, head) chains of the workload, full T, as a B'=n, H'=1 problem."""
    chains = [(i // cfg.H, i % cfg.H) for i in range(min(nchains, cfg.B * cfg.H))]
    xs = synth.slice_chains({k: v for k, v in x.items() if k not in ("A", "tau")}, chains)
    xs["A"] = xs["tau"] = None
    cts = synth.slice_chains(ct, chains)
    return chains, xs, cts


def time_oracle(cfg: synth.Config, x: dict, ct: dict, steps: int, warmup: int):
    from oracle import carve_oracle as orc
    cores = orc.num_threads()
    n = min(cfg.B * cfg.H, 2 * cores)
    chains, xs, cts = oracle_sample(cfg, x, ct, n)
    s = orc.Shape(B=len(chains), H=1, T=cfg.T, L=cfg.L, dk=cfg.dk, dv=cfg.dv, r=cfg.r,
                  qk_l2norm=cfg.qk_l2norm, scale=cfg.scale, eps=cfg.eps)
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        orc.fwd(s, xs)
        if not cfg.fwd_only:
            orc.bwd(s, xs, cts["dO"], cts["dS_final"])
        if i >= warmup:
            times.append(time.perf_counter() - t0)
    tok_equiv = len(chains) * cfg.T / cfg.H   # a token carries all H heads; the sample holds n of B*H chains
    sec = sum(times) / len(times)
    return dict(value=tok_equiv / sec, unit="tokens/s", cores=cores, kind="oracle",
                sample=f"{len(chains)} of {cfg.B * cfg.H} (batch,head) chains of {cfg.name}, full T={cfg.T}, "
                       f"fp64 oracle fwd{'' if cfg.fwd_only else '+bwd'}, {sec:.2f} s per step"), sec


def base_line(cfg: synth.Config, args, n_gpus: int) -> dict:
    return {"metric": METRIC, "unit": "tokens/s", "n_gpus": n_gpus, "steps": args.steps, "warmup": args.warmup,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16 tokens, f32 state/accumulate" if cfg.dtype == "bf16" else "f32", "data": "synthetic",
            "config": {"workload": f"{cfg.name}: B={cfg.B} (per GPU),H={cfg.H},T={cfg.T},L={cfg.L},dk={cfg.dk},"
                                   f"dv={cfg.dv},r={cfg.r},{cfg.dtype},S0={'N(0,%g)' % cfg.s0_std if cfg.s0_std else 0}"
                                   f"{', fwd only' if cfg.fwd_only else ', fwd+bwd'}"
                                   f"{', scalar-write variant (w == 1)' if getattr(args, 'scalar_write', False) else ''}",
                       "seed": cfg.seed, "parallelism": f"dp{n_gpus} over batch (independent chains)",
                       "l2": "inputs (>=0.8 GB per pass) exceed the 126 MB L2; no explicit flush"},
            "context": PAPER_CONTEXT}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = get_cfg(args.config)
    cores = os.cpu_count() or 1
    n = min(cfg.B * cfg.H, 2 * cores)
    small = cfg.with_(B=max(1, -(-n // cfg.H)))       # only generate the batches the sample touches
    x, ct = synth.make_inputs(small), synth.make_cotangents(small)
    cb, sec = time_oracle(small.with_(name=cfg.name), x, ct, args.steps, min(args.warmup, 1))
    cb["sample"] = cb["sample"].replace(f"of {small.B * small.H}", f"of {cfg.B * cfg.H}")
    line = base_line(cfg, args, args.gpus)
    line.update({"impl": "reference", "value": cb["value"], "ms_per_step": sec * 1e3, "cpu_baseline": cb,
                 "e2e": {"value": cb["value"], "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                 "gpu_launches": 0, "dtype": "f64"})
    print(json.dumps(line), flush=True)


def run_step(args):
    """`--op step`: the recurrent decode call carve_step, one new token per sequence and call.
    Not the BASELINE.json metric: decode tokens/s (B sequences x 1 token per step) and the fraction of the HBM roofline
    of a decode step, whose algorithmic traffic is the state's round trip, 2 x 4 dv dk bytes per (batch, head) chain."""
    import torch
    from paper_2606_27229_b200 import carve
    torch.cuda.set_device(0)
    base = get_cfg(args.config)
    cfg = base.with_(B=args.decode_batch, T=1, L=16, s0_std=0.1)
    x = synth.make_inputs(cfg)
    tok_dt = torch.bfloat16 if cfg.dtype == "bf16" else torch.float32
    xd = {}
    for n, a in x.items():
        if a is None:
            xd[n] = None
            continue
        t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
        xd[n] = (t.to(tok_dt) if n in synth.TOKEN_TENSORS else t).cuda()
    p = carve.Params(B=cfg.B, H=cfg.H, T=1, L=16, dk=cfg.dk, dv=cfg.dv, r=cfg.r,
                     dtype=carve.CARVE_BF16 if cfg.dtype == "bf16" else carve.CARVE_F32)
    # several state buffers in rotation, together larger than the 126 MB L2
    nbuf = max(2, int(200e6 // (cfg.B * cfg.H * cfg.dv * cfg.dk * 4)) + 1)
    S = [xd["S0"].clone() for _ in range(nbuf)]
    O = torch.empty(cfg.B, 1, cfg.H, cfg.dv, dtype=tok_dt, device="cuda")
    st = torch.cuda.current_stream()
    for i in range(max(args.warmup, 3)):
        carve.carve_step(p, xd, S[i % nbuf], O, st.cuda_stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for i in range(args.steps):
        carve.carve_step(p, xd, S[i % nbuf], O, st.cuda_stream)
    e1.record(st)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    peaks = load_peaks()
    bytes_alg = cfg.B * cfg.H * cfg.dv * cfg.dk * 4 * 2
    ach = bytes_alg / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "CARVE decode step (carve_step) tokens/sec", "unit": "tokens/s", "n_gpus": 1, "steps": args.steps,
                      "warmup": args.warmup, "higher_is_better": True, "value": cfg.B / (ms * 1e-3), "ms_per_step": ms,
                      "dtype": "bf16 tokens, f32 state/arithmetic", "data": "synthetic",
                      "config": {"workload": f"decode: B={cfg.B} sequences x 1 new token, H={cfg.H}, dk={cfg.dk}, dv={cfg.dv}, r={cfg.r}; "
                                             f"{nbuf} state buffers in rotation (> L2)"},
                      "gpu_launches": args.steps,
                      "roofline": {"bound": "hbm", "kernel": "carve_step_kernel", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                   "frac": ach / peaks["hbm_gbs"], "traffic": None, "algorithmic_bytes_per_launch": bytes_alg}}), flush=True)


def run_layer_ends(args):
    """`--op layer_ends`: the two chunk-local passes around the operator: SiLU on q,k,v and RMSNorm
    of the assembled output, forward and backward, at the token shape of --config.  Not the BASELINE.json metric: tokens/s
    through the four launches and, per launch, the fraction of the HBM roofline (algorithmic bytes = every tensor read or
    written once).  The tensors of one step (1.2 GB at config 1) exceed the 126 MB L2."""
    import torch
    from paper_2606_27229_b200 import carve
    torch.cuda.set_device(0)
    cfg = get_cfg(args.config)
    tok_dt = torch.bfloat16 if cfg.dtype == "bf16" else torch.float32
    e = 2 if cfg.dtype == "bf16" else 4
    p = carve.Params(B=cfg.B, H=cfg.H, T=cfg.T, L=cfg.L, dk=cfg.dk, dv=cfg.dv, r=cfg.r,
                     dtype=carve.CARVE_BF16 if cfg.dtype == "bf16" else carve.CARVE_F32)
    g = torch.Generator(device="cuda").manual_seed(0)
    mk = lambda d: torch.randn(cfg.B, cfg.T, cfg.H, d, device="cuda", generator=g).to(tok_dt)
    qx, kx, vx, o, dy = mk(cfg.dk), mk(cfg.dk), mk(cfg.dv), mk(cfg.dv), mk(cfg.dv)
    q, k, v, y, d_o = (torch.empty_like(t) for t in (qx, kx, vx, o, dy))
    dq, dk, dv = mk(cfg.dk), mk(cfg.dk), mk(cfg.dv)
    gain = torch.ones(cfg.H * cfg.dv, device="cuda")
    dgain = torch.empty_like(gain)
    ws = torch.empty(carve.carve_out_norm_workspace_bytes(p), dtype=torch.uint8, device="cuda")
    st = torch.cuda.current_stream()
    tokh = cfg.B * cfg.T * cfg.H
    calls = {
        "silu_qkv_fwd": (lambda: carve.carve_silu_qkv_fwd(p, qx, kx, vx, q, k, v, st.cuda_stream), 2 * tokh * (2 * cfg.dk + cfg.dv) * e, 1),
        "silu_qkv_bwd": (lambda: carve.carve_silu_qkv_bwd(p, qx, kx, vx, dq, dk, dv, st.cuda_stream), 3 * tokh * (2 * cfg.dk + cfg.dv) * e, 1),
        "out_norm_fwd": (lambda: carve.carve_out_norm_fwd(p, o, gain, 1e-5, y, st.cuda_stream), 2 * tokh * cfg.dv * e, 1),
        "out_norm_bwd": (lambda: carve.carve_out_norm_bwd(p, o, gain, 1e-5, dy, d_o, dgain, ws, st.cuda_stream), 3 * tokh * cfg.dv * e, 2),
    }
    peaks = load_peaks()
    per, total_ms, launches = {}, 0.0, 0
    for name, (fn, nbytes, nl) in calls.items():
        for _ in range(max(args.warmup, 3)):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(args.steps):
            fn()
        e1.record(st)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        ach = nbytes / (ms * 1e-3) / 1e9
        per[name] = {"ms": ms, "algorithmic_bytes": nbytes, "achieved_GBps": ach, "frac": ach / peaks["hbm_gbs"]}
        total_ms += ms
        launches += nl * args.steps
    tot_bytes = sum(c[1] for c in calls.values())
    ach = tot_bytes / (total_ms * 1e-3) / 1e9
    print(json.dumps({"metric": "CARVE layer ends (SiLU q,k,v + RMSNorm(o), fwd+bwd) tokens/sec", "unit": "tokens/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": args.warmup, "higher_is_better": True,
                      "value": cfg.B * cfg.T / (total_ms * 1e-3), "ms_per_step": total_ms, "dtype": cfg.dtype, "data": "synthetic",
                      "config": {"workload": f"{cfg.name}: B={cfg.B},H={cfg.H},T={cfg.T},dk={cfg.dk},dv={cfg.dv}; tensors of a step exceed L2"},
                      "gpu_launches": launches, "calls": per,
                      "roofline": {"bound": "hbm", "kernel": "the four launches together", "achieved": ach, "peak": peaks["hbm_gbs"],
                                   "unit": "GB/s", "frac": ach / peaks["hbm_gbs"], "traffic": None,
                                   "algorithmic_bytes_per_launch": tot_bytes}}), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2606_27229_b200 import carve

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CARVE path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = get_cfg(args.config).with_(seed=rank)       # each rank owns a different batch shard
    if args.fwd_only:
        cfg = cfg.with_(fwd_only=True)
    carve.load_library()
    tok_dt = torch.bfloat16 if cfg.dtype == "bf16" else torch.float32
    p = carve.Params(B=cfg.B, H=cfg.H, T=cfg.T, L=cfg.L, dk=cfg.dk, dv=cfg.dv, r=cfg.r,
                     dtype=carve.CARVE_BF16 if cfg.dtype == "bf16" else carve.CARVE_F32,
                     qk_l2norm=cfg.qk_l2norm, scale=cfg.scale, eps=cfg.eps)
    with_bwd = not cfg.fwd_only

    # ---- seeded synthetic inputs: host (pinned) and device copies
    x, ct = synth.make_inputs(cfg), synth.make_cotangents(cfg)

    def host_t(name, a):
        if a is None:
            return None
        t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
        if name in synth.TOKEN_TENSORS or name == "dO":
            t = t.to(tok_dt)
        return t.contiguous().pin_memory()

    xh = {n: host_t(n, a) for n, a in x.items()}
    dOh, dSfh = host_t("dO", ct["dO"]), host_t("dS_final", ct["dS_final"])
    if args.scalar_write:      # P section 4.2 l.145: w == 1, the scalar write gate is inside beta (carve.h)
        for n in ("wx", "Uw", "Vw"):
            xh[n] = None
    xd = {n: (None if t is None else t.cuda()) for n, t in xh.items()}
    dOd, dSfd = dOh.cuda(), dSfh.cuda()
    dev = torch.device("cuda", local)
    O = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, dtype=tok_dt, device=dev)
    Sf = torch.empty(cfg.B, cfg.H, cfg.dv, cfg.dk, dtype=torch.float32, device=dev)
    wgrad = torch.zeros(2 * cfg.r * cfg.dv + cfg.dk * cfg.r + cfg.dv * cfg.r + 2 * cfg.H * cfg.dk,
                        dtype=torch.float32, device=dev)     # packed weight grads: one all-reduce buffer

    def mk_grads(device, pin=False):
        B, H, T, dk, dv, r = cfg.B, cfg.H, cfg.T, cfg.dk, cfg.dv, cfg.r
        mk = lambda dt, *s: (torch.empty(*s, dtype=dt).pin_memory() if pin else torch.empty(*s, dtype=dt, device=device))
        g = {"dq": mk(tok_dt, B, T, H, dk), "dk": mk(tok_dt, B, T, H, dk), "dv": mk(tok_dt, B, T, H, dv),
             "df": mk(tok_dt, B, T, H, dk), "dbx": mk(tok_dt, B, T, H, dk), "dwx": mk(tok_dt, B, T, H, dv),
             "dbeta": mk(tok_dt, B, T, H), "dS0": mk(torch.float32, B, H, dv, dk)}
        if pin:
            g.update({"dUb": mk(torch.float32, r, dv), "dUw": mk(torch.float32, r, dv),
                      "dVb": mk(torch.float32, dk, r), "dVw": mk(torch.float32, dv, r),
                      "dA": mk(torch.float32, H, dk), "dtau": mk(torch.float32, H, dk)})
        else:
            o = 0
            for n, shp in (("dUb", (r, dv)), ("dUw", (r, dv)), ("dVb", (dk, r)), ("dVw", (dv, r)),
                           ("dA", (H, dk)), ("dtau", (H, dk))):
                k = shp[0] * shp[1]
                g[n] = wgrad[o:o + k].view(*shp)
                o += k
        return g

    grads = mk_grads(dev) if with_bwd else None
    if args.scalar_write and grads:
        for n in ("dwx", "dUw", "dVw"):
            grads[n] = None
    ws = torch.empty(carve.carve_workspace_bytes(p, True), dtype=torch.uint8, device=dev) if with_bwd else None
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step(evs=None):
        if evs: evs[0].record(stream)
        carve.carve_fwd(p, xd, O, Sf, ws, stream.cuda_stream)
        if evs: evs[1].record(stream)
        if with_bwd:
            carve.carve_bwd(p, xd, dOd, dSfd, grads, ws, stream.cuda_stream)
            if evs: evs[2].record(stream)
            if world > 1:
                dist.all_reduce(wgrad)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    kev = [[ev(), ev(), ev()] for _ in range(args.steps)]
    t_begin, t_end = ev(), ev()
    barrier()
    sampler.mark()
    t_begin.record(stream)
    for i in range(args.steps):
        step(kev[i])
    t_end.record(stream)
    barrier()
    sampler.mark()
    ms_total = t_begin.elapsed_time(t_end)
    clocks = sampler.stop() if rank == 0 else None
    fwd_ms = statistics.mean(k[0].elapsed_time(k[1]) for k in kev)
    bwd_ms = statistics.mean(k[1].elapsed_time(k[2]) for k in kev) if with_bwd else 0.0
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / args.steps
    tokens_job = cfg.tokens * world
    value = tokens_job / (ms_step * 1e-3)

    # ---- e2e: the host-buffer C-ABI call, copies inside the timed region
    Oh = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, dtype=tok_dt).pin_memory()
    Sfh = torch.empty(cfg.B, cfg.H, cfg.dv, cfg.dk, dtype=torch.float32).pin_memory()
    gh = mk_grads("cpu", pin=True) if with_bwd else None
    del ws
    arena = torch.empty(carve.carve_host_arena_bytes(p, with_bwd), dtype=torch.uint8, device=dev)
    nb = lambda t: 0 if t is None else t.numel() * t.element_size()
    h2d = sum(nb(t) for t in xh.values()) + (nb(dOh) + nb(dSfh) if with_bwd else 0)
    d2h = nb(Oh) + nb(Sfh) + (sum(nb(t) for t in gh.values()) if with_bwd else 0)
    e2e_steps = 0 if args.scalar_write else max(1, min(args.steps, 5))   # the host entry point takes the full write gate only

    hctx = carve.carve_host_ctx_create()     # the call's side streams and events, created once

    def e2e_step():
        carve.carve_fwd_bwd_host(p, with_bwd, xh, Oh, Sfh, dOh if with_bwd else None, dSfh if with_bwd else None,
                                 gh, arena, stream.cuda_stream, ctx=hctx)
    if e2e_steps:
        e2e_step()
    barrier()
    e0, e1 = ev(), ev()
    e0.record(stream)
    for _ in range(e2e_steps):
        e2e_step()
    e1.record(stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    if world > 1:
        t = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t.item())
    e2e_value = tokens_job / (e2e_ms / e2e_steps * 1e-3) if e2e_steps else None

    if rank == 0:
        alg = algorithmic(cfg, args.scalar_write)
        peaks = load_peaks()
        dom = "bwd" if (with_bwd and bwd_ms >= fwd_ms) else "fwd"
        dom_ms = bwd_ms if dom == "bwd" else fwd_ms
        dom_bytes = alg[f"{dom}_bytes"]
        achieved = dom_bytes / (dom_ms * 1e-3) / 1e9
        traffic = None      # DRAM bytes of that call from the newest committed ncu capture (config 1, tensor path only)
        tpath = os.path.join(ROOT, "profiles", "r2_tc_traffic.csv")
        if not os.path.exists(tpath):
            tpath = os.path.join(ROOT, "profiles", "r1_tc_traffic.csv")
        if cfg.name == synth.CFG1.name and not args.fwd_only and not args.scalar_write and os.path.exists(tpath):
            for ln in open(tpath).read().splitlines()[1:]:
                f = ln.split(",")
                if f[0] == f"carve_{dom}":
                    traffic = int(f[2]) + int(f[3])
        t_hbm = (alg["fwd_bytes"] + alg["bwd_bytes"]) / (peaks["hbm_gbs"] * 1e9)
        t_tc = (alg["fwd_flops"] + alg["bwd_flops"]) / (peaks["bf16_tflops"] * 1e12)
        path = carve.carve_resolved_path(p, with_bwd)
        line = base_line(cfg, args, world)
        line.update({
            "value": value, "ms_per_step": ms_step, "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "tokens/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps if e2e_steps else None},
            "gpu_launches": args.steps * (carve.carve_num_launches(p, False) +
                                          (carve.carve_num_launches(p, True) if with_bwd else 0)),
            "kernel_path": {1: "simt-fp32", 2: "tensor-tcgen05"}.get(path, str(path)),
            "fwd_ms": fwd_ms, "bwd_ms": bwd_ms,
            "roofline": {"bound": "hbm",
                         "kernel": (f"carve_{dom} call" + (" (reverse kernel + chunk-local epilogue + 2 reductions)"
                                                           if dom == "bwd" and path == 2 else "")),
                         "achieved": achieved, "peak": peaks["hbm_gbs"],
                         "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"], "traffic": traffic,
                         "traffic_source": (f"profiles/{os.path.basename(tpath)} (ncu --set full capture of this command; "
                                            "dram__bytes_read.sum + dram__bytes_write.sum per launch)") if traffic else None,
                         "peak_source": f"{peaks['source']} (MEASURED_PEAKS.json hbm_gbs)" if peaks["source"] == "measured"
                         else "fallback 6650 GB/s",
                         "algorithmic_bytes_per_launch": dom_bytes},
            "layer_roofline": {"t_hbm_ms": t_hbm * 1e3, "t_tensor_ms": t_tc * 1e3, "binding": "hbm" if t_hbm >= t_tc else "tensor",
                               "roofline_tokens_per_s": cfg.tokens / max(t_hbm, t_tc),
                               "frac": max(t_hbm, t_tc) * 1e3 / ms_step,
                               "algorithmic_bytes": alg["fwd_bytes"] + alg["bwd_bytes"],
                               "algorithmic_flops": alg["fwd_flops"] + alg["bwd_flops"]},
        })
        if world == 1 and not args.no_cpu_baseline:
            cb, _ = time_oracle(cfg, x, ct, 1, 1)     # one warm-up pass (page faults, thread pool), one timed
            line["cpu_baseline"] = cb
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg1")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fwd-only", action="store_true", help="time carve_fwd alone (inference call, nothing saved)")
    ap.add_argument("--op", default="train", choices=["train", "step", "layer_ends"],
                    help="step: time the decode call carve_step instead; layer_ends: the SiLU / RMSNorm passes around the operator")
    ap.add_argument("--decode-batch", type=int, default=256)
    ap.add_argument("--scalar-write", action="store_true",
                    help="the scalar-write variant (wx = Uw = Vw = NULL, PAPER.md section 4.2): not the BASELINE.json metric's workload")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        # plain `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU, NCCL), the same way the
        # driver does with torchrun
        import socket
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            raise SystemExit(f"bench.py --gpus {args.gpus}: only {have} CUDA device(s) visible")
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        env = dict(os.environ, NCCL_DEBUG=os.environ.get("NCCL_DEBUG", "WARN"))
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd, env=env))
    if args.op == "step":
        run_step(args)
    elif args.op == "layer_ends":
        run_layer_ends(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
