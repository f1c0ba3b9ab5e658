#!/usr/bin/env python
"""bench.py -- GDN chunk-forward throughput on B200 (BASELINE.json's metric and workload).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2|3] [--mode token|frame]

A "step" is one pass of the whole hot path (one gdn_forward_chunk call = one streaming chunk) over one
batch of synthetic input; the state of step i is the state_in of step i+1 (a real stream).  Prints ONE
JSON line (rank 0).  See DESIGN.md "Measurement" for what every field means.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "gdn_chunk_fwd_tokens_per_s"
UNIT = "tokens/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
L2_BYTES = 126e6


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            d = json.loads(p.read_text())
            return {k: float(d[k]) for k in FALLBACK_PEAKS}, "measured"
        except Exception:
            pass
    return dict(FALLBACK_PEAKS), "fallback"


def workload(args):
    from paper_2605_30409_b200 import inputs as gin
    if args.paper_shape:
        return gin.paper_shape(3, d=112 if args.d112 else 128)   # 3 x 880 tokens, 20 heads, d = 112 or padded 128
    wl = gin.config(args.config, frame=(args.mode == "frame"), chunk=args.chunk)
    return wl


def flops_per_call(wl, chunk):
    """Algorithmic flops: mode T 6d^2 + 10 C d per token-head; mode F 6 d^2 per token-head
    + 2 d^3 per frame-head.  (Inverse and element-wise work excluded.)"""
    d = wl.d_k
    th = wl.B * wl.H * wl.T
    if wl.group == 1:
        C = chunk or 64
        return th * (6 * d * d + 10 * C * d)           # depends on the compute tile C: see flops_report for the C = 64 figure
    return th * 6 * d * d + wl.B * wl.H * (wl.T // wl.group) * 2 * d ** 3


def flops_report(wl, chunk, ms_per_step, by, pk):
    """TFLOP/s and % of the bf16 peak with BOTH flop formulas of SURVEY 8d (the token-wise count grows with the compute
    tile C the implementation picks, so the C = 64 figure is the one that compares across implementations), and the
    HBM-limited cap of each: flops / algorithmic bytes x measured HBM peak, as % of the measured bf16 peak."""
    out = {}
    for tag, C in (("c_in_use", chunk or 64), ("c64", 64)):
        fl = flops_per_call(wl, C)
        tf = fl / (ms_per_step * 1e-3) / 1e12
        out[tag] = {"C": C if wl.group == 1 else None, "gflop_per_call": fl / 1e9, "tflops": tf,
                    "pct_bf16_peak": 100 * tf / pk["bf16_tflops"],
                    "hbm_limited_cap_pct_bf16_peak": 100 * (fl / by) * pk["hbm_gbs"] * 1e9 / 1e12 / pk["bf16_tflops"]}
        if wl.group != 1:
            break
    return out


def bytes_per_call(wl):
    """Algorithmic HBM bytes: q,k,v read once, out written once (2 B each), alpha/beta fp32, state in+out."""
    th = wl.B * wl.H * wl.T
    es = 4 if str(wl.dtype).endswith("float32") else 2
    per_tok = (2 * wl.d_k + 2 * wl.d_v) * es + 4 + (4 if wl.group == 1 else 0)
    return th * per_tok + 2 * wl.B * wl.H * wl.d_k * wl.d_v * 4 + (0 if wl.group == 1 else wl.B * wl.H * (wl.T // wl.group) * 4)


# ---------------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU during the timed region (pynvml)."""

    def __init__(self, index: int, period: float = 0.002):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._halt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._halt.set()
        if self.is_alive():
            self.join(timeout=2)
        s = self.samples
        return {"sm_mhz": statistics.median(s) if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# ---------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the CPU oracle as it stands, timed on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    from paper_2605_30409_b200 import inputs as gin
    wl = workload(args)
    inp = gin.make_inputs(wl)
    cores = oracle.max_threads()
    st = inp.state
    for _ in range(args.warmup):
        _, st = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, st, group=wl.group)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, st = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, st, group=wl.group)
    dt = time.perf_counter() - t0
    tokens = wl.B * wl.T * args.steps
    val = tokens / dt
    sample = f"full {wl.name} workload ({wl.B}x{wl.T} tokens, {wl.H} heads, d={wl.d_k}) per step, {args.steps} steps"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(wl, None),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def config_dict(wl, info, extra=None):
    src = f"BASELINE.json configs[{int(wl.name[3]) - 1}]" if wl.name.startswith("cfg") else "the paper's production chunk"
    d = {"workload": f"{src} ({wl.name}): B={wl.B} H={wl.H} T={wl.T} "
                     f"d_k=d_v={wl.d_k} {str(wl.dtype).split('.')[-1]}, "
                     + ("token-wise (G=1)" if wl.group == 1 else f"frame-wise (G={wl.group})"),
         "B": wl.B, "H": wl.H, "T": wl.T, "d_k": wl.d_k, "d_v": wl.d_v, "group": wl.group,
         "parallelism": "replicas only (no collective)"}
    if info is not None:
        d.update({"path": info[0], "chunk": info[1], "launches_per_call": info[2]})
    if extra:
        d.update(extra)
    return d


def cpu_baseline(wl, budget_s=12.0):
    """The oracle, as it stands, on a bounded sample of the same workload (rank 0, N=1): the full workload repeated
    with carried state until `budget_s` seconds of CPU work have been spent."""
    import oracle
    from paper_2605_30409_b200 import inputs as gin
    inp = gin.make_inputs(wl)
    cores = oracle.max_threads()
    _, st = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=wl.group)   # warm-up, untimed
    reps = 0
    t0 = time.perf_counter()
    while True:
        _, st = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, st, group=wl.group)
        reps += 1
        dt = time.perf_counter() - t0
        if dt >= budget_s or reps >= 100000:
            break
    return {"value": wl.B * wl.T * reps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"full {wl.name} workload x {reps} carried-state repeats ({dt:.1f} s of CPU work)"}


def max_over_ranks(ms, dist, device=None):
    """Device time of the slowest rank (every rank gets it). `dist` is torch.distributed or None (one process)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_tokens_per_s(world, wl, steps, ms):
    """Whole-job throughput of `world` independent replicas (replicas only, weak scaling):
    the tokens all ranks processed divided by the slowest rank's time."""
    return world * wl.B * wl.T * steps / (ms * 1e-3)


def rank_seed(wl, rank, i):
    """Seed of input set i on `rank`: every replica streams its own data."""
    return wl.seed + 17 * i + 1000 * rank


def run_ours(args):
    import torch
    import paper_2605_30409_b200 as gdn
    from paper_2605_30409_b200 import inputs as gin

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    wl = workload(args)
    es = 2 if wl.dtype == torch.bfloat16 else 4
    set_bytes = wl.B * wl.T * wl.H * (2 * wl.d_k + 2 * wl.d_v) * es
    n_sets = max(2, int(L2_BYTES * 1.5 // set_bytes) + 1)         # rotate so the inputs of a step are cold in L2
    n_sets = min(n_sets, 16)
    norm = bool(args.normalizer) or bool(args.full)
    if norm:
        set_bytes += wl.B * wl.T * wl.H * 2 * wl.d_k * es
        n_sets = min(16, max(2, int(L2_BYTES * 1.5 // set_bytes) + 1))
    sets = []
    for i in range(n_sets):
        inp = (gin.make_normalizer_inputs if norm else gin.make_inputs)(wl, seed=rank_seed(wl, rank, i))
        d = dict(q=inp.q.to(dev), k=inp.k.to(dev), v=inp.v.to(dev), alpha=inp.alpha.to(dev),
                 beta=inp.beta.to(dev), out=torch.empty(wl.B, wl.T, wl.H, wl.d_v, dtype=wl.dtype, device=dev))
        if norm:
            d.update(q_raw=inp.extras["q_raw"].to(dev), k_raw=inp.extras["k_raw"].to(dev))
        sets.append(d)
    first = (gin.make_normalizer_inputs if norm else gin.make_inputs)(wl)
    state = first.state.to(dev)
    zstate = first.extras["z_in"].to(dev) if norm else None
    flags = (gdn.GDN_FLAG_NORMALIZER if norm else 0) | (gdn.GDN_FLAG_BIDIR if args.bidir else 0) | (gdn.GDN_FLAG_UNFUSED if args.unfused else 0)
    plan = gdn.GdnPlan(B=wl.B, H=wl.H, T=wl.T, d_k=wl.d_k, d_v=wl.d_v, group=wl.group, chunk=wl.chunk, flags=flags,
                       io_dtype=gdn.GDN_BF16 if wl.dtype == torch.bfloat16 else gdn.GDN_FP32)
    info = plan.info
    stream = torch.cuda.Stream(device=dev)         # a stream of its own (the library replays CUDA graphs on non-default streams)
    stream.wait_stream(torch.cuda.current_stream())

    full = None
    if args.full:
        # operands of the front end; one packed qkv tensor per input set (the q / k / v views carry the packed token stride)
        full = []
        for i in range(n_sets):
            fi = gin.make_frontend_inputs(wl, seed=rank_seed(wl, rank, i) + 17)
            dd = {n: fi[n].to(dev) for n in ("qkv", "x", "w_q", "w_k", "cos", "sin", "w_alpha", "b_alpha", "a_log", "w_beta", "b_beta", "gate")}
            dd["fm"] = gdn.make_featmap_args(dd["qkv"][:, :, 0], dd["qkv"][:, :, 1], dd["w_q"], dd["w_k"], dd["cos"], dd["sin"], 1e-6)
            dd["ga"] = gdn.make_gate_args(dd["x"], dd["w_alpha"], dd["b_alpha"], dd["a_log"], dd["w_beta"], dd["b_beta"])
            full.append(dd)
        plan.close()
        st3 = 3 * wl.H * wl.d_k
        plan = gdn.GdnPlan(B=wl.B, H=wl.H, T=wl.T, d_k=wl.d_k, d_v=wl.d_v, group=wl.group, flags=flags | gdn.GDN_FLAG_LOG_ALPHA,
                           q_token_stride=st3, k_token_stride=st3, v_token_stride=st3)
        info = plan.info

    def step(i):
        s = sets[i % n_sets]
        if full is not None:
            f = full[i % n_sets]
            plan.forward_full(f["fm"], f["qkv"][:, :, 2], f["ga"], None, None, f["gate"], state, zstate, s["out"], state, zstate, stream=stream)
        elif norm:
            plan.forward_norm(s["q"], s["k"], s["v"], s["q_raw"], s["k_raw"], s["alpha"], s["beta"], state, zstate,
                              s["out"], state, zstate, stream=stream)
        else:
            plan.forward(s["q"], s["k"], s["v"], s["alpha"], s["beta"], state, s["out"], state, stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    for i in range(args.warmup):
        step(i)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(args.steps):
        step(i)
    e1.record(stream)
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, dev)
    assert torch.isfinite(state).all(), "state diverged"
    ms_per_step = ms / args.steps
    tokens_per_s = job_tokens_per_s(world, wl, args.steps, ms)

    # ---- per-kernel durations (separate pass with CUDA events between the launches) ----------------
    kernels = plan_kernel_times(plan, step, args.steps, barrier)

    # ---- end to end through the host entry point (pinned host buffers, copies inside the timing) ----
    e2e = None
    if not args.no_e2e and not norm:
        inp = gin.make_inputs(wl)
        pin = lambda t: t.contiguous().pin_memory()
        hq, hk, hv, ha, hb, hs = map(pin, (inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state))
        hout = torch.empty(wl.B, wl.T, wl.H, wl.d_v, dtype=wl.dtype).pin_memory()
        k_e2e = max(3, min(args.steps, 50))
        for _ in range(3):
            plan.forward_host(hq, hk, hv, ha, hb, hs, hout, hs, stream)
        barrier()
        e0.record(stream)
        for _ in range(k_e2e):
            plan.forward_host(hq, hk, hv, ha, hb, hs, hout, hs, stream)
        e1.record(stream)
        barrier()
        ms_e = max_over_ranks(e0.elapsed_time(e1), dist, dev)
        nbytes = lambda *ts: int(sum(t.numel() * t.element_size() for t in ts))
        e2e = {"value": job_tokens_per_s(world, wl, k_e2e, ms_e), "unit": UNIT,
               "h2d_bytes_per_step": nbytes(hq, hk, hv, ha, hb, hs), "d2h_bytes_per_step": nbytes(hout, hs),
               "steps": k_e2e, "ms_per_step": ms_e / k_e2e}

    clocks = sampler.stop()                        # sampled from before the warm-up to the end of the e2e leg
    pk, pk_src = peaks()
    fl = flops_per_call(wl, info.chunk)
    by = bytes_per_call(wl)
    if norm:                                       # + 2 d^2 flops and + 4 d bytes per token-head (q_raw, k_raw), + z in/out
        fl += wl.B * wl.H * wl.T * 2 * wl.d_k * wl.d_k
        by += wl.B * wl.H * wl.T * 2 * wl.d_k * es + 2 * wl.B * wl.H * wl.d_k * 4
    if args.full:                                  # qkv, x and the output gate read once, out written once; alpha / beta never leave the device
        by = wl.B * wl.H * wl.T * 6 * wl.d_k * es + 2 * wl.B * wl.H * (wl.d_k * wl.d_v + wl.d_k) * 4
    tflops = fl / (ms_per_step * 1e-3) / 1e12
    roof = roofline(wl, info, kernels, ms_per_step, pk, pk_src, by)
    line = {
        "metric": METRIC, "value": tokens_per_s, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16" if wl.dtype == torch.bfloat16 else "f32", "data": "synthetic",
        "config": config_dict(wl, (gdn.PATH_NAMES[info.path], info.chunk, info.launches_per_call),
                              {"l2": f"rotating {n_sets} input sets ({n_sets * set_bytes / 1e6:.0f} MB > 126 MB L2), carried state"}),
        "tflops": tflops, "pct_bf16_peak": 100 * tflops / pk["bf16_tflops"], "peaks": pk_src,
        "flops": flops_report(wl, info.chunk, ms_per_step, by, pk),
        "hbm_gbs_algorithmic": by / (ms_per_step * 1e-3) / 1e9,
        "clocks": clocks, "e2e": e2e, "gpu_launches": args.steps * (info.launches_per_call + (1 if args.full else 0)),      # --full: + the front-end kernel
        "roofline": roof, "kernels": kernels,
    }
    if norm or args.bidir:
        line["config"]["variant"] = "+".join(x for x, on in (("full operator (feature map, gates, output gate)", bool(args.full)), ("normalizer", norm), ("bidir", args.bidir)) if on)
    if rank == 0 and world == 1 and not args.no_cpu and not norm and not args.bidir:
        line["cpu_baseline"] = cpu_baseline(wl)
    plan.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def plan_kernel_times(plan, step, steps, barrier):
    """Average duration of every kernel of a call, from CUDA events the library records between its own
    launches on the launching stream (gdn_plan_set_profiling; a separate pass, not the timed region)."""
    import paper_2605_30409_b200 as gdn
    if not hasattr(gdn, "gdn_plan_kernel_times"):
        return None
    n = min(steps, 200)
    gdn.gdn_plan_set_profiling(plan.handle, 1)
    for i in range(n):
        step(i)
    barrier()
    names, ms = gdn.gdn_plan_kernel_times(plan.handle)
    gdn.gdn_plan_set_profiling(plan.handle, 0)
    return [{"name": nm, "avg_us": 1e3 * m} for nm, m in zip(names, ms)]


def ncu_traffic(kernel, wl):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on this workload, from the committed
    ncu --set full summaries (profiles/ncu_traffic.csv); None when that kernel/workload was not captured."""
    f = ROOT / "profiles" / "ncu_traffic.csv"
    if not f.exists():
        return None
    key = (kernel, wl.name, "token" if wl.group == 1 else "frame")
    best = None
    for line in f.read_text().splitlines():
        c = [x.strip() for x in line.split(",")]
        if len(c) >= 5 and not line.startswith("#") and (c[0], c[1], c[2]) == key:
            best = float(c[3]) + float(c[4])          # later rows (later rounds) win
    return best


def ncu_counters(kernel, wl):
    """Tensor-pipe utilisation and DRAM throughput of `kernel` on this workload from the same committed ncu capture
    (north_star: "tensor-pipe utilisation and achieved HBM GB/s from ncu"); None when it was not captured."""
    f = ROOT / "profiles" / "ncu_traffic.csv"
    if not f.exists():
        return None
    key = (kernel, wl.name, "token" if wl.group == 1 else "frame")
    best = None
    for line in f.read_text().splitlines():
        c = [x.strip() for x in line.split(",")]
        if len(c) >= 9 and not line.startswith("#") and (c[0], c[1], c[2]) == key:
            us = float(c[6])
            best = {"source": "profiles/" + c[5], "gpu_time_us": us, "tensor_pipe_pct_of_active": float(c[7]),
                    "dram_pct_of_peak": float(c[8]), "dram_gbs": (float(c[3]) + float(c[4])) / (us * 1e-6) / 1e9}
    return best


def kernel_bytes(name, wl, by_call):
    """Algorithmic HBM bytes of ONE launch of kernel `name`: the user tensors that launch must
    read or write once; workspace traffic is not algorithmic."""
    th = wl.B * wl.H * wl.T
    es = 4 if str(wl.dtype).endswith("float32") else 2
    st = wl.B * wl.H * wl.d_k * wl.d_v * 4
    table = {
        "gdn_tok_prepass": th * ((2 * wl.d_k + wl.d_v) * es + 8),
        "gdn_tok_tile64": th * ((2 * wl.d_k + wl.d_v) * es + 8),
        "gdn_tok_output": th * wl.d_v * es,
        "gdn_tok_chain": 2 * st,
        "gdn_frm_summaries": th * ((wl.d_k + wl.d_v) * es + 4),
        "gdn_frm_summaries_dual": th * ((2 * wl.d_k + wl.d_v) * es + 4),      # k, k_raw, v, beta
        "gdn_frm_readout": th * (wl.d_k + wl.d_v) * es,
        "gdn_frontend_kernel": th * 7 * wl.d_k * es,      # q, k read; q_rot, k_rot, q_raw, k_raw written
    }
    if name.startswith("gdn_tok_chain"):
        return 2 * st                              # the scans only carry the state in and out; their summaries are workspace
    return table.get(name, by_call)               # single-kernel paths: the whole call


def roofline(wl, info, kernels, ms_per_step, pk, pk_src, by):
    """Roofline of the dominant kernel. HBM-bound: achieved = that kernel's algorithmic bytes / its duration."""
    dur_ms, name, kb = ms_per_step, "whole step", by
    if kernels:
        top = max(kernels, key=lambda k: k["avg_us"])
        dur_ms, name = top["avg_us"] * 1e-3, top["name"]
        kb = kernel_bytes(name, wl, by)
        if len(kernels) == 1 and info.launches_per_call == 1:
            # one launch per step: the kernel's average launch duration over the TIMED region is the step time itself (CUDA
            # events around the K steps).  The per-kernel pass puts an event pair around every launch, which keeps the
            # programmatic launches of consecutive calls from overlapping their set-up with the previous grid's tail.
            dur_ms = ms_per_step
    achieved = kb / (dur_ms * 1e-3) / 1e9
    # what the measurements say limits the kernel: below half of the HBM roofline (and, for the token path, with the
    # tensor pipe at 10-20 % in the ncu captures) the dominant kernel is bound by the latency of its dependent steps
    limiter = "hbm" if achieved / pk["hbm_gbs"] >= 0.5 else "latency (dependent MMA round trips / per-SM TMA rate; see DESIGN.md section 7)"
    return {"bound": "hbm", "observed_limiter": limiter, "kernel": name, "achieved": achieved, "peak": pk["hbm_gbs"], "unit": "GB/s",
            "frac": achieved / pk["hbm_gbs"], "traffic": ncu_traffic(name, wl), "peak_source": pk_src,
            "algorithmic_bytes": kb, "kernel_avg_us": dur_ms * 1e3, "ncu": ncu_counters(name, wl),
            "whole_call": {"algorithmic_bytes": by, "achieved": by / (ms_per_step * 1e-3) / 1e9,
                           "frac": by / (ms_per_step * 1e-3) / 1e9 / pk["hbm_gbs"]}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 5])
    ap.add_argument("--mode", default="token", choices=["token", "frame"])
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--normalizer", action="store_true", help="frame mode: the paper's normalised readout (Eq. 20-22)")
    ap.add_argument("--bidir", action="store_true", help="frame mode: bidirectional in-chunk scan (Alg. 1)")
    ap.add_argument("--paper-shape", action="store_true", help="3 x 880 tokens, 20 heads, d = 128, frame-wise")
    ap.add_argument("--d112", action="store_true", help="with --paper-shape: unpadded head dim 112")
    ap.add_argument("--full", action="store_true", help="frame mode: the operator at the paper's kernel boundary (Alg. 1): feature map + gates + "
                    "normalised (--bidir: bidirectional) recurrence + output gate through gdn_forward_chunk_full, from a packed qkv tensor")
    ap.add_argument("--unfused", action="store_true", help="token mode: the three-kernel path (prepass / chain / output) for A/B runs")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 5 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        run_reference(args)
    else:
        args.steps = 2000 if args.steps is None else args.steps
        args.warmup = max(3, 50 if args.warmup is None else args.warmup)
        run_ours(args)


if __name__ == "__main__":
    main()
