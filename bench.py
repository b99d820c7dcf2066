#!/usr/bin/env python
"""bench.py -- MPPI sample-steps/s and iteration latency on B200 (BASELINE.json:metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

One "step" = one MPPI iteration of the whole hot path (noise -> clamp -> RK4 rollout -> cost ->
softmax weights -> update) on the workload BASELINE.json's metric is quoted on: configs[1],
gate progress, K=4096 samples, N=50 steps, one controller, warm-started in place.  The timed
region has its inputs resident in HBM; L2 is flushed between timed iterations (a 256 MiB write,
outside the events).  Rank 0 prints ONE JSON line.  Multi-GPU: the path does not shard
(north_star: one GPU, no collectives) -> N independent replicas, value = N * units / max time.

--impl reference times the float64 CPU oracle (oracle/) as it stands on the host cores.
--survey (one GPU) times one iteration of EVERY workload of workloads.py -- the five configs, the
paper's own J_gate, input model and contouring -- for one controller and for 64, and prints a table
(not the JSON line; DESIGN.md section 7 quotes it).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "mppi_sample_steps_per_sec"
UNIT = "sample-steps/s"
# Algorithmic FP32 work per sample-step of the gate objective (
# SURVEY.md 8(d)): add/sub/mul = 1, FMA = 2, MUFU = 1, integer / min / max / compare = 0.
FLOPS_PER_SAMPLE_STEP = {0: 417.0, 1: 449.0, 2: 685.0}
FP32_LANES_PER_SM = 128
L2_FLUSH_BYTES = 256 << 20
# Issue slots of the scalar gate loop per warp-step (32 sample-steps), by instruction class (
# cuobjdump -sass of rollout_kernel<OBJ_GATE, fast math>): 154 FFMA (53 with three register operands, 101 with a
# constant operand), 67 FMUL, 44 FADD, 20 Philox half-rounds (IMAD.WIDE + LOP3), 11 MUFU, 8 FMNMX, 7 LDS.128.
GATE_LOOP_MIX = {"ffma_rrr": 53, "ffma_const": 101, "fmul": 67, "fadd": 44, "philox_half_round": 20, "mufu": 11, "fmnmx": 8, "lds": 7}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernel that runs cfg1, from the committed ncu --set full
# captures (not measured live): rollout_scan_kernel<gate> 75.8 KB read + 0 B written (profiles/README_r02f.md,
# ncu_details_scan_r02f.txt), rollout_pipe_kernel<gate> 55.6 KB + 0 B (profiles/README_r02e.md, ncu_details_pipe_r02e.txt)
NCU_DRAM_BYTES_PER_LAUNCH = {"time-parallel": (75776, "profiles/README_r02f.md"), "pipelined": (55552, "profiles/README_r02e.md")}


def kernel_label(info, P=None) -> str:
    """Which rollout kernel a context launches, from mppi_get_info (the library states shapes, not names)."""
    rate = bool(P and P.get("input_model", 0) == 1)
    if rate:
        return ("rate-model pipelined" if info["block_threads"] == 320 else
                "rate-model packed fp32x2" if info["samples_per_thread"] == 2 else "rate-model scalar")
    if info["rollout_warps_per_block"] == 16:
        return "time-parallel"
    if info["rollout_warps_per_block"] == 3 and info["block_threads"] == 256:
        return "pipelined"
    if info["samples_per_thread"] == 2:
        return "packed fp32x2"
    return "latency" if info["block_threads"] == 256 and info["rollout_warps_per_block"] < 8 else "scalar"


KERNEL_SYMBOL = {"time-parallel": "rollout_scan_kernel", "pipelined": "rollout_pipe_kernel", "packed fp32x2": "rollout2_kernel",
                 "latency": "rollout_lat_kernel", "scalar": "rollout_kernel"}


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def reduce_max_ms(ms: float, world: int, backend_device=None) -> float:
    """max over ranks of a duration (the contract's multi-GPU timing rule)."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=backend_device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(units_per_rank: float, world: int, max_ms: float) -> float:
    """whole-job throughput of N independent replicas: all ranks' units / the slowest rank's time."""
    return units_per_rank * world / (max_ms * 1e-3)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    _NAMES = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
              0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
              0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._halt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self._NAMES.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            self._halt.wait(self.period)

    def finish(self) -> dict:
        self._halt.set()
        if self.is_alive():
            self.join(timeout=1.0)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------
# the reference arm / cpu_baseline: the oracle as it stands, on the host cores
# ---------------------------------------------------------------------------------------------

def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def set_oracle_threads(n: int | None):
    """OpenMP team size of the oracle's sample loop (None = all online cores).  The oracle itself is not touched:
    this calls omp_set_num_threads of the OpenMP runtime it is linked against."""
    import ctypes
    from oracle import oracle as O
    O.lib()                                     # make sure libgomp is loaded
    gomp = ctypes.CDLL("libgomp.so.1")
    gomp.omp_set_num_threads(int(n or os.cpu_count() or 1))


def time_oracle(wl, budget_s: float, max_iters: int, sample_K: int | None = None):
    """Runs full oracle iterations of `wl` (optionally on the first sample_K samples) until the
    budget or max_iters is reached.  Returns (sample-steps/s, seconds per iteration, iterations, threads)."""
    from oracle import oracle as O
    p = dict(wl.params)
    if sample_K:
        p["K"] = int(sample_K)
    trk = O.Track(gates=wl.gates, ref=wl.ref, path=wl.path, closed=wl.closed)
    u = wl.u_nom.astype(np.float64)
    O.step(p, trk, wl.x0, wl.start, u, wl.seed, 0, want_diag=False)           # build + warm
    t0 = time.perf_counter()
    n = 0
    while n < max_iters and (time.perf_counter() - t0 < budget_s or n == 0):
        r = O.step(p, trk, wl.x0, wl.start, u, wl.seed, n, want_diag=False)
        u = r["u_new"]
        n += 1
    dt = time.perf_counter() - t0
    units = p["K"] * p["N"] * p["B"] * n
    return units / dt, dt / n, n, O.num_threads()


def run_reference(args):
    from paper_2509_14726_b200 import workloads as W
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    wl = W.cfg1()
    from oracle import oracle as O
    # size the per-step sample so that steps+warmup steps end within ~2 minutes
    rate, s_iter, _, threads = time_oracle(wl, 1.0, 3)
    total = args.steps + args.warmup
    sample_K = wl.params["K"]
    while sample_K > 32 and s_iter * sample_K / wl.params["K"] * total > 120.0:
        sample_K //= 2
    p = dict(wl.params); p["K"] = sample_K
    trk = O.Track(gates=wl.gates, ref=wl.ref, path=wl.path, closed=wl.closed)
    u = wl.u_nom.astype(np.float64)
    for i in range(args.warmup):
        u = O.step(p, trk, wl.x0, wl.start, u, wl.seed, i, want_diag=False)["u_new"]
    t0 = time.perf_counter()
    for i in range(args.steps):
        u = O.step(p, trk, wl.x0, wl.start, u, wl.seed, args.warmup + i, want_diag=False)["u_new"]
    dt = time.perf_counter() - t0
    units = sample_K * wl.params["N"] * args.steps
    value = units / dt
    sample = (f"{args.steps} iterations of {wl.name} restricted to the first {sample_K} of {wl.params['K']} samples"
              if sample_K != wl.params["K"] else f"{args.steps} full iterations of {wl.name}")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": wl.name, "K": wl.params["K"], "N": wl.params["N"], "B": 1,
                       "objective": "gate", "sample_K": sample_K},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                             "cpu": cpu_model()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------

def _events(n):
    import torch
    return [torch.cuda.Event(enable_timing=True) for _ in range(n)]


def time_steps(step_fn, flush_fn, steps, warmup):
    """W untimed steps, then exactly `steps` steps, each bracketed by CUDA events on the launching
    stream with an L2 flush before it (outside the events).  Returns per-step ms (numpy)."""
    import torch
    for _ in range(warmup):
        flush_fn(); step_fn()
    torch.cuda.synchronize()
    e0, e1 = _events(steps), _events(steps)
    for i in range(steps):
        flush_fn()
        e0[i].record()
        step_fn()
        e1[i].record()
    torch.cuda.synchronize()
    return np.array([a.elapsed_time(b) for a, b in zip(e0, e1)])


def time_back_to_back(step_fn, steps, warmup):
    import torch
    for _ in range(warmup):
        step_fn()
    torch.cuda.synchronize()
    a, b = _events(2)
    a.record()
    for _ in range(steps):
        step_fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / steps


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2509_14726_b200 import binding as Bd
    from paper_2509_14726_b200 import workloads as W

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank % torch.cuda.device_count())
    dev = torch.device("cuda", torch.cuda.current_device())
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    wl = W.cfg1()
    P = wl.params
    units = P["K"] * P["N"] * P["B"]
    m = Bd.Mppi(P, fast_math=args.fast_math, pipeline=args.pipeline, use_graph=args.graph)
    m.set_track(wl)
    x0 = torch.from_numpy(wl.x0).to(dev); start = torch.from_numpy(wl.start).to(dev)
    u = torch.from_numpy(wl.u_nom).to(dev)
    cost = torch.empty((P["B"], P["K"]), device=dev); w = torch.empty_like(cost)
    flush_buf = torch.empty(L2_FLUSH_BYTES // 4, dtype=torch.float32, device=dev)
    it = [0]

    def step():
        m.step(x0, start, u, wl.seed, it[0], u_new=u, cost=cost, weights=w)     # warm start in place
        it[0] += 1

    def flush():
        flush_buf.fill_(float(it[0] & 7))

    # roofline denominators measured live on this device
    fma_tflops, clock_attr_mhz = Bd.measure_fma_peak(3)
    info = m.info()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(torch.cuda.current_device())
    barrier()
    l0 = m.launch_count()
    sampler.start()
    ms = time_steps(step, flush, args.steps, args.warmup)
    clocks = sampler.finish()
    barrier()
    launches = m.launch_count() - l0 - args.warmup * info["kernels_per_step"]
    my_ms = float(ms.sum())
    max_ms = reduce_max_ms(my_ms, world, dev)
    ms_per_step = max_ms / args.steps
    value = aggregate_value(units * args.steps, world, max_ms)

    line = None
    if rank == 0:
        hot_ms = time_back_to_back(step, args.steps, args.warmup)

        # ---- e2e: the same iteration through mppi_step_host with pinned HOST buffers
        hx0 = torch.from_numpy(wl.x0).pin_memory(); hstart = torch.from_numpy(wl.start).pin_memory()
        hu = torch.from_numpy(wl.u_nom.copy()).pin_memory()
        hout = torch.empty_like(hu).pin_memory()
        n_e2e = min(args.steps, 2000)

        host_call = m.step_host_fn(hx0.numpy(), hstart.numpy(), hu.numpy(), hout.numpy())

        def host_step(i):
            host_call(wl.seed, i)
        for i in range(max(args.warmup, 3)):
            host_step(i)
        lat = np.empty(n_e2e)
        t_all = time.perf_counter()
        for i in range(n_e2e):
            t0 = time.perf_counter()
            host_step(i)
            lat[i] = time.perf_counter() - t0
        t_all = time.perf_counter() - t_all
        h2d = hx0.numel() * 4 + hstart.numel() * 4 + hu.numel() * 4
        d2h = hout.numel() * 4
        # the same call returning everything north_star lists (u_new, per-sample costs, weights): 32 KB more through
        # mapped host memory
        hcost = np.empty((P["B"], P["K"]), np.float32); hw = np.empty_like(hcost)
        host_call_all = m.step_host_fn(hx0.numpy(), hstart.numpy(), hu.numpy(), hout.numpy(), cost=hcost, weights=hw)
        for i in range(max(args.warmup, 3)):
            host_call_all(wl.seed, i)
        lat_all = np.empty(n_e2e)
        for i in range(n_e2e):
            t0 = time.perf_counter()
            host_call_all(wl.seed, i)
            lat_all[i] = time.perf_counter() - t0
        d2h_all = d2h + hcost.nbytes + hw.nbytes

        # ---- configs[1] as stated: 10 warm-started iterations at a fixed x0, as ONE CUDA-graph launch (mppi_optimize)
        mg = Bd.Mppi(P, fast_math=args.fast_math, pipeline=args.pipeline, use_graph=1)
        mg.set_track(wl)
        ug = torch.from_numpy(wl.u_nom).to(dev)
        n_chain = wl.iters

        def chain():
            ug.copy_(u0_dev)
            mg.optimize(x0, start, ug, wl.seed, 0, n_chain, cost=cost, weights=w)
        u0_dev = torch.from_numpy(wl.u_nom).to(dev)
        for _ in range(5):
            chain()
        torch.cuda.synchronize()
        ce0, ce1 = _events(50), _events(50)
        for i in range(50):
            flush()
            ug.copy_(u0_dev)
            ce0[i].record()
            mg.optimize(x0, start, ug, wl.seed, 0, n_chain, cost=cost, weights=w)
            ce1[i].record()
        torch.cuda.synchronize()
        chain_ms = np.array([a.elapsed_time(b) for a, b in zip(ce0, ce1)])
        mg.close()
        # the same chain as plain launches: the pipelined kernel chains them by programmatic dependent launch
        for _ in range(5):
            ug.copy_(u0_dev); m.optimize(x0, start, ug, wl.seed, 0, n_chain, cost=cost, weights=w)
        torch.cuda.synchronize()
        for i in range(50):
            flush()
            ug.copy_(u0_dev)
            ce0[i].record()
            m.optimize(x0, start, ug, wl.seed, 0, n_chain, cost=cost, weights=w)
            ce1[i].record()
        torch.cuda.synchronize()
        chain_pdl_ms = np.array([a.elapsed_time(b) for a, b in zip(ce0, ce1)])

        # ---- the batched configuration (configs[4] shape): where the FP32 roofline is reachable
        wl4 = W.cfg4()
        P4 = wl4.params
        m4 = Bd.Mppi(P4, fast_math=args.fast_math, pipeline=args.pipeline)
        m4.set_track(wl4)
        x4 = torch.from_numpy(wl4.x0).to(dev); s4 = torch.from_numpy(wl4.start).to(dev)
        u4 = torch.from_numpy(wl4.u_nom).to(dev); un4 = torch.empty_like(u4)
        c4 = torch.empty((P4["B"], P4["K"]), device=dev); w4 = torch.empty_like(c4)
        j = [0]

        def step4():
            m4.step(x4, s4, u4, 0, j[0], u_new=un4, cost=c4, weights=w4); j[0] += 1
        ms4 = time_steps(step4, flush, 30, 5)
        units4 = P4["K"] * P4["N"] * P4["B"]

        # configs[4] as stated: the closed loop -- MPPI iteration, plant step, gate advance and shift of
        # the nominal every control step, 500 steps, per-step latency by CUDA events (no L2 flush: the
        # loop's own working set is what a controller sees)
        n_loop = wl4.iters
        x4.copy_(torch.from_numpy(wl4.x0).to(dev)); s4.copy_(torch.from_numpy(wl4.start).to(dev))
        u4.copy_(torch.from_numpy(wl4.u_nom).to(dev))
        ev = _events(n_loop + 1)
        ev[0].record()
        for i in range(n_loop):
            m4.step(x4, s4, u4, wl4.seed, i, u_new=un4, cost=c4, weights=w4)
            m4.sim_step(x4, s4, un4, u_nom_next=u4)
            ev[i + 1].record()
        torch.cuda.synchronize()
        loop_ms = np.array([ev[i].elapsed_time(ev[i + 1]) for i in range(n_loop)])[5:]
        final_height_min = float(x4[:, 2].min().item())
        # untimed replay of the same loop (same seeds: bit-identical) that counts the gate passes of every drone
        x4.copy_(torch.from_numpy(wl4.x0).to(dev)); s4.copy_(torch.from_numpy(wl4.start).to(dev))
        u4.copy_(torch.from_numpy(wl4.u_nom).to(dev))
        passes = torch.zeros(P4["B"], dtype=torch.int64, device=dev)
        for i in range(n_loop):
            before = s4.clone()
            m4.step(x4, s4, u4, wl4.seed, i, u_new=un4, cost=c4, weights=w4)
            m4.sim_step(x4, s4, un4, u_nom_next=u4)
            passes += (s4 != before)
        passes = passes.cpu().numpy()
        flops = FLOPS_PER_SAMPLE_STEP[0]
        sm = info["sm_count"]
        peak_tf = sm * FP32_LANES_PER_SM * 2 * (clocks["sm_max_mhz"] or clock_attr_mhz) * 1e6 / 1e12
        ach = units * flops / (float(ms.mean()) * 1e-3) / 1e12
        ach4 = units4 * flops / (float(ms4.mean()) * 1e-3) / 1e12

        # ---- the instruction mix's own ceiling: issue rates measured on this device x the
        # instruction counts of the scalar gate loop per 32 sample-steps (cuobjdump -sass of rollout_kernel<gate, fast>)
        rates = Bd.measure_issue_rates()
        mix = GATE_LOOP_MIX
        pipes32 = {   # clocks per warp-step (32 sample-steps) each resource of a sub-partition is busy
            "fma_pipe": (mix["ffma_rrr"] * rates["ffma_rrr"] + mix["ffma_const"] * rates["ffma_const"] + mix["fmul"] * rates["fmul"]
                         + mix["fadd"] * rates["fadd"] + mix["philox_half_round"] * rates["philox_half_round"]),
            "alu_pipe": mix["philox_half_round"] * 1.0 + mix["fmnmx"] * rates["fmnmx"],
            "mufu_pipe": mix["mufu"] * rates["mufu"],
            "issue_slots": float(sum(v * (2 if k == "philox_half_round" else 1) for k, v in mix.items())),
        }
        clocks32 = max(pipes32.values())
        ideal32 = 32 * flops / (2 * FP32_LANES_PER_SM / 4)          # 64 flops per clock and sub-partition
        launch_floor_us = Bd.measure_launch_floor(400)

        # ---- cpu_baseline: the oracle as it stands on this host's cores, bounded samples:
        # all online cores and ONE thread on the metric's config, and 5 control steps x 64 drones of configs[4]
        from oracle import oracle as O   # noqa: F401  (cpu_baseline leg only)
        set_oracle_threads(None)
        cpu_rate, cpu_s_iter, cpu_n, cpu_threads = time_oracle(wl, args.cpu_budget, 5000)
        set_oracle_threads(1)
        cpu1_rate, cpu1_s_iter, cpu1_n, _ = time_oracle(wl, min(args.cpu_budget, 5.0), 5000)
        set_oracle_threads(None)
        wl4c = W.cfg4(steps=5)
        trk4 = O.Track(gates=wl4c.gates)
        xo, so, uo = wl4c.x0.astype(np.float64), wl4c.start.copy(), wl4c.u_nom.astype(np.float64)
        O.step(wl4c.params, trk4, xo, so, uo, wl4c.seed, 0, want_diag=False)                   # warm
        t0 = time.perf_counter()
        for i in range(5):
            r4 = O.step(wl4c.params, trk4, xo, so, uo, wl4c.seed, i, want_diag=False)
            xo, so, uo = O.sim_step(wl4c.params, trk4, xo, so, r4["u_new"])
        cpu4_s = (time.perf_counter() - t0) / 5

        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl.name, "K": P["K"], "N": P["N"], "B": P["B"], "objective": "gate",
                       "dt": P["dt"], "sigma": P["sigma"], "lambda": P["lambda"], "warm_start": "in place, iter = step",
                       "l2": "flushed between timed iterations (256 MiB write outside the events)",
                       "pipeline": "fused" if args.pipeline == 0 else "two_pass", "fast_math": args.fast_math,
                       "cuda_graph": bool(args.graph), "block_threads": info["block_threads"],
                       "kernel": KERNEL_SYMBOL.get(kernel_label(info, P), "rollout"),
                       "grid_blocks": info["grid_blocks"], "replicas": world},
            "clocks": clocks,
            "latency_us": {"p50": float(np.median(ms) * 1e3), "p99": float(np.percentile(ms, 99) * 1e3),
                           "mean": float(ms.mean() * 1e3), "back_to_back_no_flush": hot_ms * 1e3},
            "e2e": {"value": units * n_e2e / t_all, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                    "d2h_bytes_per_step": int(d2h), "latency_us_p50": float(np.median(lat) * 1e6),
                    "latency_us_p99": float(np.percentile(lat, 99) * 1e6),
                    "timer": "host perf_counter around mppi_step_host returning u_new only (cost / weights pointers NULL): one packed H2D copy from pinned memory, the kernel, u_new written by the kernel into mapped host memory, completion flag polled by the host",
                    "with_cost_and_weights": {"value": units * n_e2e / float(lat_all.sum()), "unit": UNIT, "d2h_bytes_per_step": int(d2h_all),
                                              "latency_us_p50": float(np.median(lat_all) * 1e6), "latency_us_p99": float(np.percentile(lat_all, 99) * 1e6),
                                              "timer": "the same call returning u_new, the K costs and the K weights (what north_star's mppi_step returns), all written by the kernel into mapped host memory"}},
            "optimize_chain": {"iterations": int(n_chain), "us_per_chain_p50": float(np.median(chain_ms) * 1e3),
                               "us_per_iteration": float(np.median(chain_ms) * 1e3 / n_chain),
                               "programmatic_dependent_launch": {"us_per_chain_p50": float(np.median(chain_pdl_ms) * 1e3),
                                                                 "us_per_iteration": float(np.median(chain_pdl_ms) * 1e3 / n_chain),
                                                                 "what": "the same chain as plain stream launches (use_graph = 0): iteration i + 1 is launched with the programmatic-stream-serialization attribute, starts while iteration i combines, and waits (griddepcontrol.wait) before it reads the nominal"},
                               "what": "configs[1] as stated: 10 warm-started iterations at a fixed x0 through mppi_optimize, one CUDA-graph launch per chain (use_graph = 1), CUDA events around the launch, L2 flushed before each chain"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf,
                         # dram__bytes_read.sum + dram__bytes_write.sum of this kernel, per launch, from the
                         # ncu --set full capture summarised in profiles/README_r01e.md (not measured live)
                         "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(kernel_label(info, P), (None, None))[0] if args.pipeline == 0 else None,
                         "kernel": f"the iteration's single kernel ({kernel_label(info, P)} rollout + cost + fused softmax update)" if args.pipeline == 0 else "rollout kernel of the two-pass pipeline",
                         "flops_per_sample_step": flops, "units_per_launch": units,
                         "peak_how": f"{sm} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 x clocks.max.sm (B200_PROFILING.md)",
                         "peak_measured_ffma_tflops": fma_tflops, "frac_of_measured_ffma": ach / fma_tflops,
                         "regs_per_thread": info["regs_per_thread"], "spill_bytes": info["local_bytes_per_thread"],
                         "traffic_source": (f"{NCU_DRAM_BYTES_PER_LAUNCH.get(kernel_label(info, P), (None, 'no capture'))[1]} (ncu --set full capture of this kernel, dram__bytes_read.sum + dram__bytes_write.sum per launch; not measured in this run)") if args.pipeline == 0 else None,
                         "note": "K=4096 rollouts of 50 dependent steps on 148 SMs: latency-bound by construction (the time-parallel kernel splits every rollout over 16 lanes along the horizon); see 'batched' for the FP32 roofline"},
            "batched": {"workload": wl4.name, "K": P4["K"], "N": P4["N"], "B": P4["B"],
                        "value": units4 / (float(ms4.mean()) * 1e-3), "unit": UNIT, "ms_per_step": float(ms4.mean()),
                        "roofline": {"bound": "alu", "achieved": ach4, "peak": peak_tf, "unit": "TFLOP/s",
                                     "frac": ach4 / peak_tf, "frac_of_measured_ffma": ach4 / fma_tflops,
                                     "mix_ceiling": {"issue_cycles_per_warp_instr": rates, "gate_loop_instr_per_32_sample_steps": GATE_LOOP_MIX,
                                                     "busy_clocks_per_32_sample_steps": pipes32, "clocks_per_32_sample_steps": clocks32,
                                                     "clocks_at_fp32_peak": ideal32, "frac_of_peak": ideal32 / clocks32,
                                                     "how": "per resource of a sub-partition: sum over the loop's instruction classes of count x cycles per warp-instruction measured by mppi_measure_issue_rates (FFMA / FMUL / FADD and the 32x32->64 multiply of a Philox half-round occupy the FMA pipe, LOP3 / FMNMX the ALU pipe, MUFU its own; one issue slot per instruction); the busiest resource bounds the loop, and 32 x flops_per_sample_step / 64 flops per clock is the time at the FP32 peak -- their ratio is the fraction of the peak this instruction mix can reach however it is scheduled"}},
                        "closed_loop": {"control_steps": n_loop, "value": units4 / (float(loop_ms.mean()) * 1e-3),
                                        "unit": UNIT, "latency_us_p50": float(np.median(loop_ms) * 1e3),
                                        "latency_us_p99": float(np.percentile(loop_ms, 99) * 1e3),
                                        "gate_passes_per_drone": {"min": int(passes.min()), "median": float(np.median(passes)), "max": int(passes.max())},
                                        "final_height_min_m": final_height_min,
                                        "note": "configs[4] as stated (sigma 1.5 N, lambda 0.5): the drones pass at most one gate and then lose height, so most timed control steps roll out from states below the track; the work per step is the same (checked against the oracle at steps 0, 50, .., 499: tests/test_parity_gpu.py::test_cfg4_closed_loop_teacher_forced)",
                                        "what": "mppi_step + mppi_sim_step per control step, 64 drones, CUDA events"}},
            "cpu_baseline": {"value": cpu_rate, "unit": UNIT, "cores": cpu_threads, "kind": "oracle", "cpu": cpu_model(),
                             "sample": f"{cpu_n} full iterations of {wl.name} ({cpu_s_iter * 1e3:.1f} ms each), float64, OpenMP over samples",
                             "single_thread": {"value": cpu1_rate, "unit": UNIT, "cores": 1,
                                               "sample": f"{cpu1_n} full iterations of {wl.name} ({cpu1_s_iter * 1e3:.1f} ms each)"},
                             "cfg4": {"value": units4 / cpu4_s, "unit": UNIT, "cores": cpu_threads, "s_per_control_step": cpu4_s,
                                      "extrapolated_s_for_500_control_steps": 500 * cpu4_s,
                                      "sample": "5 control steps x 64 drones of configs[4] (iteration + plant step), timed in full; the 500-step figure is a linear extrapolation"}},
            "launch_floor_us": launch_floor_us,
        }
        m4.close()
    m.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)
    return 0


def run_survey(args):
    """One iteration of every workload, alone and x64: device time per iteration (CUDA events, L2 flushed
    between iterations), sample-steps/s, the kernel that ran.  Prints a markdown table."""
    import torch
    from paper_2509_14726_b200 import binding as Bd
    from paper_2509_14726_b200 import workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --survey: no CUDA device")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    flush_buf = torch.empty(L2_FLUSH_BYTES // 4, dtype=torch.float32, device=dev)
    names = ["cfg0", "cfg1", "cfg2", "cfg3", "gate_paper", "rate_gate_paper", "rate_track", "contour_paper",
             "table1_gate", "table1_contour"]
    print("| workload | objective | input model | K | N | B | kernel | launches / iteration | us / iteration | sample-steps/s |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for name in ([args.only] if args.only else names):
        for B in ((args.batch,) if args.batch else (1, 64)):
            wl = W.ALL[name]()
            if B > 1:
                wl = W.replicate(wl, B, 0.3)
            P = wl.params
            m = Bd.Mppi(P, fast_math=args.fast_math, variant=args.variant, pipeline=args.pipeline)
            m.set_track(wl)
            x0 = torch.from_numpy(wl.x0).to(dev); start = torch.from_numpy(wl.start).to(dev)
            u = torch.from_numpy(wl.u_nom).to(dev); un = torch.empty_like(u)
            cost = torch.empty((P["B"], P["K"]), device=dev); w = torch.empty_like(cost)
            it = [0]

            def step():
                m.step(x0, start, u, wl.seed, it[0], u_new=un, cost=cost, weights=w); it[0] += 1
            ms = time_steps(step, lambda: flush_buf.fill_(float(it[0] & 7)), 40 if B > 1 else 200, 5)
            info = m.info()
            k = kernel_label(info, P)
            units = P["K"] * P["N"] * P["B"]
            print(f"| {name} | {P['objective']} | {P.get('input_model', 0)} | {P['K']} | {P['N']} | {P['B']} | {k} "
                  f"({info['block_threads']} thr x {info['grid_blocks']} blocks, {info['regs_per_thread']} regs) | "
                  f"{info['kernels_per_step']} | {float(np.median(ms)) * 1e3:.1f} | {units / (float(ms.mean()) * 1e-3):.3g} |", flush=True)
            m.close()
    return 0


def _time_workload(Bd, wl, dev, flush_buf, steps, warmup, **opts):
    """One context, `steps` timed iterations (CUDA events, L2 flushed between them).  Returns (per-step ms, info, ESS
    of the last iteration's weights per controller)."""
    import torch
    P = wl.params
    m = Bd.Mppi(P, **opts)
    m.set_track(wl)
    x0 = torch.from_numpy(wl.x0).to(dev); start = torch.from_numpy(wl.start).to(dev)
    u = torch.from_numpy(wl.u_nom).to(dev); un = torch.empty_like(u)
    cost = torch.empty((P["B"], P["K"]), device=dev); w = torch.empty_like(cost)
    it = [0]

    def step():
        m.step(x0, start, u, wl.seed, it[0], u_new=un, cost=cost, weights=w); it[0] += 1
    ms = time_steps(step, lambda: flush_buf.fill_(float(it[0] & 7)), steps, warmup)
    info = m.info()
    ess = (1.0 / (w.double() ** 2).sum(-1)).cpu().numpy()
    J = cost.cpu().numpy()
    m.close()
    return ms, info, ess, J


VARIANT_NAMES = {0: "AUTO", 1: "scalar", 2: "latency", 3: "packed", 4: "pipelined", 5: "time-parallel"}


def run_sweep(args):
    """Two tables the headline numbers do not cover:
    (i)  the batch sizes between the lone controller and configs[4]: B in {1..64} at K=4096, N=50, gate objective,
         for every rollout kernel AUTO could pick, and AUTO itself;
    (ii) the configs[4] shape at a MIXING temperature (lambda = 0.25 std(J): hundreds of samples carry weight, so
         the fused update re-derives the whole noise stream) for the fused and the two-pass pipeline.
    Device time per iteration by CUDA events, L2 flushed between iterations."""
    import torch
    from paper_2509_14726_b200 import binding as Bd
    from paper_2509_14726_b200 import workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sweep: no CUDA device")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    flush_buf = torch.empty(L2_FLUSH_BYTES // 4, dtype=torch.float32, device=dev)
    K = args.sweep_K
    base = {"gate": lambda B: W.cfg4(K=K, B=B), "track": lambda B: W.replicate(W.cfg2(K=K), B, 0.3),
            "contour": lambda B: W.replicate(W.cfg3(K=2 * K), B, 0.3)}
    print(f"## (i) batch sweep at K = {K} (contouring: {2 * K}), N = 50, us per iteration (median of 60; AUTO's choice in brackets)\n")
    for obj in args.sweep_objectives.split(","):
        print(f"objective: {obj}\n")
        print("| B | " + " | ".join(VARIANT_NAMES[v] for v in (5, 4, 2, 3, 1, 0)) + " | AUTO vs best |")
        print("|---|" + "---|" * 7)
        for B in [int(b) for b in args.sweep_batches.split(',')]:
            wl = base[obj](B)
            row, best = [], None
            for v in (5, 4, 2, 3, 1, 0):
                try:
                    ms, info, _, _ = _time_workload(Bd, wl, dev, flush_buf, 60, 5, fast_math=args.fast_math, variant=v)
                    t = float(np.median(ms)) * 1e3
                    tag = f"{t:.1f}"
                    if v == 0:
                        k = kernel_label(info)
                        tag += f" [{k}, {info['block_threads']} thr x {info['grid_blocks']}]"
                        row.append(tag)
                        row.append(f"{t / best:.2f}x")
                        continue
                    best = t if best is None else min(best, t)
                    row.append(tag)
                except Bd.MppiError as e:
                    row.append("n/a")
            print(f"| {B} | " + " | ".join(row) + " |", flush=True)
        print()
    if args.sweep_K != 4096:
        return
    print("## (ii) configs[4] shape (K=4096, N=50, B=64, gate), one-hot vs mixing weights, us per iteration (median of 40)\n")
    print("| weights | lambda | ESS (median over controllers) | fused packed | fused scalar | two-pass packed (rollout + reduce) | two-pass scalar | fused packed, dU also stored |")
    print("|---|---|---|---|---|---|---|---|")
    wl = W.cfg4()
    _, _, _, J = _time_workload(Bd, wl, dev, flush_buf, 1, 3, fast_math=args.fast_math)
    lam_mix = float(np.float32(0.25 * np.median(J.std(-1))))
    for label, lam in (("configs[4] as stated", wl.params["lambda"]), ("mixing, 0.25 std(J)", lam_mix), ("flat, 4 std(J)", 16 * lam_mix)):
        wl = W.cfg4(); wl.params["lambda"] = lam
        cells, ess_med = [], None
        for pipe, v, sn in ((0, 3, 0), (0, 1, 0), (1, 3, 0), (1, 1, 0), (0, 3, 1)):
            ms, info, ess, _ = _time_workload(Bd, wl, dev, flush_buf, 40, 5, fast_math=args.fast_math, variant=v, pipeline=pipe, store_noise=sn)
            ess_med = float(np.median(ess))
            cells.append(f"{float(np.median(ms)) * 1e3:.1f}")
        print(f"| {label} | {lam:.4g} | {ess_med:.1f} | " + " | ".join(cells) + " |", flush=True)
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--pipeline", type=int, default=0, help="0 fused (default), 1 two-pass")
    ap.add_argument("--fast-math", dest="fast_math", type=int, default=1)
    ap.add_argument("--graph", type=int, default=0)
    ap.add_argument("--cpu-budget", dest="cpu_budget", type=float, default=10.0)
    ap.add_argument("--survey", action="store_true", help="time one iteration of every workload (table, one GPU)")
    ap.add_argument("--sweep", action="store_true", help="batch-size sweep over the rollout kernels and the mixing-weight regime (tables, one GPU)")
    ap.add_argument("--sweep-objectives", dest="sweep_objectives", default="gate", help="--sweep: comma list of gate,track,contour")
    ap.add_argument("--sweep-batches", dest="sweep_batches", default="1,2,3,4,6,8,12,16,32,64")
    ap.add_argument("--sweep-K", dest="sweep_K", type=int, default=4096, help="--sweep: samples per controller (table (i) only when not 4096)")
    ap.add_argument("--only", default=None, help="--survey: this workload only (a key of workloads.ALL)")
    ap.add_argument("--batch", type=int, default=0, help="--survey: this number of controllers only")
    ap.add_argument("--variant", type=int, default=0, help="--survey: mppi_variant (0 AUTO, 1 THROUGHPUT, 2 LATENCY, 3 PACKED, 4 PIPELINED)")
    args = ap.parse_args(argv)
    if args.survey:
        return run_survey(args)
    if args.sweep:
        return run_sweep(args)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
