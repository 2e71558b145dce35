#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native MPMI-SC tick (BASELINE.json metric:
"rollout sample-steps/sec and p50/p99 per-tick latency at N=10k and 1M; % FP32 peak").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl reference]

One "step" is one whole control tick: sample N candidates -> lift ->
H-step rollout with per-step safe test -> argmin selection -> result, on one batch of synthetic
input (a fresh x0, u_user and Philox tick per step).  Default workload: C4 at N = 2^20, H = 100
(BASELINE.json configs[3], the configuration the throughput half of the metric is quoted on).
The rest of the metric rides on the same JSON line under "extra" (N = 1 only): the scale sweep
N = 2^14 .. 2^20, C5 with a roofline of its own, the paper-scale latencies (C1, C2, C3), the two
HBM-bound trajectory dumps and the comparison rows (FP32-only, bare tensor-core, noise, re-lift, affine) -- each with its own clock record.

value    = executed sample-steps/s with inputs resident in HBM (mpmi_step_device), CUDA-event timed
e2e      = the same metric through mpmi_step_sync with HOST buffers (H2D + D2H inside the region)
roofline = the dominant kernel, timed by CUDA events around its launches (mpmi_profile_enable), against
           the FP32 FMA peak ("alu") or the 3xTF32 tensor peak ("tensor"); DESIGN.md section 6
cpu_baseline = the FP64 oracle, as it stands, on this box's host cores (bounded sample), and on one thread

One "sample-step" = one evaluation of z <- K z + B u followed by isSafe; candidate i executes
min(steps_i + 1, H) of them (Algorithm 2 l.4 stops at the first violation).  The nominal N*H count
is reported beside it.

--gpus N with N > 1 and no WORLD_SIZE in the environment starts the N ranks itself (torch.distributed.run,
127.0.0.1); under torchrun it is one of the ranks.  Candidates are sharded (weak scaling: 2^20 per GPU)
with one 24-byte exchange per tick.
"""
import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # 74.45: SMs x FP32 lanes x 2 flop x max SM clock
# one M128 N128 K8 kind::tf32 tcgen05.mma per 64 clk and SM (N = 32: 16 clk), measured:
# 2*128*128*8 / 64 = 4096 TF32 flop per clk and SM
TF32_PEAK_TFLOPS = 148 * 4096 * 1.965e9 / 1e12         # 1191
KERNEL_NAMES = {1: "rollout_reg_kernel", 2: "rollout_tile_kernel", 3: "rollout_lat_kernel", 4: "rollout_tc_kernel",
                5: "rollout_relift_kernel", 6: "rollout_affine_kernel"}


def _flop_per_sample_step(w):
    if getattr(w, "model_kind", 0) == 1:                # re-lift model: n physical rows + the lift itself (cos / sin counted as 1)
        lift = 3.0 * w.d if w.lift_kind == 0 else (2.0 * w.n + 2.0) * (w.d - w.n)
        return 2.0 * w.n * (w.d + w.m) + lift
    return 2.0 * w.d * (w.d + w.m)                      # dense K and B, nothing discounted


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    return json.load(open(p)) if os.path.exists(p) else {}


class ClockSampler(threading.Thread):
    """nvidia-smi style clock / throttle-reason samples DURING the timed region (NVML)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag = index, [], False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        while not self.stop_flag:
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                mx = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
                rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                self.samples.append((sm, mx, rs))
            except Exception:
                pass
            time.sleep(0.004)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        nv = self.nv
        names = {nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap", nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksEventReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        seen = set()
        for _, _, rs in self.samples:
            for bit, name in names.items():
                if rs & bit:
                    seen.add(name)
        sm = sorted(s[0] for s in self.samples)
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": self.samples[0][1], "reasons": sorted(seen),
                "samples": len(sm)}


class clocked:
    """with clocked(dev) as c: ... ; c.summary -- the clock record of one timed region"""

    def __init__(self, index):
        self.s = ClockSampler(index)

    def __enter__(self):
        self.s.start()
        return self

    def __exit__(self, *exc):
        self.s.stop_flag = True
        self.s.join(timeout=1.0)
        self.summary = self.s.summary()


def _variant(args, mp):
    V = mp.mpmi
    return ((V.VARIANT_NO_TENSOR if args.no_tensor else 0) | (V.VARIANT_AFFINE if args.affine else 0) | (V.VARIANT_NO_PREDICT if args.no_predict else 0)
            | (V.VARIANT_TENSOR32 if args.tensor32 else 0) | (V.VARIANT_TC_UNVERIFIED if args.unverified else 0))


def _percentiles(v):
    v = np.sort(np.asarray(v, dtype=np.float64))
    return float(v[len(v) // 2]), float(v[min(len(v) - 1, int(0.99 * len(v)))])


def _workload_string(args, w, n_per):
    """the one description of the timed workload, printed by both arms (so that their configs compare equal)"""
    return (f"{args.workload}: n={w.n} m={w.m} d={w.d} N={n_per}/GPU (+1 user slot) H={w.H}, Philox/grid sampler, "
            f"calibrated 40% safe (DESIGN.md section 4)"
            + (f", safe set scaled x{args.bounds_scale}" if args.bounds_scale != 1.0 else "")
            + (f", prediction noise sigma={args.noise}" if args.noise else "")
            + (", re-lift model" if args.relift else ""))


def _set_oracle_threads(n):
    """the oracle's only OpenMP pragma is the paper's parallel-for; its team size is set through libgomp"""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def _time_oracle(w, x0s, uus, ticks, first, budget_s, max_ticks, n_s):
    from oracle import oracle as O
    o = O.Oracle(w, N=n_s)
    o.step(x0s[0], uus[0], 0)
    ne, t0, nt = 0, time.perf_counter(), 0
    while time.perf_counter() - t0 < budget_s and nt < max_ticks:
        ne += o.step(x0s[first + nt], uus[first + nt], int(ticks[first + nt]))["n_exec"]; nt += 1
    dt = time.perf_counter() - t0
    return ne / dt, nt, O.num_threads()


def run_reference(args):
    """--impl reference: the FP64 oracle as it stands, on the host cores, same config / metric / unit.
    Under torchrun rank 0 alone runs and prints; the other ranks exit 0 without work."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return
    import workloads as W
    from oracle import oracle as O
    w1 = W.make(args.workload, N=args.N)
    n_per = w1.N
    w = W.make(args.workload, N=n_per * world)                  # the same global candidate set as our arm at this rank count
    if args.bounds_scale != 1.0:
        w = W.generate.scaled_bounds(w, args.bounds_scale)
    w.noise_sigma = args.noise
    w.model_kind = 1 if args.relift else 0
    x0s, uus, ticks = W.tick_inputs(w, args.warmup + args.steps)
    # bounded sample: the first n_ref candidates of the same workload, sized from one probe tick
    n_ref = min(w.N, 1 << 14)
    t0 = time.perf_counter()
    r = O.Oracle(w, N=n_ref).step(x0s[0], uus[0], 0)
    rate = r["n_exec"] / (time.perf_counter() - t0)
    budget_s = 150.0 / max(1, args.steps + args.warmup)
    n_ref = int(min(w.N, max(1 << 12, rate * budget_s / (w.H * 0.7))))
    o = O.Oracle(w, N=n_ref)
    for t in range(args.warmup):
        o.step(x0s[t], uus[t], int(ticks[t]))
    n_exec, t0 = 0, time.perf_counter()
    for t in range(args.warmup, args.warmup + args.steps):
        n_exec += o.step(x0s[t], uus[t], int(ticks[t]))["n_exec"]
    dt = time.perf_counter() - t0
    val = n_exec / dt
    sample = f"first {n_ref} of {w.N} candidates (+ user slot) per tick, {args.steps} ticks, H={w.H}"
    print(json.dumps({
        "impl": "reference", "metric": "rollout sample-steps/s", "value": val, "unit": "sample-steps/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _workload_string(args, w, n_per), "sample": sample},
        "cpu_baseline": {"value": val, "unit": "sample-steps/s", "cores": O.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "sample-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ----------------------------------------------------------------------------------------------------------------------
def measure_ticks(mp, ctx, w, x0s, uus, ticks, K_, W_, flush, stream, tick_fn=None, dist=None):
    """W_ warm-up + K_ timed device-resident ticks (CUDA events on `stream`, L2 flushed between them, the dominant
    kernel timed separately through mpmi_profile_*).  Returns a dict of raw measurements."""
    import torch
    dX0 = torch.as_tensor(x0s).cuda().contiguous()
    dUU = torch.as_tensor(uus).cuda().contiguous()
    dRes = torch.zeros((W_ + K_, 56), dtype=torch.uint8, device="cuda")
    if tick_fn is None:
        def tick_fn(t):
            ctx.step_device(dX0[t].data_ptr(), dUU[t].data_ptr(), int(ticks[t]), stream, dRes[t].data_ptr())
    else:
        inner = tick_fn

        def tick_fn(t):
            inner(t, dX0, dUU, dRes)
    for t in range(W_):
        tick_fn(t)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    ctx.profile_enable(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K_)]
    torch.cuda.synchronize()
    for i in range(K_):
        flush.fill_(i & 0xFF)                                  # L2 flush between timed iterations (untimed)
        ev[i][0].record()
        tick_fn(W_ + i)
        ev[i][1].record()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    kern_ms, second_ms = ctx.profile_read(64)
    ctx.profile_enable(False)
    step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    res = np.frombuffer(dRes.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)
    return {"step_ms": step_ms, "kern_ms": kern_ms[-K_:], "second_ms": second_ms[-K_:], "res": res[W_:],
            "n_exec": int(res["n_exec"][W_:].sum())}


def host_latency(ctx, xs, us, ticks, stream, warm=50):
    """wall time of mpmi_step_sync (host buffers in, host result out) per tick -> (p50, p99) in microseconds"""
    for t in range(min(warm, len(xs))):
        ctx.step_sync(xs[t], us[t], int(ticks[t]), stream)
    wall = []
    for t in range(len(xs)):
        t0 = time.perf_counter()
        ctx.step_sync(xs[t], us[t], int(ticks[t]), stream)
        wall.append(time.perf_counter() - t0)
    p50, p99 = _percentiles(wall)
    return 1e6 * p50, 1e6 * p99


def _traffic(key):
    """dram bytes per launch of the dominant kernel, from the ncu --set full capture named in profiles/roofline_traffic.md
    (bench.py cannot read DRAM counters itself)"""
    tj = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if os.path.exists(tj):
        for line in open(tj).read().splitlines()[1:]:
            f = line.split(",")
            if f and f[0] == key:
                return int(f[2]), f[1] + (": " + f[4] if len(f) > 4 else "")
    return None, None


def make_roofline(info, w, m, world=1, key=None):
    """roofline of the dominant kernel of a tick: algorithmic flop (2 d (d + m) per executed sample-step)
    / the kernel's own event-timed duration."""
    K_ = len(m["step_ms"])
    flop = _flop_per_sample_step(w) if info["variant"] != 6 else 2.0 * w.n * w.m      # affine path: n*m FMAs per sample-step
    # (the profile ring holds the last 64 ticks: scale their mean to the K_ timed ticks)
    total_ms, kern_ms, second_ms = float(m["step_ms"].sum()), float(m["kern_ms"].mean()) * K_, float(m["second_ms"].mean()) * K_
    work = m["n_exec"] / world * flop                                            # per GPU, all timed ticks
    traffic, tsrc = _traffic(key or "")
    nominal = float(w.N + 1) / world * w.H * K_ * flop
    common = {"unit": "TFLOP/s", "traffic": traffic, "traffic_source": tsrc,
              "kernel_ms_per_tick": kern_ms / K_, "kernel_share_of_tick": kern_ms / total_ms,
              "achieved_whole_tick": work / (total_ms * 1e-3) / 1e12,
              "flop_per_sample_step": flop, "launches_per_tick": info["launches_per_tick"]}
    if info["variant"] == 4:
        # 3xTF32 split contraction on the tcgen05 tensor cores (rollout_tc.cuh): every algorithmic flop costs three TF32
        # tensor flops.  Peak: the measured MMA rate (one M128 N128 K8 kind::tf32 MMA per 64 clk and SM) at the max SM clock.
        peak = TF32_PEAK_TFLOPS / 3.0
        bf16 = float(_peaks().get("bf16_tflops", 1590.0))
        achieved = work / (kern_ms * 1e-3) / 1e12              # the first pass rolls EVERY candidate (the second pass re-rolls a few)
        r = {"bound": "tensor", "achieved": achieved, "peak": peak, "frac": achieved / peak,
             "peak_source": "derived: 148 SM x 4096 TF32 flop/clk/SM (one M128 N128 K8 kind::tf32 tcgen05.mma per 64 clk, measured; "
                            "DESIGN.md section 6) x 1.965 GHz / 3 (3xTF32 split products per algorithmic flop)",
             "peak_prescribed": bf16 * (1.1 / 2.25) / 3.0,
             "peak_prescribed_source": ("MEASURED_PEAKS.json bf16_tflops (burst)" if _peaks() else "fallback 1590 TFLOP/s bf16")
                                       + " x 1.1/2.25 (nominal tf32:bf16) / 3",
             "kernel": "rollout_tc_kernel (first pass of the verified tick)" if info["launches_per_tick"] > 4 or second_ms > 0 else "rollout_tc_kernel",
             "dtype": "3xTF32 (fp32 accumulate)",
             "tensor_tflops_executed": achieved * 3.0 * (info["d_pad"] + 8.0) / (w.d + w.m),     # K padded to d_pad + one 8-wide input block
             "fp32_alu_frac_whole_tick": work / (total_ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS,
             "second_pass": {"kernel": "rollout_split_kernel / rollout_reg_kernel (FP32, deferred candidates)" if info["d_pad"] <= 32 else "rollout_tile_kernel (FP32, deferred candidates)",
                             "ms_per_tick": second_ms / K_, "share_of_tick": second_ms / total_ms,
                             "deferred_fraction": info.get("deferred_fraction")}}
    else:
        achieved = work / (kern_ms * 1e-3) / 1e12
        r = {"bound": "alu", "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "frac": achieved / FP32_PEAK_TFLOPS,
             "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md section 6; no FP32 ALU figure in MEASURED_PEAKS.json)",
             "kernel": KERNEL_NAMES.get(info["variant"], "?"),
             "nominal_frac_whole_tick": nominal / (total_ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS}
    r.update(common)
    return r


def extra_sweep(mp, args, local, flush, stream):
    """BASELINE.json configs[3]: the C4 model at N = 2^14 .. 2^20, device-timed tick, host p50 / p99, fraction of FP32 peak"""
    import workloads as W
    rows = []
    K_, W_ = 20, 5
    with clocked(local) as ck:
        for lg in range(14, 21):
            w = W.make("C4", N=1 << lg)
            x0s, uus, ticks = W.tick_inputs(w, W_ + K_)
            ctx = mp.Context(w, device=local)
            m = measure_ticks(mp, ctx, w, x0s, uus, ticks, K_, W_, flush, stream)
            xs = [np.ascontiguousarray(x) for x in x0s]; us = [np.ascontiguousarray(u) for u in uus]
            p50, p99 = host_latency(ctx, xs, us, ticks, stream, warm=5)
            info = ctx.info()
            ms = float(m["step_ms"].sum())
            rows.append({"N": 1 << lg, "tick_ms": ms / K_, "host_p50_us": p50, "host_p99_us": p99,
                         "sample_steps_per_s": m["n_exec"] / (ms * 1e-3),
                         "nominal_sample_steps_per_s": float(w.N + 1) * w.H * K_ / (ms * 1e-3),
                         "fp32_frac_whole_tick": m["n_exec"] * _flop_per_sample_step(w) / (ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS,
                         "kernel": KERNEL_NAMES[info["variant"]], "launches_per_tick": info["launches_per_tick"]})
            ctx.close()
    return {"workload": "C4 model (n=6 m=2 d=32 H=100, Philox), N = 2^14 .. 2^20 (+1 user slot), 20 timed ticks each, L2 flushed between ticks",
            "rows": rows, "clocks": ck.summary}


def extra_c5(mp, args, local, flush, stream):
    import workloads as W
    K_, W_ = 10, 4
    w = W.make("C5")
    x0s, uus, ticks = W.tick_inputs(w, W_ + K_)
    ctx = mp.Context(w, device=local)
    with clocked(local) as ck:
        m = measure_ticks(mp, ctx, w, x0s, uus, ticks, K_, W_, flush, stream)
        xs = [np.ascontiguousarray(x) for x in x0s]; us = [np.ascontiguousarray(u) for u in uus]
        p50, p99 = host_latency(ctx, xs, us, ticks, stream, warm=4)
    info = ctx.info()
    info["deferred_fraction"] = info["reserved"] / float(w.N + 1)
    ms = float(m["step_ms"].sum())
    out = {"workload": "C5: n=8 m=3 d=128 N=262144 (+1 user slot) H=100, Philox, calibrated 40% safe; verified 3xTF32 tcgen05 tick",
           "tick_ms": ms / K_, "host_p50_us": p50, "host_p99_us": p99, "sample_steps_per_s": m["n_exec"] / (ms * 1e-3),
           "roofline": make_roofline(info, w, m, key="C5"), "clocks": ck.summary}
    ctx.close()
    return out


def extra_variants(mp, args, local, flush, stream):
    """the comparison rows of BASELINE.md's table (own metrics, not the headline): FP32-only ticks, the bare tensor-core kernel,
    prediction noise, the re-lift model and the affine-in-u fast path -- a few ticks each, device-timed"""
    import workloads as W
    V = mp.mpmi
    K_, W_ = 6, 3
    rows = [("C4_fp32", "C4", V.VARIANT_NO_TENSOR, 0.0, 0), ("C4_bare_tensor_core", "C4", V.VARIANT_TC_UNVERIFIED, 0.0, 0),
            ("C5_fp32", "C5", V.VARIANT_NO_TENSOR, 0.0, 0), ("C5_bare_tensor_core", "C5", V.VARIANT_TC_UNVERIFIED, 0.0, 0),
            ("C4_noise_0.02", "C4", 0, 0.02, 0), ("C5_noise_0.01", "C5", 0, 0.01, 0), ("C4_relift", "C4", 0, 0.0, 1),
            ("C4_affine", "C4", V.VARIANT_AFFINE, 0.0, 0), ("C5_affine", "C5", V.VARIANT_AFFINE, 0.0, 0)]
    out = {}
    with clocked(local) as ck:
        for key, name, variant, sigma, relift in rows:
            w = W.make(name)
            w.noise_sigma = sigma; w.model_kind = relift
            x0s, uus, ticks = W.tick_inputs(w, W_ + K_)
            ctx = mp.Context(w, device=local, variant=variant)
            m = measure_ticks(mp, ctx, w, x0s, uus, ticks, K_, W_, flush, stream)
            info = ctx.info()
            ms = float(m["step_ms"].sum())
            out[key] = {"tick_ms": ms / K_, "sample_steps_per_s": m["n_exec"] / (ms * 1e-3), "kernel": KERNEL_NAMES.get(info["variant"], "?"),
                        "launches_per_tick": info["launches_per_tick"]}
            ctx.close()
    out["clocks"] = ck.summary
    return out


def extra_latency(mp, args, local, stream):
    """paper-scale ticks (N ~ 1e4): host p50 / p99 of mpmi_step_sync; C2 replays its 1,000 stored closed-loop ticks"""
    import workloads as W
    out = {}
    with clocked(local) as ck:
        w2 = W.make("C2")
        seq = np.loadtxt(W.generate.C2_SEQUENCE, comments="#")
        c2 = mp.Context(w2, device=local)
        xs = [np.ascontiguousarray(row[1:5], dtype=np.float32) for row in seq]
        us = [np.ascontiguousarray(row[5:6], dtype=np.float32) for row in seq]
        p50, p99 = host_latency(c2, xs, us, np.arange(len(seq)), stream)
        out["C2_N10000"] = {"host_p50_us": p50, "host_p99_us": p99, "ticks": len(seq)}
        c2.close()
        for name in ("C1", "C3"):
            w = W.make(name)
            x0s, uus, ticks = W.tick_inputs(w, 400)
            c = mp.Context(w, device=local)
            xs = [np.ascontiguousarray(x) for x in x0s]; us = [np.ascontiguousarray(u) for u in uus]
            p50, p99 = host_latency(c, xs, us, ticks, stream)
            out[f"{name}_N{w.N}"] = {"host_p50_us": p50, "host_p99_us": p99, "ticks": len(xs)}
            c.close()
    out["clocks"] = ck.summary
    return out


def measure_dump(mp, ctx, w, x0s, ticks, K_, W_, kind_name, stream):
    import torch
    N, H = w.N, w.H
    J = w.d if kind_name == "lifted" else w.n
    kind = mp.DUMP_LIFTED if kind_name == "lifted" else mp.DUMP_PHYS
    traj = torch.empty((H, J, N), dtype=torch.float32, device="cuda")
    steps = torch.empty(N, dtype=torch.int32, device="cuda")
    dX0 = torch.as_tensor(x0s).cuda().contiguous()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K_)]
    for t in range(W_ + K_):
        if t >= W_:
            ev[t - W_][0].record()
        ctx.rollout_batch(0, dX0[t].data_ptr(), 1, N, H, kind, traj.data_ptr(), steps.data_ptr(), 0, int(ticks[t]), stream)
        if t >= W_:
            ev[t - W_][1].record()
    torch.cuda.synchronize()
    ms = np.array([a.elapsed_time(b) for a, b in ev])
    nbytes = float(N) * H * J * 4 + 4.0 * N
    peaks = _peaks()
    peak = float(peaks.get("hbm_gbs", 6650.0))
    gbs = nbytes / (ms.mean() * 1e-3) / 1e9
    n_exec = int(torch.clamp(steps.to(torch.int64) + 1, max=H).sum().item())
    del traj
    torch.cuda.empty_cache()
    return {"ms": float(ms.mean()), "gbs": gbs, "nbytes": nbytes, "J": J, "n_exec": n_exec,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                         "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy; of measured)" if peaks else "fallback 6650 GB/s",
                         "flop_per_byte": _flop_per_sample_step(w) / (4.0 * J), "machine_balance_flop_per_byte": FP32_PEAK_TFLOPS * 1e3 / peak,
                         "fp32_frac_nominal": float(N) * H * _flop_per_sample_step(w) / (ms.mean() * 1e-3) / 1e12 / FP32_PEAK_TFLOPS}}


def extra_dumps(mp, args, local, stream):
    """a9: the two lifted trajectory dumps whose intensity is below the machine balance (d = 8: 4.5 flop/B, d = 16: 8.5 flop/B):
    HBM write bandwidth against the measured copy peak.  Output 1.7 / 6.7 GB per launch: larger than L2, no flush needed."""
    import workloads as W
    out = {}
    with clocked(local) as ck:
        for name in ("C1", "C2"):
            w = W.make(name, N=1 << 20)
            x0s, _, ticks = W.tick_inputs(w, 8)
            ctx = mp.Context(w, device=local)
            d = measure_dump(mp, ctx, w, x0s, ticks, 5, 3, "lifted", stream)
            out[f"{name}_model_lifted_N2^20"] = {"gbs": d["gbs"], "ms_per_launch": d["ms"], "gb_per_launch": d["nbytes"] / 1e9, "roofline": d["roofline"]}
            ctx.close()
    out["clocks"] = ck.summary
    return out


def run_dump(args, ctx, w, x0s, ticks, stream, info):
    """a9: trajectory-dump path. Every launch writes H*J*N fp32 (NaN after a candidate's first
    violating state), candidate fastest; bounded by HBM write bandwidth where 2d(d+m)/(4J) flop/B is
    below the machine balance (lifted dumps at d = 8, 16), by the FP32 pipe otherwise."""
    import paper_1906_02318_b200 as mp
    d = measure_dump(mp, ctx, w, x0s, ticks, args.steps, args.warmup, args.dump, stream)
    print(json.dumps({
        "metric": "trajectory dump bandwidth", "value": d["gbs"], "unit": "GB/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": d["ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"{args.workload} dump={args.dump}: d={w.d} J={d['J']} N={w.N} H={w.H}; output {d['nbytes'] / 1e9:.2f} GB per launch "
                               "(larger than L2, so no flush is needed)", "kernel": info},
        "roofline": d["roofline"], "executed_sample_steps": d["n_exec"], "gpu_launches": args.steps}))


def run_sweep(args, local):
    import torch
    import paper_1906_02318_b200 as mp
    stream = torch.cuda.current_stream().cuda_stream
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    s = extra_sweep(mp, args, local, flush, stream)
    print(json.dumps({"metric": "rollout sample-steps/s (scale sweep)", "unit": "sample-steps/s", "n_gpus": 1, "steps": 20, "warmup": 5,
                      "value": s["rows"][-1]["sample_steps_per_s"], "higher_is_better": True, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": s["workload"], "l2": "256 MB buffer written between timed iterations"},
                      "sweep": s["rows"], "clocks": s["clocks"]}))


def run_timeline(args, local):
    """Where a paper-scale tick spends its time: %globaltimer stamps of the latency kernel's stages
    (mpmi_profile_timeline) on device-resident ticks, and the host's view of mpmi_step / mpmi_step_result."""
    import torch
    import workloads as W
    import paper_1906_02318_b200 as mp
    stream = torch.cuda.current_stream().cuda_stream
    w = W.make(args.workload)
    ctx = mp.Context(w, device=local)
    info = ctx.info()
    nt = 300
    x0s, uus, ticks = W.tick_inputs(w, nt)
    dX0 = torch.as_tensor(x0s).cuda().contiguous(); dUU = torch.as_tensor(uus).cuda().contiguous()
    dRes = torch.zeros(56, dtype=torch.uint8, device="cuda")
    stamps = torch.zeros((info["blocks"], 8), dtype=torch.int64, device="cuda")
    ctx.profile_timeline(stamps.data_ptr())
    rows, ev_us = [], []
    with clocked(local) as ck:
        for t in range(nt):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.step_device(dX0[t].data_ptr(), dUU[t].data_ptr(), int(ticks[t]), stream, dRes.data_ptr())
            e1.record()
            torch.cuda.synchronize()
            s = stamps.cpu().numpy().astype(np.int64)
            if t >= 50:
                t0 = s[:, 0].min()
                rows.append([s[:, 0].max() - t0, np.median(s[:, 1] - s[:, 0]), np.median(s[:, 2] - s[:, 1]), np.median(s[:, 3] - s[:, 2]),
                             np.median(s[:, 4] - s[:, 3]), (s[:, 4] - s[:, 3]).max(), np.median(s[:, 5] - s[:, 4]), s[:, 5].max() - t0,
                             s[:, 4].max() - t0])
                ev_us.append(1e3 * e0.elapsed_time(e1))
        ctx.profile_timeline(0)
        r = np.median(np.array(rows, dtype=np.float64), axis=0) / 1e3
        # host view
        xs = [np.ascontiguousarray(x) for x in x0s]; us = [np.ascontiguousarray(u) for u in uus]
        t_enq, t_wait, t_tot = [], [], []
        for t in range(nt):
            a0 = time.perf_counter(); ctx.step(xs[t], us[t], int(ticks[t]), stream)
            a1 = time.perf_counter(); ctx.step_result()
            a2 = time.perf_counter()
            if t >= 50:
                t_enq.append(a1 - a0); t_wait.append(a2 - a1); t_tot.append(a2 - a0)
    med = lambda v: 1e6 * float(np.median(v))
    print(json.dumps({
        "metric": "tick timeline", "workload": f"{args.workload}: n={w.n} m={w.m} d={w.d} N={w.N} H={w.H}", "kernel": info, "ticks": nt - 50,
        "device_us_median": {"first CTA start -> last CTA start": r[0], "entry -> model rows requested": r[1], "-> lift done + __syncthreads": r[2],
                             "-> candidate sampled, state initialised": r[3], "-> horizon loop left (median CTA)": r[4], "horizon loop (slowest CTA)": r[5],
                             "-> keys reduced, ticket taken": r[6], "first CTA start -> last CTA leaves the horizon loop": r[8],
                             "first CTA start -> last CTA done (kernel span)": r[7], "CUDA events around the launch": float(np.median(ev_us))},
        "host_us_median": {"mpmi_step (copy inputs, 1 node-param update, cudaGraphLaunch)": med(t_enq),
                           "mpmi_step_result (poll the mapped result)": med(t_wait), "total": med(t_tot)},
        "clocks": ck.summary}))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--N", type=int, default=None, help="override candidates per GPU")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-latency", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the 'extra' block (scale sweep, C5, paper-scale latencies, HBM-bound dumps)")
    ap.add_argument("--dump", choices=["lifted", "phys"], default=None,
                    help="measure the trajectory-dump path (mpmi_rollout_batch, SURVEY 8(a) a9) instead of the tick")
    ap.add_argument("--noise", type=float, default=0.0,
                    help="std of the additive prediction noise of Alg. 2 l.5 (PAPER.md:150); 0 = the noise-free configs of BASELINE.json")
    ap.add_argument("--relift", action="store_true", help="re-lift model x' = C(K Psi(x) + B u) instead of the linear lifted model")
    ap.add_argument("--timeline", action="store_true", help="stage timeline of a paper-scale tick (latency kernel: C1, C2, C3) instead of the bench line")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE.json configs[3] alone: N = 2^14 .. 2^20 on the C4 model, sample-steps/s and tick latency at each N")
    ap.add_argument("--affine", action="store_true",
                    help="affine-in-u fast path x_k = a_k + G_k u (SURVEY 8(f) NEXT-4): same selections, n*m FMAs per sample-step; its own metric")
    ap.add_argument("--tensor32", action="store_true", help="d = 32: take the verified tensor-core tick for small candidate sets too (it is the default above 256 candidates per SM)")
    ap.add_argument("--unverified", action="store_true", help="tensor-core kernels without the verification pass (measurement only: the bare 3xTF32 rollout)")
    ap.add_argument("--no-predict", action="store_true", help="d > 32: pre-sort by input-box cell instead of by predicted life time")
    ap.add_argument("--no-tensor", action="store_true", help="FP32 kernels only (d = 32: register kernel, d = 128: SIMT warp-tile kernel)")
    ap.add_argument("--bounds-scale", type=float, default=1.0,
                    help="scale the safe set (100 = every rollout safe: no early exit, full N*H work)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    # --gpus N without a launcher: start the N ranks ourselves (one process per GPU, NCCL over 127.0.0.1)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import workloads as W
    import paper_1906_02318_b200 as mp
    mp.load_library()                                        # fails loudly if the CUDA extension is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if local >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} has no GPU (LOCAL_RANK {local}, {torch.cuda.device_count()} visible): one process per GPU")
    torch.cuda.set_device(local)
    dist = None
    # MPMI_BENCH_FORCE_SHARD=1 runs the sharded (multi-GPU) code path on one rank: a real single-rank NCCL group,
    # shard_step -> all-gather -> shard_finalize, so that the N > 1 path can be exercised on a 1-GPU box
    sharded = world > 1 or os.environ.get("MPMI_BENCH_FORCE_SHARD") == "1"
    if sharded:
        import torch.distributed as dist
        if world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", str(_free_port()))
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    stream = torch.cuda.current_stream().cuda_stream
    if args.sweep:
        return run_sweep(args, local)
    if args.timeline:
        return run_timeline(args, local)

    # ---- workload: weak scaling -- every rank owns N_per candidates of a global set of world*N_per
    w1 = W.make(args.workload, N=args.N)
    n_per = w1.N
    w = W.make(args.workload, N=n_per * world)
    if args.bounds_scale != 1.0:
        w = W.generate.scaled_bounds(w, args.bounds_scale)
    w.noise_sigma = args.noise
    w.model_kind = 1 if args.relift else 0
    K_, W_ = args.steps, args.warmup
    x0s, uus, ticks = W.tick_inputs(w, W_ + K_)
    from paper_1906_02318_b200.shard import shard_plan, gather_partials
    begin, count = shard_plan(w.N, 1, world, rank)             # the injected u_user (index N) goes to the last rank
    ctx = mp.Context(w, device=local, shard=(begin, count) if sharded else (0, 0), variant=_variant(args, mp))
    info = ctx.info()
    if args.dump:
        return run_dump(args, ctx, w, x0s, ticks, stream, info)

    dPart = torch.zeros(3, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    def tick_sharded(t, dX0, dUU, dRes):                       # shard -> 24-byte all-gather -> finalise
        px, pu, pr = dX0[t].data_ptr(), dUU[t].data_ptr(), dRes[t].data_ptr()
        ctx.shard_step(px, pu, int(ticks[t]), stream, dPart.data_ptr())
        parts = gather_partials(dPart, world)
        ctx.shard_finalize(parts.data_ptr(), world, pu, int(ticks[t]), stream, pr)

    with clocked(local) as ck:
        m = measure_ticks(mp, ctx, w, x0s, uus, ticks, K_, W_, flush, stream, tick_fn=tick_sharded if sharded else None, dist=dist)
    step_ms, res = m["step_ms"], m["res"]
    total_ms = float(step_ms.sum())
    n_exec = m["n_exec"]                                       # whole-job executed sample-steps (all shards)
    if dist:
        tmax = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        total_ms = float(tmax.item())
    nominal = float(w.N + 1) * w.H * K_
    value = n_exec / (total_ms * 1e-3)

    # ---- e2e: the public host API, host buffers, H2D + D2H inside the timed region
    e2e = None
    lat = {}
    if not sharded:
        x0c = [np.ascontiguousarray(x) for x in x0s]; uuc = [np.ascontiguousarray(u) for u in uus]
        for t in range(W_):
            ctx.step_sync(x0c[t], uuc[t], int(ticks[t]), stream)
        torch.cuda.synchronize()
        e_exec, wall = 0, []
        t_all = time.perf_counter()
        for t in range(W_, W_ + K_):
            t0 = time.perf_counter()
            rr = ctx.step_sync(x0c[t], uuc[t], int(ticks[t]), stream)
            wall.append(time.perf_counter() - t0)
            e_exec += rr.n_exec
        t_all = time.perf_counter() - t_all
        e2e = {"value": e_exec / t_all, "unit": "sample-steps/s", "h2d_bytes_per_step": 4 * (w.n + w.m) + 8, "d2h_bytes_per_step": 56,
               "transport": "x0, u_user, tick ride in the graph's kernel-node parameters; the 56-byte result is written "
                            "by the kernel into mapped pinned host memory and polled",
               "ms_per_step": 1e3 * t_all / K_}
        p50, p99 = _percentiles(wall)
        lat[f"{args.workload}_N{w.N}"] = {"host_p50_us": 1e6 * p50, "host_p99_us": 1e6 * p99,
                                          "gpu_p50_us": 1e3 * _percentiles(step_ms)[0], "ticks": K_}
        info["deferred_fraction"] = ctx.info()["reserved"] / float(w.N + 1) if info["launches_per_tick"] > 4 else None
    else:
        # e2e at N GPUs: x0 / u_user from pinned host memory every tick, sharded tick, 24-byte exchange, result back to the host
        try:
            hx = torch.as_tensor(x0s).contiguous().pin_memory(); hu = torch.as_tensor(uus).contiguous().pin_memory()
            hres = torch.zeros(56, dtype=torch.uint8).pin_memory()
            dx = torch.empty(w.n, dtype=torch.float32, device="cuda"); du = torch.empty(w.m, dtype=torch.float32, device="cuda")
            dres = torch.zeros(56, dtype=torch.uint8, device="cuda")
            cur = torch.cuda.current_stream()

            def tick_e2e(t):
                dx.copy_(hx[t], non_blocking=True); du.copy_(hu[t], non_blocking=True)
                ctx.shard_step(dx.data_ptr(), du.data_ptr(), int(ticks[t]), stream, dPart.data_ptr())
                parts = gather_partials(dPart, world)
                ctx.shard_finalize(parts.data_ptr(), world, du.data_ptr(), int(ticks[t]), stream, dres.data_ptr())
                hres.copy_(dres, non_blocking=True)
                cur.synchronize()
                return int(np.frombuffer(hres.numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)[0]["n_exec"])

            for t in range(W_):
                tick_e2e(t)
            dist.barrier()
            t_all = time.perf_counter()
            e_exec = sum(tick_e2e(t) for t in range(W_, W_ + K_))
            t_all = time.perf_counter() - t_all
            tm = torch.tensor([t_all], device="cuda", dtype=torch.float64)
            dist.all_reduce(tm, op=dist.ReduceOp.MAX)
            e2e = {"value": e_exec / float(tm.item()), "unit": "sample-steps/s", "h2d_bytes_per_step": 4 * (w.n + w.m), "d2h_bytes_per_step": 56,
                   "transport": "per rank: x0, u_user copied from pinned host memory, sharded tick, 24-byte NCCL all-gather, 56-byte result copied back",
                   "ms_per_step": 1e3 * float(tm.item()) / K_}
        except Exception as ex:                                  # never lose the bench line over the e2e leg
            e2e = {"value": None, "unit": "sample-steps/s", "error": repr(ex)[:200]}

    m["step_ms"] = step_ms * (total_ms / float(step_ms.sum()))    # (max over ranks)
    roofline = make_roofline(info, w, m, world=world, key=args.workload + ("-fp32" if info["variant"] != 4 else ""))

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    # ---- latency half of the metric + the rest of the metric's configs (N = 1 only)
    extra = None
    if not sharded:
        if not args.no_latency:
            lat.update(extra_latency(mp, args, local, stream))
        if not args.no_extras:
            extra = {"sweep": extra_sweep(mp, args, local, flush, stream), "C5": extra_c5(mp, args, local, flush, stream),
                     "dumps": extra_dumps(mp, args, local, stream), "variants": extra_variants(mp, args, local, flush, stream)}

    # ---- CPU baseline: the oracle as it stands on this box's host cores (bounded sample), then on one thread
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_s = min(w.N, 1 << 18)
        v, nt, cores = _time_oracle(w, x0s, uus, ticks, W_, 10.0, K_, n_s)
        cpu = {"value": v, "unit": "sample-steps/s", "cores": cores, "kind": "oracle",
               "sample": f"first {n_s} of {w.N} candidates (+ user slot), {nt} ticks, H={w.H}, fp64"}
        if _set_oracle_threads(1):
            n1 = min(w.N, 1 << 15)
            v1, nt1, c1 = _time_oracle(w, x0s, uus, ticks, W_, 6.0, K_, n1)
            cpu["one_thread"] = {"value": v1, "unit": "sample-steps/s", "cores": c1,
                                 "sample": f"first {n1} of {w.N} candidates (+ user slot), {nt1} ticks, H={w.H}, fp64"}
            _set_oracle_threads(cores)

    out = {
        "metric": "rollout sample-steps/s", "value": value, "unit": "sample-steps/s", "n_gpus": world,
        "steps": K_, "warmup": W_, "ms_per_step": total_ms / K_, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 (3xTF32 split products, fp32 accumulate; candidates near the safe-set boundary re-rolled in fp32)" if info["variant"] == 4 else "f32", "data": "synthetic",
        "config": {"workload": _workload_string(args, w, n_per),
                   "path": ("verified tensor-core tick: 3xTF32 tcgen05 rollout of every candidate, FP32 second pass over the candidates that came within the derived "
                            "bound tau of the safe-set boundary -- same flags and winner as the FP32 tick (DESIGN.md section 6a)" if info["variant"] == 4 and not args.unverified
                            else "bare 3xTF32 tcgen05 rollout (measurement only)" if info["variant"] == 4
                            else "affine-in-u fast path (NEXT-4: separate metric, 2nm flop per sample-step)" if info["variant"] == 6
                            else "FP32 kernels"),
                   "candidates_total": int(w.N + 1), "l2": "256 MB buffer written between timed iterations",
                   "parallelism": f"candidate shards x{world}, one 24-byte all-gather per tick" if sharded else "single GPU",
                   "kernel": info},
        "nominal_value": nominal / (total_ms * 1e-3), "executed_fraction": n_exec / nominal,
        "safe_fraction": float(res["n_safe"].mean() / (w.N + 1)),
        "clocks": ck.summary, "e2e": e2e, "gpu_launches": K_ * (info["launches_per_tick"] + (1 if sharded else 0)),
        "roofline": roofline, "cpu_baseline": cpu, "latency": lat, "extra": extra,
        "paper_context": "paper: >10,000 trajectories per tick at ~100 Hz / ~60 Hz on a GeForce 860M (PAPER.md:12, 266)",
    }
    print(json.dumps(out))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
