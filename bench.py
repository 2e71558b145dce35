#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native MPMI-SC tick (BASELINE.json metric:
"rollout sample-steps/sec and p50/p99 per-tick latency at N=10k and 1M; % FP32 peak").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl reference]

One "step" is one whole control tick: sample N candidates -> lift ->
H-step rollout with per-step safe test -> argmin selection -> result, on one batch of synthetic
input (a fresh x0, u_user and Philox tick per step).  Default workload: C4 at N = 2^20, H = 100
(BASELINE.json configs[3], the configuration the throughput half of the metric is quoted on);
the latency half (p50/p99 at N = 10k, C2, and at N = 2^20) is reported under "latency".

value    = executed sample-steps/s with inputs resident in HBM (mpmi_step_device), CUDA-event timed
e2e      = the same metric through mpmi_step_sync with HOST buffers (H2D + D2H inside the region)
roofline = the rollout kernel against the FP32 FMA peak ("alu")
cpu_baseline = the FP64 oracle, as it stands, on this box's host cores (bounded sample)

One "sample-step" = one evaluation of z <- K z + B u followed by isSafe; candidate i executes
min(steps_i + 1, H) of them (Algorithm 2 l.4 stops at the first violation).  The nominal N*H count
is reported beside it.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # 74.45: SMs x FP32 lanes x 2 flop x max SM clock


def _flop_per_sample_step(w):
    if getattr(w, "model_kind", 0) == 1:                # re-lift model: n physical rows + the lift itself (cos / sin counted as 1)
        lift = 3.0 * w.d if w.lift_kind == 0 else (2.0 * w.n + 2.0) * (w.d - w.n)
        return 2.0 * w.n * (w.d + w.m) + lift
    return 2.0 * w.d * (w.d + w.m)                      # dense K and B, nothing discounted


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


def _variant(args, mp):
    V = mp.mpmi
    return ((V.VARIANT_NO_TENSOR if args.no_tensor else 0) | (V.VARIANT_AFFINE if args.affine else 0) | (V.VARIANT_NO_PREDICT if args.no_predict else 0)
            | (V.VARIANT_TENSOR32 if args.tensor32 else 0) | (V.VARIANT_TC_UNVERIFIED if args.unverified else 0))


def _percentiles(v):
    v = np.sort(np.asarray(v, dtype=np.float64))
    return float(v[len(v) // 2]), float(v[min(len(v) - 1, int(0.99 * len(v)))])


def run_reference(args):
    """--impl reference: the FP64 oracle as it stands, on the host cores, same config / metric / unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads as W
    from oracle import oracle as O
    w = W.make(args.workload, N=args.N)
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
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload}: n={w.n} m={w.m} d={w.d} N={w.N} H={w.H}", "sample": sample},
        "cpu_baseline": {"value": val, "unit": "sample-steps/s", "cores": O.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "sample-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_dump(args, ctx, w, x0s, ticks, stream, info):
    """a9: trajectory-dump path. Every launch writes H*J*N fp32 (NaN after a candidate's first
    violating state), candidate fastest; bounded by HBM write bandwidth where 2d(d+m)/(4J) flop/B is
    below the machine balance (lifted dumps at d = 8, 16), by the FP32 pipe otherwise."""
    import torch
    import paper_1906_02318_b200 as mp
    N, H = w.N, w.H
    J = w.d if args.dump == "lifted" else w.n
    kind = mp.DUMP_LIFTED if args.dump == "lifted" else mp.DUMP_PHYS
    traj = torch.empty((H, J, N), dtype=torch.float32, device="cuda")
    steps = torch.empty(N, dtype=torch.int32, device="cuda")
    dX0 = torch.as_tensor(x0s).cuda().contiguous()
    K_, W_ = args.steps, args.warmup
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
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    peak = float(peaks.get("hbm_gbs", 6650.0))
    gbs = nbytes / (ms.mean() * 1e-3) / 1e9
    n_exec = int(torch.clamp(steps.to(torch.int64) + 1, max=H).sum().item())
    flop_b = _flop_per_sample_step(w) / (4.0 * J)
    print(json.dumps({
        "metric": "trajectory dump bandwidth", "value": gbs, "unit": "GB/s", "n_gpus": 1, "steps": K_, "warmup": W_,
        "ms_per_step": float(ms.mean()), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"{args.workload} dump={args.dump}: d={w.d} J={J} N={N} H={H}; output {nbytes / 1e9:.2f} GB per launch "
                               "(larger than L2, so no flush is needed)", "kernel": info},
        "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                     "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy; of measured)" if peaks else "fallback 6650 GB/s",
                     "flop_per_byte": flop_b, "machine_balance_flop_per_byte": FP32_PEAK_TFLOPS * 1e3 / peak,
                     "fp32_frac_nominal": float(N) * H * _flop_per_sample_step(w) / (ms.mean() * 1e-3) / 1e12 / FP32_PEAK_TFLOPS},
        "executed_sample_steps": n_exec, "gpu_launches": K_}))


def run_sweep(args, w_full, local):
    """Scale sweep (BASELINE.json configs[3]): the same model at N = 2^14 .. 2^20 candidates, device-timed tick,
    host p50 / p99 of mpmi_step_sync, executed sample-steps/s and the FP32 fraction at each N."""
    import torch
    import workloads as W
    import paper_1906_02318_b200 as mp
    stream = torch.cuda.current_stream().cuda_stream
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    K_, W_ = args.steps, args.warmup
    rows = []
    variant = _variant(args, mp)
    for lg in range(14, 21):
        w = W.make(args.workload, N=1 << lg)
        w.noise_sigma = args.noise; w.model_kind = 1 if args.relift else 0
        x0s, uus, ticks = W.tick_inputs(w, W_ + K_)
        ctx = mp.Context(w, device=local, variant=variant)
        dX0 = torch.as_tensor(x0s).cuda().contiguous(); dUU = torch.as_tensor(uus).cuda().contiguous()
        dRes = torch.zeros((W_ + K_, 56), dtype=torch.uint8, device="cuda")
        for t in range(W_):
            ctx.step_device(dX0[t].data_ptr(), dUU[t].data_ptr(), int(ticks[t]), stream, dRes[t].data_ptr())
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K_)]
        torch.cuda.synchronize()
        for i in range(K_):
            flush.fill_(i & 0xFF)
            ev[i][0].record()
            ctx.step_device(dX0[W_ + i].data_ptr(), dUU[W_ + i].data_ptr(), int(ticks[W_ + i]), stream, dRes[W_ + i].data_ptr())
            ev[i][1].record()
        torch.cuda.synchronize()
        ms = np.array([a.elapsed_time(b) for a, b in ev])
        res = np.frombuffer(dRes.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)
        n_exec = int(res["n_exec"][W_:].sum())
        wall = []
        for t in range(W_, W_ + K_):
            t0 = time.perf_counter()
            ctx.step_sync(np.ascontiguousarray(x0s[t]), np.ascontiguousarray(uus[t]), int(ticks[t]), stream)
            wall.append(time.perf_counter() - t0)
        p50, p99 = _percentiles(wall)
        info = ctx.info()
        flop = _flop_per_sample_step(w) if info["variant"] != 6 else 2.0 * w.n * w.m
        rows.append({"N": 1 << lg, "gpu_ms": float(ms.mean()), "host_p50_us": 1e6 * p50, "host_p99_us": 1e6 * p99,
                     "sample_steps_per_s": n_exec / (ms.sum() * 1e-3), "nominal_sample_steps_per_s": float(w.N + 1) * w.H * K_ / (ms.sum() * 1e-3),
                     "fp32_frac": n_exec * flop / (ms.sum() * 1e-3) / 1e12 / FP32_PEAK_TFLOPS, "variant": info["variant"]})
        ctx.close()
    print(json.dumps({"metric": "rollout sample-steps/s (scale sweep)", "unit": "sample-steps/s", "n_gpus": 1, "steps": K_, "warmup": W_,
                      "value": rows[-1]["sample_steps_per_s"], "higher_is_better": True, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": f"{args.workload} scale sweep: n={w_full.n} m={w_full.m} d={w_full.d} H={w_full.H}, N = 2^14 .. 2^20 (+1 user slot)",
                                 "l2": "256 MB buffer written between timed iterations"},
                      "sweep": rows}))


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
    ap.add_argument("--dump", choices=["lifted", "phys"], default=None,
                    help="measure the trajectory-dump path (mpmi_rollout_batch, SURVEY 8(a) a9) instead of the tick")
    ap.add_argument("--noise", type=float, default=0.0,
                    help="std of the additive prediction noise of Alg. 2 l.5 (PAPER.md:150); 0 = the noise-free configs of BASELINE.json")
    ap.add_argument("--relift", action="store_true", help="re-lift model x' = C(K Psi(x) + B u) instead of the linear lifted model")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE.json configs[3]: N = 2^14 .. 2^20 on the chosen workload, sample-steps/s and tick latency at each N")
    ap.add_argument("--affine", action="store_true",
                    help="affine-in-u fast path x_k = a_k + G_k u (SURVEY 8(f) NEXT-4): same selections, n*m FMAs per sample-step; its own metric")
    ap.add_argument("--tensor32", action="store_true", help="d = 32: take the verified tensor-core tick below 2^17 candidates too (it is the default from 2^17)")
    ap.add_argument("--unverified", action="store_true", help="tensor-core kernels without the verification pass (measurement only: the bare 3xTF32 rollout)")
    ap.add_argument("--no-predict", action="store_true", help="d > 32: pre-sort by input-box cell instead of by predicted life time")
    ap.add_argument("--no-tensor", action="store_true", help="d = 128: FP32 SIMT tile kernel instead of the 3xTF32 tcgen05 kernel")
    ap.add_argument("--bounds-scale", type=float, default=1.0,
                    help="scale the safe set (100 = every rollout safe: no early exit, full N*H work)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
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
    torch.cuda.set_device(local)
    dist = None
    # MPMI_BENCH_FORCE_SHARD=1 runs the sharded (multi-GPU) code path on one rank: a real single-rank NCCL group,
    # shard_step -> all-gather -> shard_finalize, so that the N > 1 path can be exercised on a 1-GPU box
    sharded = world > 1 or os.environ.get("MPMI_BENCH_FORCE_SHARD") == "1"
    if sharded:
        import torch.distributed as dist
        if world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29531")
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))

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
    ctx = mp.Context(w, device=local, shard=(begin, count) if sharded else (0, 0),
                     variant=_variant(args, mp))
    info = ctx.info()
    stream = torch.cuda.current_stream().cuda_stream
    if args.dump:
        return run_dump(args, ctx, w, x0s, ticks, stream, info)
    if args.sweep:
        return run_sweep(args, w, local)

    dX0 = torch.as_tensor(x0s).cuda().contiguous()
    dUU = torch.as_tensor(uus).cuda().contiguous()
    dRes = torch.zeros((W_ + K_, 56), dtype=torch.uint8, device="cuda")
    dPart = torch.zeros(3, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    def tick_device(t):
        px, pu, pr = dX0[t].data_ptr(), dUU[t].data_ptr(), dRes[t].data_ptr()
        if not sharded:
            ctx.step_device(px, pu, int(ticks[t]), stream, pr)
        else:                                                  # shard -> 24-byte all-gather -> finalise
            ctx.shard_step(px, pu, int(ticks[t]), stream, dPart.data_ptr())
            parts = gather_partials(dPart, world)
            ctx.shard_finalize(parts.data_ptr(), world, pu, int(ticks[t]), stream, pr)

    for t in range(W_):
        tick_device(t)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    clocks = ClockSampler(local)
    clocks.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K_)]
    torch.cuda.synchronize()
    for i in range(K_):
        flush.fill_(i & 0xFF)                                  # L2 flush between timed iterations (untimed)
        ev[i][0].record()
        tick_device(W_ + i)
        ev[i][1].record()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    clocks.stop_flag = True
    step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    total_ms = float(step_ms.sum())
    res = np.frombuffer(dRes.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)
    n_exec = int(res["n_exec"][W_:].sum())                     # whole-job executed sample-steps (all shards)
    if dist:
        tmax = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        total_ms = float(tmax.item())
    nominal = float(w.N + 1) * w.H * K_
    value = n_exec / (total_ms * 1e-3)

    # ---- e2e: the public host API, host buffers, H2D + D2H inside the timed region (N = 1 only)
    e2e = None
    lat = {}
    if not sharded:
        r = mp.Result()
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
        if not args.no_latency:
            # latency half of the metric: C2 (N = 10k), 1,000 stored closed-loop ticks, host API
            w2 = W.make("C2")
            seq = np.loadtxt(W.generate.C2_SEQUENCE, comments="#")
            c2 = mp.Context(w2, device=local)
            xs = [np.ascontiguousarray(row[1:5], dtype=np.float32) for row in seq]
            us = [np.ascontiguousarray(row[5:6], dtype=np.float32) for row in seq]
            for t in range(50):
                c2.step_sync(xs[t], us[t], t, stream)
            wall = []
            for t in range(len(seq)):
                t0 = time.perf_counter()
                c2.step_sync(xs[t], us[t], t, stream)
                wall.append(time.perf_counter() - t0)
            p50, p99 = _percentiles(wall)
            lat["C2_N10000"] = {"host_p50_us": 1e6 * p50, "host_p99_us": 1e6 * p99, "ticks": len(seq)}
            c2.close()

    if sharded:
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

    # ---- roofline of the dominant (only) kernel: plain FP32 FMA arithmetic
    flop = _flop_per_sample_step(w) if info["variant"] != 6 else 2.0 * w.n * w.m      # affine path: n*m FMAs per sample-step
    achieved = n_exec / world * flop / (total_ms * 1e-3) / 1e12            # per GPU
    traffic = None
    tj = os.path.join(ROOT, "profiles", "roofline_traffic.csv")     # ncu --set full, dram bytes per launch
    if os.path.exists(tj):
        for line in open(tj).read().splitlines()[1:]:
            f = line.split(",")
            if f and f[0] == args.workload + ("-tensor32" if info["variant"] == 4 and w.d <= 32 else ""):
                traffic = int(f[2])
    nominal_frac = nominal / K_ / max(world, 1) * flop / (total_ms * 1e-3 / K_) / 1e12 / FP32_PEAK_TFLOPS
    if info["variant"] == 4:
        # d = 128 runs as a 3xTF32 split contraction on the tcgen05 tensor cores (rollout_tc.cuh): every
        # algorithmic flop costs three TF32 tensor flops, so the peak for this path is the measured bf16
        # GEMM peak x the guide's nominal tf32:bf16 ratio (1.1 : 2.25 PFLOP/s) / 3.
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
        bf16 = float(peaks.get("bf16_tflops", 1590.0))
        peak = bf16 * (1.1 / 2.25) / 3.0
        roofline = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                    "traffic": traffic,
                    "peak_source": ("MEASURED_PEAKS.json bf16_tflops (burst; of measured)" if peaks else "fallback 1590 TFLOP/s bf16 (of fallback)")
                                   + " x 1.1/2.25 (nominal tf32:bf16) / 3 (3xTF32 split products per algorithmic flop)",
                    "kernel": "rollout_tc_kernel", "dtype": "3xTF32 (fp32 accumulate)",
                    "tensor_tflops_executed": achieved * 3.0 * (info["d_pad"] + 8.0) / (w.d + w.m),     # K padded to d_pad + one 8-wide input block
                    "fp32_alu_frac": achieved / FP32_PEAK_TFLOPS, "nominal_fp32_alu_frac": nominal_frac}
    else:
        roofline = {"bound": "alu", "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "frac": achieved / FP32_PEAK_TFLOPS, "traffic": traffic,
                    "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md section 6)",
                    "kernel": {1: "rollout_reg_kernel", 2: "rollout_tile_kernel", 3: "rollout_lat_kernel", 5: "rollout_relift_kernel",
                               6: "rollout_affine_kernel"}.get(info["variant"], "?"),
                    "nominal_frac": nominal_frac}

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    # ---- CPU baseline: the oracle as it stands on this box's host cores (bounded sample)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        n_s = min(w.N, 1 << 18)
        o = O.Oracle(w, N=n_s)
        o.step(x0s[0], uus[0], 0)
        ne, t0, nt = 0, time.perf_counter(), 0
        while time.perf_counter() - t0 < 10.0 and nt < K_:
            ne += o.step(x0s[W_ + nt], uus[W_ + nt], int(ticks[W_ + nt]))["n_exec"]; nt += 1
        dt = time.perf_counter() - t0
        cpu = {"value": ne / dt, "unit": "sample-steps/s", "cores": O.num_threads(), "kind": "oracle",
               "sample": f"first {n_s} of {w.N} candidates (+ user slot), {nt} ticks, H={w.H}, fp64"}

    out = {
        "metric": "rollout sample-steps/s", "value": value, "unit": "sample-steps/s", "n_gpus": world,
        "steps": K_, "warmup": W_, "ms_per_step": total_ms / K_, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 (3xTF32 split products, fp32 accumulate)" if info["variant"] == 4 else "f32", "data": "synthetic",
        "config": {"workload": f"{args.workload}: n={w.n} m={w.m} d={w.d} N={n_per}/GPU (+1 user slot) H={w.H}, "
                               f"Philox/grid sampler, calibrated 40% safe (DESIGN.md section 4)"
                               + (f", safe set scaled x{args.bounds_scale}" if args.bounds_scale != 1.0 else "")
                               + (f", prediction noise sigma={args.noise}" if args.noise else "")
                               + (", re-lift model" if args.relift else "")
                               + (", opt-in VERIFIED tensor-core tick at d = 32: 3xTF32 tcgen05 rollout, candidates that came near the safe-set boundary "
                                  "are rolled again by the FP32 register kernel (same result as the FP32 tick; DESIGN.md section 6)" if args.tensor32 and info["variant"] == 4 else "")
                               + (", affine-in-u fast path (NEXT-4: separate metric, 2nm flop per sample-step)" if info["variant"] == 6 else ""),
                   "candidates_total": int(w.N + 1), "l2": "256 MB buffer written between timed iterations",
                   "parallelism": f"candidate shards x{world}, one 24-byte all-gather per tick" if sharded else "single GPU",
                   "kernel": info},
        "nominal_value": nominal / (total_ms * 1e-3), "executed_fraction": n_exec / nominal,
        "safe_fraction": float(res["n_safe"][W_:].mean() / (w.N + 1)),
        "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": K_ * (info["launches_per_tick"] + (1 if sharded else 0)),
        "roofline": roofline, "cpu_baseline": cpu, "latency": lat,
        "paper_context": "paper: >10,000 trajectories per tick at ~100 Hz / ~60 Hz on a GeForce 860M (PAPER.md:12, 266)",
    }
    print(json.dumps(out))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
