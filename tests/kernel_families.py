"""One small tick and one small batch launch of EVERY kernel family through the C ABI -- the workload that
compute-sanitizer is run on (summaries under profiles/):

    compute-sanitizer --tool memcheck  python tests/kernel_families.py
    compute-sanitizer --tool racecheck python tests/kernel_families.py
    compute-sanitizer --tool synccheck python tests/kernel_families.py
    compute-sanitizer --tool initcheck python tests/kernel_families.py --dump-only

Not a pytest module (the parity of these launches is asserted in test_parity_gpu.py / test_parity_full_gpu.py); it
only checks that every launch finishes, returns a candidate index and -- for the verified ticks -- agrees with the
FP32 tick, so that a hazard the tools report can be tied to a family by the label printed before it.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def families(mp):
    V = mp.mpmi
    return [
        # label, workload, N, variant flags, noise sigma, re-lift
        ("register kernel, constant-bank model (d=16)", "C2", 30000, 0, 0.0, 0),
        ("register kernel, shared-memory model, wide packing (d=8)", "C1", 5000, V.VARIANT_WIDE | V.VARIANT_SMEM_MODEL, 0.0, 0),
        ("register kernel + input-box binning (d=32)", "C4", 40000, V.VARIANT_FORCE_BINNING | V.VARIANT_NO_TENSOR, 0.0, 0),
        ("register kernel with prediction noise (d=32)", "C4", 30000, V.VARIANT_NO_TENSOR, 0.02, 0),
        ("latency kernel, 2 rows per lane (d=32)", "C3", 2500, 0, 0.0, 0),
        ("latency kernel, 4 rows per lane (d=16)", "C2", 10000, 0, 0.0, 0),
        ("warp-tile kernel (d=48 -> 64)", "T48", 3000, 0, 0.0, 0),
        ("warp-tile kernel (d=128) + life-time order", "C5", 3000, V.VARIANT_NO_TENSOR | V.VARIANT_FORCE_BINNING, 0.0, 0),
        ("tcgen05 kernel (d=128) + life-time order", "C5", 3000, V.VARIANT_FORCE_BINNING, 0.0, 0),
        ("tcgen05 kernel (d=128) with prediction noise", "C5", 2000, 0, 0.01, 0),
        ("verified tensor-core tick (d=32): tcgen05 first pass + FP32 second pass", "C4", 1 << 17, V.VARIANT_TENSOR32, 0.0, 0),
        ("re-lift kernel (d=32)", "C4", 3000, 0, 0.0, 1),
        ("affine-in-u kernel (d=32)", "C4", 20000, V.VARIANT_AFFINE, 0.0, 0),
    ]


def main():
    import torch
    import workloads as W
    import paper_1906_02318_b200 as mp
    mp.load_library()
    dump_only = "--dump-only" in sys.argv
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    for label, name, N, variant, sigma, relift in families(mp):
        w = W.make(name, N=N)
        if name == "C3":
            side = int(round(N ** 0.5)); w.N = side * side; w.grid_counts = np.array([side, side], np.int32)
        w.noise_sigma = sigma; w.model_kind = relift
        print("==", label, flush=True)
        ctx = mp.Context(w, variant=variant)
        x0s, uus, ticks = W.tick_inputs(w, 2)
        dres = torch.zeros(56, dtype=torch.uint8, device="cuda")
        dsteps = torch.zeros(w.N + 1, dtype=torch.int32, device="cuda")
        if not dump_only:
            for x0, uu, t in zip(x0s, uus, ticks):
                r = ctx.step_sync(x0, uu, int(t), stream)                        # graph path, mapped result
                dx, du = torch.as_tensor(x0).cuda(), torch.as_tensor(uu).cuda()
                ctx.step_trace(dx.data_ptr(), du.data_ptr(), int(t), stream, dres.data_ptr(), dsteps.data_ptr())
                torch.cuda.synchronize()
                d = np.frombuffer(dres.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)[0]
                assert r.index >= 0 and (r.index, r.safe, r.steps, r.n_safe, r.n_exec) == \
                       (int(d["index"]), int(d["safe"]), int(d["steps"]), int(d["n_safe"]), int(d["n_exec"])), label
            # shard path: two shards + finalize
            cut = w.N // 3
            sh = [mp.Context(w, shard=(0, cut), variant=variant), mp.Context(w, shard=(cut, w.N + 1 - cut), variant=variant)]
            parts = torch.zeros(48, dtype=torch.uint8, device="cuda")
            dx, du = torch.as_tensor(x0s[0]).cuda(), torch.as_tensor(uus[0]).cuda()
            for g in range(2):
                sh[g].shard_step(dx.data_ptr(), du.data_ptr(), 0, stream, parts.data_ptr() + 24 * g)
            sh[0].shard_finalize(parts.data_ptr(), 2, du.data_ptr(), 0, stream, dres.data_ptr())
            torch.cuda.synchronize()
            for c in sh:
                c.close()
        # batch entry with both dumps (every output element must be written: initcheck reads them back)
        nb = 1000 + 13
        for kind, J in ((mp.DUMP_LIFTED, w.d), (mp.DUMP_PHYS, w.n)):
            traj = torch.empty((w.H, J, nb), dtype=torch.float32, device="cuda")
            steps = torch.empty(nb, dtype=torch.int32, device="cuda")
            safe = torch.empty(nb, dtype=torch.uint8, device="cuda")
            dX = torch.as_tensor(x0s[:1]).cuda()
            ctx.rollout_batch(0, dX.data_ptr(), 1, nb, w.H, kind, traj.data_ptr(), steps.data_ptr(), safe.data_ptr(), 5, stream)
            torch.cuda.synchronize()
            tot = float(torch.nan_to_num(traj).sum().item()) + float(steps.sum().item()) + float(safe.sum().item())
            assert np.isfinite(tot), label
        ctx.close()
    print("all kernel families ran")


if __name__ == "__main__":
    main()
