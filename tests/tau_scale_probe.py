"""How conservative is the derived bound tau of the verified tensor-core tick (csrc/bound.cuh)?  MPMI_TC_TAU_SCALE scales tau down
until the verified tick's per-candidate step counts differ from the FP32 tick's (mpmi_step_trace on both).  Not a pytest module;
run on the B200:  python tests/tau_scale_probe.py   (summary: profiles/r2_tau_scale.md)."""
import sys, os, json
import numpy as np, torch
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import workloads as W
import paper_1906_02318_b200 as mp
V = mp.mpmi
def steps_of(ctx, w, x0, uu, t):
    d_res = torch.zeros(56, dtype=torch.uint8, device="cuda"); d_steps = torch.full((w.N + 1,), -7, dtype=torch.int32, device="cuda")
    dx, du = torch.as_tensor(x0).cuda(), torch.as_tensor(uu).cuda()
    ctx.step_trace(dx.data_ptr(), du.data_ptr(), int(t), 0, d_res.data_ptr(), d_steps.data_ptr()); torch.cuda.synchronize()
    return d_steps.cpu().numpy()
out = {}
for name, nt in (("C4", 6), ("C5", 4)):
    w = W.make(name)
    os.environ.pop("MPMI_TC_TAU_SCALE", None)
    fp32 = mp.Context(w, variant=V.VARIANT_NO_TENSOR)
    x0s, uus, ticks = W.tick_inputs(w, nt)
    ref = [steps_of(fp32, w, x0, uu, t) for x0, uu, t in zip(x0s, uus, ticks)]
    rows = []
    for sc in (1.0, 0.5, 0.25, 0.125, 0.0625, 0.03, 0.015, 0.0):
        os.environ["MPMI_TC_TAU_SCALE"] = str(sc)
        ctx = mp.Context(w)
        nd, frac = 0, []
        for k, (x0, uu, t) in enumerate(zip(x0s, uus, ticks)):
            s = steps_of(ctx, w, x0, uu, t); nd += int((s != ref[k]).sum())
            ctx.step_sync(x0, uu, int(t)); frac.append(ctx.info()["reserved"] / (w.N + 1))
        rows.append({"tau_scale": sc, "differing_step_counts": nd, "of": nt * (w.N + 1), "deferred_fraction": float(np.mean(frac))})
        print(name, rows[-1], flush=True)
        ctx.close()
    out[name] = rows
json.dump(out, open("gpurun_out/tau_scale_probe.json", "w"), indent=1)
