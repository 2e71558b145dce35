"""Calibration of the synthetic workloads (SURVEY.md 8(d) protocol) -- calls ONLY oracle/ and
workloads/.  Writes workloads/calibration.json, which workloads.generate.make() reads.

  python -m oracle.calibrate              # C1..C5 (BASELINE.json configs) and the extra test workloads
  python -m oracle.calibrate T48 T4       # only these, merged into the existing file

For each config: (1) advance the model seed until the zero-input rollout from x_nom is safe over
H; (2) bisect the input gain gamma in [1e-3, 1e3] (geometric, 40 iterations) until the oracle's
safe fraction at x_nom on the config's own sampler is 0.40 +- 0.02 (Table I band 0.28-0.50,
PAPER.md:281-288); (3) C3/C4: S = diag(max(|Psi(x_nom)|, 1)) from the oracle's lift.
"""
import json
import numpy as np
from oracle.oracle import Oracle
from workloads import generate as G

TARGET, TOL = 0.40, 0.02
N_CAL = {"C1": 1024, "C2": 10000, "C3": 10000, "C4": 16384, "C5": 4096, "T48": 4096, "T4": 4096}


def safe_fraction(w, N):
    o = Oracle(w, N=N, include_user=0)
    r = o.step(w.x_nom, np.zeros(w.m, np.float32), 0)
    return r["n_safe"] / N


def zero_input_safe(w):
    o = Oracle(w, N=1, include_user=1)
    z0 = o.lift(w.x_nom.astype(np.float64))
    steps, _, _ = o.rollout(z0, np.zeros(w.m))
    return steps == w.H


def calibrate(name):
    S = None
    if name in ("C3", "C4"):
        w0 = G.make(name, calibrated=False)
        S = np.maximum(np.abs(Oracle(w0, N=1).lift(w0.x_nom.astype(np.float64))), 1.0)
    for seed in range(64):
        w = G.make(name, calibrated=False, model_seed=seed, gamma=1.0, S=S)
        if not zero_input_safe(w):
            continue
        lo, hi, best = 1e-3, 1e3, None
        for _ in range(40):
            g = float(np.sqrt(lo * hi))
            f = safe_fraction(G.make(name, calibrated=False, model_seed=seed, gamma=g, S=S), N_CAL[name])
            if best is None or abs(f - TARGET) < abs(best[1] - TARGET):
                best = (g, f)
            if abs(f - TARGET) <= TOL / 2:
                break
            if f > TARGET:
                lo = g
            else:
                hi = g
        if abs(best[1] - TARGET) <= TOL:
            out = dict(model_seed=seed, gamma=best[0], safe_fraction=best[1], N_cal=N_CAL[name])
            if S is not None:
                out["S"] = [float(v) for v in S]
            return out
    raise RuntimeError("no seed calibrates for " + name)


def main():
    import sys
    names = sys.argv[1:] or list(G.CONFIG_NAMES + G.TEST_NAMES)
    cal = G.load_calibration() if sys.argv[1:] else {}
    for name in names:
        if name == "C4":                       # same model as C3 (BASELINE.json configs[3])
            cal["C4"] = dict(cal["C3"])
        else:
            cal[name] = calibrate(name)
        print(name, {k: v for k, v in cal[name].items() if k != "S"})
    with open(G.CALIBRATION_JSON, "w") as f:
        json.dump(cal, f, indent=1)


if __name__ == "__main__":
    main()
