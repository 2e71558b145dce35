"""Parity rules T1-T3 (north_star): GPU vs FP64 oracle on the same seeded inputs."""
import numpy as np

TRAJ_RTOL = 1e-4      # T1: max_k ||z_gpu - z_ref||_2 / max(||z_ref||_2, 1e-3)  (north_star: <= 1e-4)
MARGIN = 1e-4         # T2 / T3: flags and selection are compared where the safe-set margin exceeds 1e-4


def traj_rel_err(gpu_traj, ref_traj, executed):
    """gpu_traj, ref_traj: (H, d) for one candidate; compares the steps executed by both."""
    e = executed
    num = np.linalg.norm(gpu_traj[:e].astype(np.float64) - ref_traj[:e], axis=1)
    den = np.maximum(np.linalg.norm(ref_traj[:e], axis=1), 1e-3)
    return float((num / den).max()) if e > 0 else 0.0


def check_flags(gpu_steps, ref_steps, ref_margin, H):
    """T2: identical steps / safe flag for every candidate whose margin exceeds 1e-4."""
    robust = ref_margin > MARGIN
    bad = np.nonzero(robust & (gpu_steps != ref_steps))[0]
    return bad, int(robust.sum())


def accept_selection(g, ref, H):
    """T3.  g: GPU result dict (index, safe, steps, u, dist); ref: oracle.step(..., detail=True).
    Returns (ok, exact, reason)."""
    steps_o, marg, dist_o = ref["steps_all"], ref["margin_all"], ref["dist_all"]
    robust = marg > MARGIN
    safe_o = steps_o == H
    gi = int(g["index"])
    if gi < 0 or gi >= len(steps_o):
        return False, False, "index out of range"
    if not np.array_equal(np.asarray(g["u"], dtype=np.float32)[: ref["U"].shape[1]], ref["U"][gi]):
        return False, False, "returned u is not bit-identical to candidate[index]"       # P4, always required
    if gi == ref["index"] and bool(g["safe"]) == bool(ref["safe"]) and int(g["steps"]) == int(ref["steps"]):
        return True, True, "exact"
    if g["safe"]:
        if not (safe_o[gi] or not robust[gi]):
            return False, False, "GPU winner is robustly unsafe in the oracle"
        rs = safe_o & robust
        if rs.any() and dist_o[rs].min() < dist_o[gi] - MARGIN:
            return False, False, "a robustly safe candidate is closer by more than 1e-4"
        return True, False, "accepted: non-robust flag or distance gap below 1e-4"
    if (safe_o & robust).any():
        return False, False, "GPU fell back although a robustly safe candidate exists"
    lim = max(int(steps_o[gi]), int(g["steps"]))
    if robust.any() and steps_o[robust].max() > lim:
        return False, False, "a robust candidate survives longer than the GPU's fallback winner"
    return True, False, "accepted: fallback among non-robust candidates"
