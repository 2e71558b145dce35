"""GPU parity at FULL size and on every shipped kernel instantiation.

Algorithm 2's result is ONE argmin over all N candidates and its safety decision is taken per step
on every candidate.  These tests therefore compare, through mpmi_step_trace (the tick kernels in the
launch configuration bench.py times, plus one 4-byte store per candidate), EVERY candidate's step count with the FP64
oracle's (rule T2) and the tick's winner with the oracle's winner (rule T3) -- at BASELINE.json's full sizes (C4:
N = 2^20, C5: N = 262,144) and for each kernel instantiation the five configs alone do not reach (D = 64 warp-tile
kernel, wide / narrow packing, forced latency variants, M = 4).  Run on the B200 box: python -m pytest tests -m gpu."""
import numpy as np
import pytest

import workloads as W
from workloads import generate as G
from parity_util import traj_rel_err, check_flags, accept_selection, TRAJ_RTOL, MARGIN

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def mp():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1906_02318_b200 as mp
    mp.load_library()            # raises if the extension is missing: no fallback
    return mp


def _oracle(w, **kw):
    from oracle.oracle import Oracle
    return Oracle(w, **kw)


def _dev(a, dtype=None):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).cuda()


def trace_tick(mp, ctx, w, x0, uu, t):
    """(result dict, per-candidate steps incl. the user slot) of one tick through mpmi_step_trace."""
    d_res = torch.zeros(56, dtype=torch.uint8, device="cuda")
    d_steps = torch.full((w.N + w.include_user,), -7, dtype=torch.int32, device="cuda")
    dx, du = _dev(x0), _dev(uu)
    ctx.step_trace(dx.data_ptr(), du.data_ptr(), int(t), torch.cuda.current_stream().cuda_stream, d_res.data_ptr(), d_steps.data_ptr())
    torch.cuda.synchronize()
    r = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)[0]
    res = dict(u=np.array(r["u"][: w.m], np.float32), index=int(r["index"]), safe=int(r["safe"]), steps=int(r["steps"]),
               n_safe=int(r["n_safe"]), dist=float(r["dist"]), n_exec=int(r["n_exec"]), key=int(r["key"]))
    return res, d_steps.cpu().numpy()


def compare_tick(mp, ctx, o, w, x0, uu, t):
    """T2 over EVERY candidate and T3 of the winner for one tick; returns (exact, robust count)."""
    ref = o.step(x0, uu, int(t), detail=True)
    r, g_steps = trace_tick(mp, ctx, w, x0, uu, t)
    H = w.H
    assert g_steps.min() >= 0 and g_steps.max() <= H                      # every candidate was written by a tick kernel
    bad, nrobust = check_flags(g_steps, ref["steps_all"], ref["margin_all"], H)
    assert len(bad) == 0, (len(bad), bad[:5], g_steps[bad[:5]], ref["steps_all"][bad[:5]], ref["margin_all"][bad[:5]])
    ok, exact, why = accept_selection(r, ref, H)
    assert ok, (why, r, {k: ref[k] for k in ("index", "safe", "steps", "dist")})
    # the tick's own aggregates are those of its per-candidate decisions
    assert r["n_safe"] == int((g_steps == H).sum()) and r["n_exec"] == int(np.minimum(g_steps + 1, H).sum())
    nonrobust = int((ref["margin_all"] <= MARGIN).sum())
    assert abs(r["n_safe"] - ref["n_safe"]) <= nonrobust and abs(r["n_exec"] - ref["n_exec"]) <= nonrobust
    # the host path (graph, mapped result) returns the same tick
    h = ctx.step_sync(x0, uu, int(t)).as_dict(w.m)
    assert (h["index"], h["safe"], h["steps"], h["n_safe"], h["n_exec"], h["key"]) == \
           (r["index"], r["safe"], r["steps"], r["n_safe"], r["n_exec"], r["key"])
    return exact, nrobust


# ------------------------------------------------------------------ BASELINE sizes, bench launch configuration ------
@pytest.mark.parametrize("name,variant,kernel", [("C4", "default", None), ("C4", "no_tensor", 1), ("C5", "default", 4),
                                                 ("C5", "no_tensor", 2)])
def test_full_size_every_candidate(mp, name, variant, kernel):
    """C4 at N = 2^20 + 1 and C5 at N = 262,144 + 1 candidates, the contexts bench.py creates: T2 on every candidate,
    T3 on the winner against the oracle's full tick (1.7 s / ~5 s of oracle time per tick on 16 cores)."""
    V = mp.mpmi
    w = W.make(name)
    o = _oracle(w)
    ctx = mp.Context(w, variant=V.VARIANT_NO_TENSOR if variant == "no_tensor" else 0)
    if kernel is not None:
        assert ctx.info()["variant"] == kernel, ctx.info()
    x0s, uus, ticks = W.tick_inputs(w, 2)
    exact = 0
    for x0, uu, t in zip(x0s, uus, ticks):
        ex, nrobust = compare_tick(mp, ctx, o, w, x0, uu, t)
        exact += ex
        assert nrobust > 0.97 * w.N
    assert exact == 2                                                     # measured: the winner is the oracle's on every tick


# ------------------------------------------------------------------ instantiations the five configs do not reach -----
def _cases(mp):
    V = mp.mpmi
    return {
        # name: (workload, N, variant flags, expected kernel id, expected candidates per block or None)
        "tile64": ("T48", 3000, 0, 2, None),                              # d = 48 zero-padded to 64: rollout_tile_kernel<64, 3>
        "wide8": ("C1", 5000, V.VARIANT_WIDE, 1, 2 * 4 * 32),             # D = 8: 8 candidates per thread
        "wide16": ("C2", 5000, V.VARIANT_WIDE, 1, 2 * 2 * 32),            # D = 16: 4 candidates per thread
        "wide8_smem": ("C1", 5000, V.VARIANT_WIDE | V.VARIANT_SMEM_MODEL, 1, 2 * 4 * 32),     # KC = false twins
        "wide16_smem": ("C2", 5000, V.VARIANT_WIDE | V.VARIANT_SMEM_MODEL, 1, 2 * 2 * 32),
        "narrow8_smem": ("C1", 30000, V.VARIANT_SMEM_MODEL, 1, None),
        "narrow16": ("C2", 40000, V.VARIANT_NARROW, 1, None),
        "narrow32": ("C4", 9000, V.VARIANT_NARROW, 1, None),
        "lat_r2_32": ("C4", 3000, V.VARIANT_LATENCY | V.VARIANT_LAT_R2, 3, 64 // 16),
        "lat_r4_32": ("C4", 3000, V.VARIANT_LATENCY | V.VARIANT_LAT_R4, 3, 64 // 8),
        "lat_r2_16": ("C2", 3000, V.VARIANT_LATENCY | V.VARIANT_LAT_R2, 3, 64 // 8),
        "lat_r4_8": ("C1", 3000, V.VARIANT_LATENCY | V.VARIANT_LAT_R4, 3, 64 // 2),
        "lat_large": ("C2", 50000, V.VARIANT_LATENCY, 3, None),           # latency kernel beyond its default range
        "m4_lat": ("T4", 4096, 0, 3, None),                               # M = 4 through the latency kernel (default for N <= 24,576)
        "m4_reg": ("T4", 4096, V.VARIANT_NARROW, 1, None),                # M = 4 through the register kernel
        "m4_wide": ("T4", 4096, V.VARIANT_WIDE, 1, None),
        "m4_binned": ("T4", 200000, 0, 1, None),                          # 4-D input box through the spatial binning
    }


@pytest.mark.parametrize("case", ["tile64", "wide8", "wide16", "wide8_smem", "wide16_smem", "narrow8_smem", "narrow16", "narrow32", "lat_r2_32", "lat_r4_32", "lat_r2_16",
                                  "lat_r4_8", "lat_large", "m4_lat", "m4_reg", "m4_wide", "m4_binned"])
def test_every_instantiation_tick(mp, case):
    """T2 on every candidate + T3, 6 ticks, for the kernel instantiations that the BASELINE configs never select."""
    name, N, variant, kernel, cpb = _cases(mp)[case]
    w = W.make(name, N=N)
    ctx = mp.Context(w, variant=variant)
    info = ctx.info()
    assert info["variant"] == kernel, info
    if cpb is not None:
        assert info["cand_per_block"] == cpb * (info["threads_per_block"] // 32 if kernel == 1 else 1), info
    o = _oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 6)
    exact, fracs = 0, []
    for x0, uu, t in zip(x0s, uus, ticks):
        ex, _ = compare_tick(mp, ctx, o, w, x0, uu, t)
        exact += ex
    assert exact >= 5, exact


@pytest.mark.parametrize("case,noise", [("tile64", 0.0), ("tile64", 0.01), ("wide8", 0.0), ("wide16", 0.0), ("wide16_smem", 0.0), ("wide8_smem", 0.03), ("m4_wide", 0.0),
                                        ("m4_reg", 0.02)])
def test_every_instantiation_batch(mp, case, noise):
    """T1 trajectories + T2 flags through mpmi_rollout_batch for the batch-mode twins of the same instantiations
    (caller-supplied inputs, lifted dump, NaN tail)."""
    name, _, variant, kernel, _ = _cases(mp)[case]
    N = 1500 + 37
    w = W.make(name, N=N)
    w.noise_sigma = noise
    o = _oracle(w)
    ctx = mp.Context(w, variant=variant)
    assert ctx.info()["variant"] == kernel
    rng = np.random.default_rng(17)
    U = rng.uniform(w.u_lo, w.u_hi, (N, w.m)).astype(np.float32)
    x0s, _, _ = W.tick_inputs(w, 1)
    H, tick = w.H, 9
    traj = torch.full((H, w.d, N), 7.0, dtype=torch.float32, device="cuda")
    steps = torch.empty(N, dtype=torch.int32, device="cuda")
    dU, dX = _dev(U), _dev(x0s)
    ctx.rollout_batch(dU.data_ptr(), dX.data_ptr(), 1, N, H, mp.DUMP_LIFTED, traj.data_ptr(), steps.data_ptr(), 0, tick=tick)
    torch.cuda.synchronize()
    g_steps, g_traj = steps.cpu().numpy(), traj.cpu().numpy()
    r_steps, r_marg, r_traj = o.rollout_batch(U, x0s, want_traj=True, tick=tick)
    bad, nrobust = check_flags(g_steps, r_steps, r_marg, H)
    assert len(bad) == 0, (bad[:5], g_steps[bad[:5]], r_steps[bad[:5]], r_marg[bad[:5]])
    assert nrobust > 0.9 * N and 0.05 < (r_steps == H).mean() < 0.95
    worst = 0.0
    for i in range(N):
        e_gpu = min(g_steps[i] + 1, H)
        worst = max(worst, traj_rel_err(g_traj[:, :, i], r_traj[i], min(r_steps[i] + 1, e_gpu)))
        assert np.all(np.isfinite(g_traj[:e_gpu, :, i])) and np.all(np.isnan(g_traj[e_gpu:, :, i]))
    assert worst <= TRAJ_RTOL, worst


def test_tile64_noise_tick(mp):
    """rollout_tile_kernel<64, 3, TICK, NOISE>: whole tick with prediction noise at padded d = 64."""
    w = W.make("T48", N=3000)
    w.noise_sigma = 0.01
    ctx = mp.Context(w)
    assert ctx.info()["variant"] == 2
    o = _oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 4)
    for x0, uu, t in zip(x0s, uus, ticks):
        compare_tick(mp, ctx, o, w, x0, uu, t)


# ------------------------------------------------------------------ flag combinations --------------------
def test_affine_and_tensor32_flags_together(mp):
    """MPMI_VARIANT_AFFINE | MPMI_VARIANT_TENSOR32 must be one consistent tick (the affine kernel finalises itself:
    no second pass may run after it), equal to the default tick on every field."""
    V = mp.mpmi
    w = W.make("C4", N=1 << 17)
    both = mp.Context(w, variant=V.VARIANT_AFFINE | V.VARIANT_TENSOR32)
    plain = mp.Context(w, variant=V.VARIANT_NO_TENSOR)
    assert both.info()["variant"] == 6
    o = _oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 4)
    for x0, uu, t in zip(x0s, uus, ticks):
        a = both.step_sync(x0, uu, int(t)).as_dict(w.m)
        b = plain.step_sync(x0, uu, int(t)).as_dict(w.m)
        ref = o.step(x0, uu, int(t), detail=True)
        assert accept_selection(a, ref, w.H)[0] and a["index"] >= 0
        if (ref["margin_all"] > MARGIN).all():
            assert (a["index"], a["safe"], a["steps"], a["n_safe"], a["n_exec"]) == (b["index"], b["safe"], b["steps"], b["n_safe"], b["n_exec"])
        compare_tick(mp, both, o, w, x0, uu, t)
