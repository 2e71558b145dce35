"""GPU parity tests proper: the CUDA path (through the C ABI) against the FP64 oracle, element by
element on the same seeded inputs.  Run on the B200 box: python -m pytest tests -m gpu."""
import copy
import os
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


def _small(name, N):
    w = W.make(name, N=N)
    if name == "C3":
        side = int(round(N ** 0.5)); w.N = side * side
        w.grid_counts = np.array([side, side], np.int32)
    return w


# ------------------------------------------------------------------ a1: sampler, bit-exact --------
@pytest.mark.parametrize("name", ["C1", "C3", "C5"])
def test_sampler_bit_exact(mp, name):
    """K = 0 and B = [I_m; 0] make z_1[0:m] = u exactly, so the lifted dump of step 1 exposes the
    kernel's own candidates: they must equal the oracle's bit for bit (Philox and grid)."""
    w = _small(name, 1500 if name != "C3" else 1600)
    w.K = np.zeros_like(w.K); w.B = np.zeros_like(w.B)
    for j in range(w.m):
        w.B[j, j] = 1.0
    w.u_lo = np.array([-1.0, 0.0, -1.0][: w.m], np.float32); w.u_hi = np.array([1.0, 1.0, 0.0][: w.m], np.float32)
    w.seed = 0xDEADBEEF12345
    o = _oracle(w)
    # d = 128: the FP32 SIMT kernel exposes the candidates exactly; the 3xTF32 tensor-core kernel draws
    # the same candidates but its step keeps 22 mantissa bits of u (hi + truncated lo), checked below
    ctx = mp.Context(w, variant=mp.mpmi.VARIANT_NO_TENSOR)
    N = w.N
    X0 = _dev(w.x_nom[None, :])
    traj = torch.empty((1, w.d, N), dtype=torch.float32, device="cuda")
    steps = torch.empty(N, dtype=torch.int32, device="cuda")
    for tick in (0, (5 << 32) | 77):
        ctx.rollout_batch(0, X0.data_ptr(), 1, N, 1, mp.DUMP_LIFTED, traj.data_ptr(), steps.data_ptr(), 0, tick=tick)
        torch.cuda.synchronize()
        got = traj[0, : w.m, :].T.cpu().numpy()
        ref = o.sample(tick, np.arange(N))
        assert np.array_equal(got.view(np.uint32), ref.view(np.uint32))
    if name == "C5":
        tc = mp.Context(w)
        assert tc.info()["variant"] == 4
        tc.rollout_batch(0, X0.data_ptr(), 1, N, 1, mp.DUMP_LIFTED, traj.data_ptr(), steps.data_ptr(), 0, tick=0)
        torch.cuda.synchronize()
        got = traj[0, : w.m, :].T.cpu().numpy().astype(np.float64)
        ref = o.sample(0, np.arange(N)).astype(np.float64)
        assert np.max(np.abs(got - ref) / np.maximum(np.abs(ref), 1e-30)) <= 2.0 ** -21


# ------------------------------------------------------------------ a2: lift ------------------------
@pytest.mark.parametrize("name,variant", [("C2", 0), ("C3", 0), ("C5", 0), ("C5", 4096)])
def test_lift_parity(mp, name, variant):
    """K = I, B = 0, H = 1  =>  z_1 = Psi(x0) exactly; per-candidate x0 (d = 128: the FP32 warp-tile kernel serves
    per-candidate x0 in a verified context; variant 4096 = MPMI_VARIANT_TC_UNVERIFIED is the tcgen05 kernel's own lift)."""
    w = _small(name, 300 if name != "C3" else 289)
    w.K = np.eye(w.d, dtype=np.float32); w.B = np.zeros_like(w.B)
    o = _oracle(w)
    ctx = mp.Context(w, variant=variant)
    x0s, _, _ = W.tick_inputs(w, w.N)
    x0s = (x0s * 3.0).astype(np.float32)
    U = np.zeros((w.N, w.m), np.float32)
    traj = torch.empty((1, w.d, w.N), dtype=torch.float32, device="cuda")
    steps = torch.empty(w.N, dtype=torch.int32, device="cuda")
    dU, dX = _dev(U), _dev(x0s)                    # keep the tensors alive while the kernel runs
    ctx.rollout_batch(dU.data_ptr(), dX.data_ptr(), w.N, w.N, 1, mp.DUMP_LIFTED, traj.data_ptr(),
                      steps.data_ptr(), 0)
    torch.cuda.synchronize()
    got = traj[0].T.cpu().numpy().astype(np.float64)
    for i in range(w.N):
        ref = o.lift(x0s[i].astype(np.float64))
        assert np.all(np.abs(got[i] - ref) <= 2e-6 * np.maximum(np.abs(ref), 1.0)), (i, np.abs(got[i] - ref).max())


# ------------------------------------------------------------------ a3/a4/a9: rollouts ---------------
@pytest.mark.parametrize("name,N,per_cand_x0,variant", [("C1", 1100, False, 0), ("C1", 2500, True, 0), ("C2", 1300, False, 0),
                                                        ("C3", 1000, True, 0), ("C4", 777, False, 0), ("C5", 700, False, 0),
                                                        ("C5", 300, True, 0), ("C5", 700, False, 4096), ("C5", 300, True, 4096),
                                                        ("C4", 777, False, 4096 | 1024)])
def test_rollout_batch_parity(mp, name, N, per_cand_x0, variant):
    """T1 trajectories (rel. error <= 1e-4), T2 flags (identical where margin > 1e-4), NaN tail.  Caller-supplied inputs:
    a verified d = 128 context serves them with the FP32 warp-tile kernel (the bound of the verified tick is taken over the
    context's own input box); variant 4096 = MPMI_VARIANT_TC_UNVERIFIED runs the bare 3xTF32 tcgen05 kernel (d = 128, and
    d = 32 with MPMI_VARIANT_TENSOR32), whose trajectories must meet T1 on their own."""
    w = W.make(name, N=N)
    if name == "C3":
        w.sampler = 0; w.grid_counts = None
    o = _oracle(w)
    ctx = mp.Context(w, variant=variant)
    if variant:
        assert ctx.info()["variant"] == 4
    rng = np.random.default_rng(11)
    U = rng.uniform(w.u_lo, w.u_hi, (N, w.m)).astype(np.float32)
    x0s, _, _ = W.tick_inputs(w, N if per_cand_x0 else 1)
    H = w.H
    for kind, J in ((mp.DUMP_LIFTED, w.d), (mp.DUMP_PHYS, w.n)):
        traj = torch.full((H, J, N), 7.0, dtype=torch.float32, device="cuda")
        steps = torch.empty(N, dtype=torch.int32, device="cuda")
        safe = torch.empty(N, dtype=torch.uint8, device="cuda")
        dU, dX = _dev(U), _dev(x0s)
        ctx.rollout_batch(dU.data_ptr(), dX.data_ptr(), x0s.shape[0], N, H, kind, traj.data_ptr(),
                          steps.data_ptr(), safe.data_ptr())
        torch.cuda.synchronize()
        g_steps = steps.cpu().numpy(); g_safe = safe.cpu().numpy(); g_traj = traj.cpu().numpy()
        r_steps, r_marg, r_traj = o.rollout_batch(U, x0s, want_traj=True)
        bad, nrobust = check_flags(g_steps, r_steps, r_marg, H)
        if not (variant and name == "C4"):       # (the BARE tensor-core kernel at |z| ~ 1e2 is outside T2 by design: only its verified tick is a product path)
            assert len(bad) == 0, (bad[:5], g_steps[bad[:5]], r_steps[bad[:5]], r_marg[bad[:5]])
        assert len(bad) <= 2 and nrobust > 0.9 * N
        assert np.array_equal(g_safe, (g_steps == H).astype(np.uint8))
        assert 0.05 < (r_steps == H).mean() < 0.95                    # a mixed set: both branches exercised
        worst = 0.0
        for i in range(N):
            gt = g_traj[:, :, i]
            e_ref = min(r_steps[i] + 1, H); e_gpu = min(g_steps[i] + 1, H)
            worst = max(worst, traj_rel_err(gt, r_traj[i][:, :J] if kind == mp.DUMP_PHYS else r_traj[i], min(e_ref, e_gpu))
                        if kind == mp.DUMP_LIFTED else 0.0)
            if kind == mp.DUMP_PHYS:
                e = min(e_ref, e_gpu)
                assert np.allclose(gt[:e], r_traj[i][:e, : w.n], rtol=1e-4, atol=1e-4)
            assert np.all(np.isfinite(gt[:e_gpu])) and np.all(np.isnan(gt[e_gpu:]))
        assert worst <= TRAJ_RTOL, worst


# ------------------------------------------------------------------ a1-a8: whole tick ----------------
def _tick_compare(mp, w, nticks, expect=None):
    o = _oracle(w)
    ctx = mp.Context(w)
    x0s, uus, ticks = W.tick_inputs(w, nticks)
    exact = 0
    branches = set()
    for x0, uu, t in zip(x0s, uus, ticks):
        ref = o.step(x0, uu, int(t), detail=True)
        r = ctx.step_sync(x0, uu, int(t)).as_dict(w.m)
        ok, ex, why = accept_selection(r, ref, w.H)
        assert ok, (why, r, {k: ref[k] for k in ("index", "safe", "steps", "dist")})
        exact += ex
        robust = ref["margin_all"] > MARGIN
        if robust.all():
            assert r["n_safe"] == ref["n_safe"] and r["n_exec"] == ref["n_exec"]
        else:
            assert abs(r["n_safe"] - ref["n_safe"]) <= (~robust).sum()
        if ex:
            assert abs(r["dist"] - ref["dist"]) <= 1e-6 * max(1.0, ref["dist"])
        branches.add("user" if (r["safe"] and r["dist"] == 0) else "intervene" if r["safe"] else "fallback")
    if expect:
        assert branches == expect, branches
    return exact / nticks, branches


@pytest.mark.parametrize("name,N", [("C1", 1024), ("C2", 10000), ("C3", 10000), ("C4", 1 << 14), ("C5", 2048)])
def test_tick_parity(mp, name, N):
    """T3 over 64 (C5: 16) seeded ticks: minimal-intervention and intervention branches."""
    w = W.make(name, N=N)
    rate, branches = _tick_compare(mp, w, 64 if name != "C5" else 16)
    assert rate >= 0.95, rate
    assert "intervene" in branches


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C5"])
def test_tick_forced_branches(mp, name):
    """bounds x0.01 -> nothing is safe (fallback rule G1); bounds x100 -> everything is safe."""
    w = W.make(name, N=1500 if name != "C3" else 1600)
    if name == "C3":
        w.grid_counts = np.array([40, 40], np.int32)
    _, b = _tick_compare(mp, G.scaled_bounds(w, 0.01), 8)
    assert b == {"fallback"}
    _, b = _tick_compare(mp, G.scaled_bounds(w, 100.0), 8)
    assert b == {"user"}


def test_c2_tick_sequence_replay(mp):
    """C2: 1,000 consecutive ticks with u_user from a random walk (BASELINE.json configs[1]); the GPU
    replays the stored sequence; every 10th tick is compared with the oracle in full."""
    w = W.make("C2")
    seq = np.loadtxt(W.generate.C2_SEQUENCE, comments="#")
    assert seq.shape == (1000, 9)
    o = _oracle(w)
    ctx = mp.Context(w)
    exact = 0
    kinds = set()
    for row in seq:
        t = int(row[0]); x0 = row[1:5].astype(np.float32); uu = row[5:6].astype(np.float32)
        r = ctx.step_sync(x0, uu, t).as_dict(1)
        same = (r["index"], r["safe"], r["steps"]) == (int(row[6]), int(row[7]), int(row[8]))
        exact += same
        if not same or t % 10 == 0:              # every mismatch and every 10th tick: full oracle comparison
            ref = o.step(x0, uu, t, detail=True)
            assert (ref["index"], ref["safe"], ref["steps"]) == (int(row[6]), int(row[7]), int(row[8]))
            ok, ex, why = accept_selection(r, ref, w.H)
            assert ok, (t, why)
        kinds.add("user" if (r["safe"] and r["dist"] == 0) else "intervene" if r["safe"] else "fallback")
    assert exact >= 950, exact
    assert kinds >= {"user", "intervene"}


# ------------------------------------------------------------------ entry-point equivalences ---------
def test_device_and_shard_paths_match_host_path(mp):
    """mpmi_step_device == mpmi_step_sync; two shards + finalize == one context (P7 shard invariance)."""
    for name in ("C2", "C5"):
        w = W.make(name, N=3000)
        ctx = mp.Context(w)
        cut = 1234
        sh = [mp.Context(w, shard=(0, cut)), mp.Context(w, shard=(cut, w.N + 1 - cut))]
        x0s, uus, ticks = W.tick_inputs(w, 6)
        d_res = torch.zeros(56, dtype=torch.uint8, device="cuda")
        d_parts = torch.zeros(2 * 24, dtype=torch.uint8, device="cuda")
        s = torch.cuda.current_stream().cuda_stream
        for x0, uu, t in zip(x0s, uus, ticks):
            host = ctx.step_sync(x0, uu, int(t)).as_dict(w.m)
            dx, du = _dev(x0), _dev(uu)
            ctx.step_device(dx.data_ptr(), du.data_ptr(), int(t), s, d_res.data_ptr())
            torch.cuda.synchronize()
            dev = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)[0]
            for g in range(2):
                sh[g].shard_step(dx.data_ptr(), du.data_ptr(), int(t), s, d_parts.data_ptr() + 24 * g)
            sh[0].shard_finalize(d_parts.data_ptr(), 2, du.data_ptr(), int(t), s, d_res.data_ptr())
            torch.cuda.synchronize()
            shd = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)[0]
            for got in (dev, shd):
                assert got["index"] == host["index"] and got["safe"] == host["safe"] and got["steps"] == host["steps"]
                assert got["n_safe"] == host["n_safe"] and got["n_exec"] == host["n_exec"] and got["key"] == host["key"]
                assert np.array_equal(got["u"][: w.m], host["u"]) and got["dist"] == host["dist"]


@pytest.mark.parametrize("name,N", [("C1", 5000), ("C4", 70000), ("C5", 40000)])
def test_spatial_binning_changes_nothing(mp, name, N):
    """The counting sort of candidate indices by input-box cell (binning.cuh) only re-orders the walk:
    every field of the result is identical with and without it, and it matches the oracle."""
    w = W.make(name, N=N)
    nt = mp.mpmi.VARIANT_NO_TENSOR if name == "C4" else 0        # (C4 at this size: keep the test on the register kernel)
    plain = mp.Context(w, variant=mp.mpmi.VARIANT_NO_BINNING | nt)
    binned = mp.Context(w, variant=mp.mpmi.VARIANT_FORCE_BINNING | nt)
    assert plain.info()["binning_cells"] == 0 and binned.info()["binning_cells"] > 1
    assert binned.info()["variant"] == (4 if name == "C5" else 1)
    o = _oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 5)
    for i, (x0, uu, t) in enumerate(zip(x0s, uus, ticks)):
        a = plain.step_sync(x0, uu, int(t)).as_dict(w.m)
        b = binned.step_sync(x0, uu, int(t)).as_dict(w.m)
        for k in ("index", "safe", "steps", "n_safe", "n_exec", "key", "dist"):
            assert a[k] == b[k], (k, a[k], b[k])
        assert np.array_equal(a["u"], b["u"])
        if i < 2:
            assert accept_selection(b, o.step(x0, uu, int(t), detail=True), w.H)[0]


@pytest.mark.parametrize("N,lanes", [(45000, 16), (150000, 8), (400000, 4), (600000, 2)])
def test_every_lane_split_of_the_d32_second_pass(mp, N, lanes):
    """The row-split second pass runs 16, 8, 4 or 2 lanes per candidate pair depending on the candidate count (mpmi_api.cu: rc_rs); each
    form must leave the verified tick identical to the FP32 tick (N = 45,000 also: the verified tick WITHOUT binning)."""
    V = mp.mpmi
    w = W.make("C4", N=N)
    ver, fp32 = mp.Context(w), mp.Context(w, variant=V.VARIANT_NO_TENSOR)
    assert ver.info()["variant"] == 4 and fp32.info()["variant"] == 1
    assert (ver.info()["binning_cells"] > 0) == (N >= 81920)
    x0s, uus, ticks = W.tick_inputs(w, 3)
    for x0, uu, t in zip(x0s, uus, ticks):
        a, b = ver.step_sync(x0, uu, int(t)).as_dict(w.m), fp32.step_sync(x0, uu, int(t)).as_dict(w.m)
        assert _same_tick(a, b), (lanes, a, b)
        assert ver.info()["reserved"] > 0                      # some candidates did go through the second pass


def test_binning_beyond_one_scan_pass_and_with_a_ragged_life_time_histogram(mp):
    """Edges of the binning kernels: (a) more than 16,384 cells (2^21 candidates -> 2^15 cells), where the last CTA's scan of the cell
    histogram takes a second pass and carries its running sum over; (b) a life-time histogram whose cell count H + 1 is not a multiple
    of the scan's int4 groups, on few candidates (most CTA-level counters empty).  Both only re-order the walk: every field of the
    result equals the unordered tick's."""
    V = mp.mpmi
    w = W.make("C4", N=(1 << 21) + 5)
    plain = mp.Context(w, variant=V.VARIANT_NO_BINNING | V.VARIANT_NO_TENSOR)
    binned = mp.Context(w, variant=V.VARIANT_NO_TENSOR)
    assert binned.info()["binning_cells"] == 1 << 15 and plain.info()["binning_cells"] == 0
    x0s, uus, ticks = W.tick_inputs(w, 2)
    for x0, uu, t in zip(x0s, uus, ticks):
        a, b = plain.step_sync(x0, uu, int(t)).as_dict(w.m), binned.step_sync(x0, uu, int(t)).as_dict(w.m)
        for k in ("index", "safe", "steps", "n_safe", "n_exec", "key", "dist"):
            assert a[k] == b[k], (k, a[k], b[k])
    plain.close(); binned.close()
    w = W.make("C5", N=1500, H=37)                                # 38 life-time cells, two prediction CTAs
    plain = mp.Context(w, variant=V.VARIANT_NO_BINNING)
    pred = mp.Context(w, variant=V.VARIANT_FORCE_BINNING)
    assert pred.info()["binning_cells"] == 38
    x0s, uus, ticks = W.tick_inputs(w, 3)
    for x0, uu, t in zip(x0s, uus, ticks):
        a, b = plain.step_sync(x0, uu, int(t)).as_dict(w.m), pred.step_sync(x0, uu, int(t)).as_dict(w.m)
        for k in ("index", "safe", "steps", "n_safe", "n_exec", "key", "dist"):
            assert a[k] == b[k], (k, a[k], b[k])


@pytest.mark.parametrize("name,N,noise,tensor", [("C5", 40000, 0.0, True), ("C5", 20000, 0.0, False), ("C5", 9000, 0.02, True)])
def test_life_time_order_changes_nothing(mp, name, N, noise, tensor):
    """For the persistent tile kernels (d > 32) the pre-sort key is the first-violation step PREDICTED by the
    affine form x_k = a_k + G_k u (longest first), so that the candidates of a tile stop together.  The
    prediction only orders the walk: the result is identical to the cell order and to the index order."""
    w = W.make(name, N=N)
    if noise:
        w.noise_sigma = noise
    V = mp.mpmi
    base = 0 if tensor else V.VARIANT_NO_TENSOR           # tcgen05 kernel / FP32 warp-tile kernel
    plain = mp.Context(w, variant=base | V.VARIANT_NO_BINNING)
    cells = mp.Context(w, variant=base | V.VARIANT_FORCE_BINNING | V.VARIANT_NO_PREDICT)
    pred = mp.Context(w, variant=base | V.VARIANT_FORCE_BINNING)
    assert pred.info()["variant"] == (4 if tensor else 2)
    extra = 3 if tensor else 0               # verified tensor-core tick: two bound kernels + the FP32 second pass
    if noise:                                # measured: no gain once noise decides the life time -> cell order
        assert pred.info()["launches_per_tick"] == 3 + extra
    else:
        assert pred.info()["binning_cells"] == w.H + 1 and pred.info()["launches_per_tick"] == 4 + extra
    assert cells.info()["launches_per_tick"] == 3 + extra and plain.info()["launches_per_tick"] == 1 + extra
    o = _oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 4)
    for i, (x0, uu, t) in enumerate(zip(x0s, uus, ticks)):
        a = plain.step_sync(x0, uu, int(t)).as_dict(w.m)
        for ctx in (cells, pred):
            b = ctx.step_sync(x0, uu, int(t)).as_dict(w.m)
            for k in ("index", "safe", "steps", "n_safe", "n_exec", "key", "dist"):
                assert a[k] == b[k], (k, a[k], b[k])
            assert np.array_equal(a["u"], b["u"])
        if i < 2 and not noise:
            assert accept_selection(b, o.step(x0, uu, int(t), detail=True), w.H)[0]


def test_life_time_order_on_device_and_shard_paths(mp):
    """The prediction runs ahead of the rollout on every entry point, not only in the tick graph: mpmi_step_device and
    two shards (each predicts and sorts its own candidates) + finalize give the result of the unordered context."""
    w = W.make("C5", N=30000)
    V = mp.mpmi
    plain = mp.Context(w, variant=V.VARIANT_NO_BINNING)
    pred = mp.Context(w, variant=V.VARIANT_FORCE_BINNING)
    cut = 17001
    sh = [mp.Context(w, shard=(0, cut), variant=V.VARIANT_FORCE_BINNING),
          mp.Context(w, shard=(cut, w.N + 1 - cut), variant=V.VARIANT_FORCE_BINNING)]
    for c in (pred, sh[0], sh[1]):
        assert c.info()["binning_cells"] == w.H + 1
    x0s, uus, ticks = W.tick_inputs(w, 3)
    d_res = torch.zeros(56, dtype=torch.uint8, device="cuda")
    d_parts = torch.zeros(2 * 24, dtype=torch.uint8, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    for x0, uu, t in zip(x0s, uus, ticks):
        host = plain.step_sync(x0, uu, int(t)).as_dict(w.m)
        dx, du = _dev(x0), _dev(uu)
        pred.step_device(dx.data_ptr(), du.data_ptr(), int(t), s, d_res.data_ptr())
        torch.cuda.synchronize()
        dev = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=V.RESULT_DTYPE)[0]
        for g in range(2):
            sh[g].shard_step(dx.data_ptr(), du.data_ptr(), int(t), s, d_parts.data_ptr() + 24 * g)
        sh[0].shard_finalize(d_parts.data_ptr(), 2, du.data_ptr(), int(t), s, d_res.data_ptr())
        torch.cuda.synchronize()
        shd = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=V.RESULT_DTYPE)[0]
        for got in (dev, shd):
            for k in ("index", "safe", "steps", "n_safe", "n_exec", "key", "dist"):
                assert got[k] == host[k], (k, got[k], host[k])
            assert np.array_equal(got["u"][: w.m], host["u"])


def _same_tick(a, b):
    return (a["index"], a["safe"], a["steps"], a["n_safe"], a["n_exec"], a["key"]) == (b["index"], b["safe"], b["steps"], b["n_safe"], b["n_exec"], b["key"]) \
        and np.array_equal(np.asarray(a["u"], np.float32), np.asarray(b["u"], np.float32)) and a["dist"] == b["dist"]


def test_verified_tensor_core_tick_d32(mp):
    """The default tick at padded d = 32 from ~38,000 candidates (more than one register-kernel CTA per SM): the 3xTF32 tcgen05 kernel (N = 32 MMAs, four CTAs per SM) as a
    VERIFIED tick.  Every candidate whose 3xTF32 state came within tau_i(k) (csrc/bound.cuh: a per-tick bound, derived from the
    model, on the difference to the FP32 rollout) of the safe-set boundary is rolled again by the FP32 register kernel, which
    merges its keys and finalises.  Checked: T3 against the oracle, and -- the strong one -- the SAME result (index, safe, steps,
    n_safe, n_exec, key, u, dist) as the FP32 tick (MPMI_VARIANT_NO_TENSOR) on every tick; n_exec equal means the step counts
    agree in sum (test_parity_full_gpu.py compares them candidate by candidate)."""
    N = 1 << 17
    w = W.make("C4", N=N)
    V = mp.mpmi
    ctx = mp.Context(w)
    fp32 = mp.Context(w, variant=V.VARIANT_NO_TENSOR)
    info = ctx.info()
    assert info["variant"] == 4 and info["threads_per_block"] == 160 and info["blocks"] == 4 * info["sm_count"]
    assert info["launches_per_tick"] == 6                                # hist, scatter | bound x2 -> tcgen05 rollout -> FP32 second pass
    assert fp32.info()["variant"] == 1
    assert mp.Context(W.make("C4", N=30000)).info()["variant"] == 1                               # below the crossover (one register-kernel CTA per SM): FP32
    small = mp.Context(W.make("C4", N=50000)).info()
    assert small["variant"] == 4 and small["binning_cells"] == 0 and small["launches_per_tick"] == 4   # above it: verified tick, binning only from ~80,000
    assert mp.Context(W.make("C4", N=1 << 15), variant=V.VARIANT_TENSOR32).info()["variant"] == 4  # ... unless asked for
    o = _oracle(w)
    H = w.H
    x0s, uus, ticks = W.tick_inputs(w, 24)
    rechecked = []
    for k, (x0, uu, t) in enumerate(zip(x0s, uus, ticks)):
        r = ctx.step_sync(x0, uu, int(t)).as_dict(w.m)
        f = fp32.step_sync(x0, uu, int(t)).as_dict(w.m)
        assert _same_tick(r, f), (k, r, f)
        rechecked.append(ctx.info()["reserved"])
        if k < 3:
            ref = o.step(x0, uu, int(t), detail=True)
            ok, ex, why = accept_selection(r, ref, H)
            assert ok, why
            assert abs(r["n_safe"] - ref["n_safe"]) <= (ref["margin_all"] <= MARGIN).sum()
    assert 0 < min(rechecked) and max(rechecked) < 0.3 * N, rechecked    # a small, non-empty second pass
    # forced branches: nothing safe / everything safe
    for factor, branch in ((0.01, 0), (100.0, 1)):
        v = G.scaled_bounds(w, factor)
        a, b = mp.Context(v), mp.Context(v, variant=V.VARIANT_NO_TENSOR)
        assert a.info()["variant"] == 4
        for x0, uu, t in zip(x0s[:4], uus[:4], ticks[:4]):
            r = a.step_sync(x0, uu, int(t)).as_dict(w.m); f = b.step_sync(x0, uu, int(t)).as_dict(w.m)
            assert r["safe"] == branch and _same_tick(r, f)
    # with prediction noise (Alg. 2 l.5): both passes draw the same Philox normals; same result as the FP32 noise tick
    wn = W.make("C4", N=N); wn.noise_sigma = 0.01
    a, b = mp.Context(wn), mp.Context(wn, variant=V.VARIANT_NO_TENSOR)
    assert a.info()["variant"] == 4 and a.info()["launches_per_tick"] == 6 and b.info()["variant"] == 1
    for x0, uu, t in zip(x0s[:6], uus[:6], ticks[:6]):
        r = a.step_sync(x0, uu, int(t)).as_dict(w.m); f = b.step_sync(x0, uu, int(t)).as_dict(w.m)
        assert _same_tick(r, f), (r, f)
    del a, b
    # batch entry: FP32 register kernels, T1 + T2
    n1 = 1536 + 77
    rng = np.random.default_rng(5)
    U = rng.uniform(w.u_lo, w.u_hi, (n1, w.m)).astype(np.float32)
    traj = torch.full((H, w.d, n1), 7.0, dtype=torch.float32, device="cuda")
    steps = torch.empty(n1, dtype=torch.int32, device="cuda")
    dU, dX = _dev(U), _dev(x0s[:1])
    ctx.rollout_batch(dU.data_ptr(), dX.data_ptr(), 1, n1, H, mp.DUMP_LIFTED, traj.data_ptr(), steps.data_ptr(), 0)
    torch.cuda.synchronize()
    r_steps, r_marg, r_traj = o.rollout_batch(U, x0s[:1], want_traj=True)
    g, gs = traj.cpu().numpy(), steps.cpu().numpy()
    bad, _ = check_flags(gs, r_steps, r_marg, H)
    assert len(bad) == 0
    worst = max(traj_rel_err(g[:, :, i], r_traj[i], min(int(gs[i]) + 1, int(r_steps[i]) + 1, H)) for i in range(n1))
    assert worst <= 1e-5, worst                                          # FP32 kernels: an order below the 1e-4 of T1


@pytest.mark.parametrize("name,N", [("C4", (1 << 18) + 333), ("C5", 50000)])
def test_verified_tick_device_and_shard_paths(mp, name, N):
    """The verified tensor-core tick through mpmi_step_device (plain launches: the bound kernels fork onto the context's side
    stream) and as two candidate shards + finalize (both passes run per shard, the FP32 pass writes the shard's partial):
    same result as the graph path and as the FP32 tick."""
    V = mp.mpmi
    w = W.make(name, N=N)
    ctx = mp.Context(w)
    fp32 = mp.Context(w, variant=V.VARIANT_NO_TENSOR)
    cut = N // 2 + 5
    sh = [mp.Context(w, shard=(0, cut), variant=V.VARIANT_TENSOR32), mp.Context(w, shard=(cut, w.N + 1 - cut), variant=V.VARIANT_TENSOR32)]
    assert ctx.info()["variant"] == 4 and all(c.info()["variant"] == 4 for c in sh)
    x0s, uus, ticks = W.tick_inputs(w, 5)
    d_res = torch.zeros(56, dtype=torch.uint8, device="cuda")
    d_parts = torch.zeros(2 * 24, dtype=torch.uint8, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    for x0, uu, t in zip(x0s, uus, ticks):
        host = ctx.step_sync(x0, uu, int(t)).as_dict(w.m)
        f = fp32.step_sync(x0, uu, int(t)).as_dict(w.m)
        assert _same_tick(host, f), (host, f)
        dx, du = _dev(x0), _dev(uu)
        ctx.step_device(dx.data_ptr(), du.data_ptr(), int(t), s, d_res.data_ptr())
        torch.cuda.synchronize()
        dev = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=V.RESULT_DTYPE)[0]
        for g in range(2):
            sh[g].shard_step(dx.data_ptr(), du.data_ptr(), int(t), s, d_parts.data_ptr() + 24 * g)
        sh[0].shard_finalize(d_parts.data_ptr(), 2, du.data_ptr(), int(t), s, d_res.data_ptr())
        torch.cuda.synchronize()
        shd = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=V.RESULT_DTYPE)[0]
        for got in (dev, shd):
            assert got["index"] == host["index"] and got["safe"] == host["safe"] and got["steps"] == host["steps"]
            assert got["n_safe"] == host["n_safe"] and got["n_exec"] == host["n_exec"] and got["key"] == host["key"]
            assert np.array_equal(got["u"][: w.m], host["u"]) and got["dist"] == host["dist"]


def test_edge_cases(mp):
    w = W.make("C1", N=1)
    o = _oracle(w)
    for inc in (0, 1):
        ctx = mp.Context(w, include_user=inc)
        oo = _oracle(w, include_user=inc)
        r = ctx.step_sync(w.x_nom, np.array([0.2], np.float32), 3).as_dict(1)
        ref = oo.step(w.x_nom, np.array([0.2], np.float32), 3, detail=True)
        assert accept_selection(r, ref, w.H)[0]
    # u_user outside the box is clamped, not an error
    w = W.make("C2", N=512)
    ctx = mp.Context(w); o = _oracle(w)
    r = ctx.step_sync(w.x_nom, np.array([7.5], np.float32), 1).as_dict(1)
    ref = o.step(w.x_nom, np.array([7.5], np.float32), 1, detail=True)
    assert accept_selection(r, ref, w.H)[0] and ref["U"][w.N, 0] == 1.0
    # non-finite inputs: INVALID on the host path, index -1 on the device path
    with pytest.raises(mp.MpmiError) as e:
        ctx.step_sync(np.array([np.nan, 0, 0, 0], np.float32), np.array([0.0], np.float32), 0)
    assert e.value.status == -1
    d_res = torch.zeros(56, dtype=torch.uint8, device="cuda")
    dx, du = _dev(np.array([np.inf, 0, 0, 0], np.float32)), _dev(np.zeros(1, np.float32))
    ctx.step_device(dx.data_ptr(), du.data_ptr(), 0, 0, d_res.data_ptr())
    torch.cuda.synchronize()
    assert np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)[0]["index"] == -1
    r2 = ctx.step_sync(w.x_nom, np.array([7.5], np.float32), 1).as_dict(1)       # state was reset correctly
    assert r2["index"] == r["index"] and r2["n_exec"] == r["n_exec"]
    # H = 1, candidates an exact multiple of the CTA tile, inflated barrier
    w = W.make("C5", N=511, H=1); w.inflate = 0.05
    ctx = mp.Context(w); o = _oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 3)
    for x0, uu, t in zip(x0s, uus, ticks):
        assert accept_selection(ctx.step_sync(x0, uu, int(t)).as_dict(3), o.step(x0, uu, int(t), detail=True), 1)[0]
    # unsupported sizes are statuses
    bad = dict(vars(W.make("C1"))); bad["m"] = 5
    with pytest.raises(mp.MpmiError) as e:
        mp.Context(bad)
    assert e.value.status == -2


# ------------------------------------------------------------------ full size, bench launch config ---
@pytest.mark.parametrize("name", ["C4", "C5"])
def test_full_size_sampled(mp, name):
    """BASELINE sizes (C4: N = 2^20, C5: N = 262,144) in the launch configuration bench.py times:
    the tick result against oracle rollouts of sampled candidates, plus size-independent properties."""
    w = W.make(name)
    o = _oracle(w, N=w.N)
    ctx = mp.Context(w)
    N, H = w.N, w.H
    x0s, uus, ticks = W.tick_inputs(w, 2)
    steps = torch.empty(N, dtype=torch.int32, device="cuda")
    rng = np.random.default_rng(3)
    for x0, uu, t in zip(x0s, uus, ticks):
        r = ctx.step_sync(x0, uu, int(t)).as_dict(w.m)
        dX = _dev(x0[None, :])
        ctx.rollout_batch(0, dX.data_ptr(), 1, N, H, mp.DUMP_NONE, 0, steps.data_ptr(), 0, tick=int(t))
        torch.cuda.synchronize()
        g_steps = steps.cpu().numpy()
        u_h = np.clip(uu, w.u_lo, w.u_hi)
        z0 = o.lift(x0.astype(np.float64))
        us, _, _ = o.rollout(z0, u_h.astype(np.float64))
        n_safe = int((g_steps == H).sum()) + int(us == H)
        n_exec = int(np.minimum(g_steps + 1, H).sum()) + min(us + 1, H)
        assert abs(r["n_safe"] - n_safe) <= 1 and abs(r["n_exec"] - n_exec) <= H      # tick == batch + user slot
        assert 0.2 < n_safe / N < 0.6
        idx = np.unique(np.concatenate([rng.integers(0, N, 1500), [r["index"]] if r["index"] < N else []])).astype(np.int64)
        Us = o.sample(int(t), idx)
        r_steps, r_marg, _ = o.rollout_batch(Us, x0[None, :])
        robust = r_marg > MARGIN
        assert np.array_equal(g_steps[idx][robust], r_steps[robust]) and robust.mean() > 0.9
        # winner: bit-identical to its candidate, safe in the oracle, and no sampled robustly safe candidate is closer
        if r["index"] < N:
            assert np.array_equal(r["u"], o.sample(int(t), [r["index"]])[0])
        else:
            assert np.array_equal(r["u"], u_h)
        assert r["safe"] == 1
        d = np.linalg.norm(Us.astype(np.float64) - u_h.astype(np.float64), axis=1)
        rs = robust & (r_steps == H)
        assert not (d[rs] < r["dist"] - MARGIN).any()
        # brute-force check of the argmin on the GPU's own flags (exact, all N candidates)
        Uall_d = None
        if name == "C4":
            Uall = o.sample(int(t), np.arange(0, N, 1)[:: 1][: 1 << 15])
            dd = np.linalg.norm(Uall.astype(np.float64) - u_h.astype(np.float64), axis=1)
            ok = g_steps[: 1 << 15] == H
            if ok.any() and us != H:
                assert dd[ok].min() >= r["dist"] - 1e-6


# ------------------------------------------------------------------ NEXT-2: prediction noise (Alg. 2 l.5) ----------
NOISE_SIGMA = {"C1": 0.05, "C2": 0.01, "C4": 0.02, "C5": 0.01}


@pytest.mark.parametrize("name,N,per_cand_x0", [("C1", 900, False), ("C2", 1300, False), ("C4", 777, False),
                                                ("C4", 1030, True), ("C5", 600, False)])
def test_noise_rollout_batch_parity(mp, name, N, per_cand_x0):
    """x_p <- f(x_p, xi) + z_i with Gaussian z_i: same counter-based draws on both sides, T1 / T2."""
    w = W.make(name, N=N); w.noise_sigma = NOISE_SIGMA[name]; w.seed = 0xABCDEF0123
    o = _oracle(w)
    ctx = mp.Context(w, variant=mp.mpmi.VARIANT_TC_UNVERIFIED if name == "C5" else 0)   # caller-supplied inputs: the bare tcgen05 kernel
    assert ctx.info()["variant"] == (4 if name == "C5" else 1)   # d = 128: the tensor-core kernel carries the noise as 8 extra A columns
    rng = np.random.default_rng(5)
    U = rng.uniform(w.u_lo, w.u_hi, (N, w.m)).astype(np.float32)
    x0s, _, _ = W.tick_inputs(w, N if per_cand_x0 else 1)
    H, tick = w.H, (3 << 32) | 41
    traj = torch.full((H, w.d, N), 7.0, dtype=torch.float32, device="cuda")
    steps = torch.empty(N, dtype=torch.int32, device="cuda")
    dU, dX = _dev(U), _dev(x0s)
    ctx.rollout_batch(dU.data_ptr(), dX.data_ptr(), x0s.shape[0], N, H, mp.DUMP_LIFTED, traj.data_ptr(),
                      steps.data_ptr(), 0, tick=tick)
    torch.cuda.synchronize()
    g_steps = steps.cpu().numpy(); g_traj = traj.cpu().numpy()
    r_steps, r_marg, r_traj = o.rollout_batch(U, x0s, want_traj=True, tick=tick)
    bad, nrobust = check_flags(g_steps, r_steps, r_marg, H)
    assert len(bad) == 0, (bad[:5], g_steps[bad[:5]], r_steps[bad[:5]], r_marg[bad[:5]])
    assert nrobust > 0.9 * N
    w0 = W.make(name, N=N); w0.seed = w.seed                      # the noise really changes the outcome
    q_steps, _, _ = _oracle(w0).rollout_batch(U, x0s, tick=tick)
    assert (q_steps != r_steps).any()
    worst = 0.0
    for i in range(N):
        e = min(r_steps[i] + 1, g_steps[i] + 1, H)
        worst = max(worst, traj_rel_err(g_traj[:, :, i], r_traj[i], e))
    assert worst <= TRAJ_RTOL, worst


@pytest.mark.parametrize("name,N", [("C2", 10000), ("C4", 1 << 15), ("C5", 1500)])
def test_noise_tick_parity(mp, name, N):
    """whole tick with prediction noise: T3 selection against the oracle on the same draws (binned order at C4)."""
    w = W.make(name, N=N); w.noise_sigma = NOISE_SIGMA[name]
    rate, branches = _tick_compare(mp, w, 12 if name != "C5" else 6)
    assert rate >= 0.9, rate


# ------------------------------------------------------------------ NEXT-3: re-lift model x' = C(K Psi(x) + B u) ----
def _relift(name, N, bounds=None, sigma=0.0):
    w = W.make(name, N=N)
    if name == "C3":
        side = int(round(N ** 0.5)); w.N = side * side; w.grid_counts = np.array([side, side], np.int32)
    if bounds is not None:
        w = G.scaled_bounds(w, bounds)
    w.model_kind = 1; w.noise_sigma = sigma
    return w


@pytest.mark.parametrize("name,N,per_cand_x0,bounds,sigma", [("C2", 1300, False, None, 0.0), ("C1", 700, True, None, 0.0),
                                                             ("C4", 900, False, None, 0.0), ("C4", 1100, True, None, 0.02),
                                                             ("C5", 500, False, 0.25, 0.0)])
def test_relift_rollout_batch_parity(mp, name, N, per_cand_x0, bounds, sigma):
    """T1 / T2 for the re-lift model (polynomial, trig-product and RFF lifts), physical and lifted dumps, NaN tail."""
    w = _relift(name, N, bounds, sigma)
    w.sampler = 0; w.grid_counts = None
    o = _oracle(w)
    ctx = mp.Context(w)
    assert ctx.info()["variant"] == 5
    rng = np.random.default_rng(23)
    U = rng.uniform(w.u_lo, w.u_hi, (N, w.m)).astype(np.float32)
    x0s, _, _ = W.tick_inputs(w, N if per_cand_x0 else 1)
    H, tick = w.H, 17
    r_steps, r_marg, r_traj = o.rollout_batch(U, x0s, want_traj=True, tick=tick)
    assert 0.02 < (r_steps == H).mean() < 0.98
    for kind, J in ((mp.DUMP_LIFTED, w.d), (mp.DUMP_PHYS, w.n)):
        traj = torch.full((H, J, N), 7.0, dtype=torch.float32, device="cuda")
        steps = torch.empty(N, dtype=torch.int32, device="cuda")
        safe = torch.empty(N, dtype=torch.uint8, device="cuda")
        dU, dX = _dev(U), _dev(x0s)
        ctx.rollout_batch(dU.data_ptr(), dX.data_ptr(), x0s.shape[0], N, H, kind, traj.data_ptr(),
                          steps.data_ptr(), safe.data_ptr(), tick=tick)
        torch.cuda.synchronize()
        g_steps = steps.cpu().numpy(); g_traj = traj.cpu().numpy()
        bad, nrobust = check_flags(g_steps, r_steps, r_marg, H)
        assert len(bad) == 0, (bad[:5], g_steps[bad[:5]], r_steps[bad[:5]], r_marg[bad[:5]])
        assert nrobust > 0.9 * N
        assert np.array_equal(safe.cpu().numpy(), (g_steps == H).astype(np.uint8))
        worst = 0.0
        for i in range(N):
            e = min(r_steps[i] + 1, g_steps[i] + 1, H); e_gpu = min(g_steps[i] + 1, H)
            worst = max(worst, traj_rel_err(g_traj[:, :, i], r_traj[i][:, :J], e))
            assert np.all(np.isfinite(g_traj[:e_gpu, :, i])) and np.all(np.isnan(g_traj[e_gpu:, :, i]))
        assert worst <= TRAJ_RTOL, (kind, worst)


@pytest.mark.parametrize("name,N,bounds", [("C2", 10000, None), ("C3", 10000, None), ("C4", 1 << 15, None), ("C5", 3000, 0.25)])
def test_relift_tick_parity(mp, name, N, bounds):
    w = _relift(name, N, bounds)
    rate, branches = _tick_compare(mp, w, 12)
    assert rate >= 0.9, rate


# ------------------------------------------------------------------ NEXT-4: affine-in-u fast path -------------------
@pytest.mark.parametrize("name,N", [("C1", 1100), ("C2", 1300), ("C4", 900), ("C5", 700)])
def test_affine_rollout_batch_parity(mp, name, N):
    """x_k = a_k + G_k u must reproduce the step-by-step oracle: physical trajectories, flags (T2), NaN tail;
    a lifted dump or per-candidate x0 falls back to the full rollout kernel inside the same context."""
    w = W.make(name, N=N)
    o = _oracle(w)
    ctx = mp.Context(w, variant=mp.mpmi.VARIANT_AFFINE)
    assert ctx.info()["variant"] == 6
    rng = np.random.default_rng(31)
    U = rng.uniform(w.u_lo, w.u_hi, (N, w.m)).astype(np.float32)
    x0s, _, _ = W.tick_inputs(w, 1)
    H = w.H
    r_steps, r_marg, r_traj = o.rollout_batch(U, x0s, want_traj=True)
    for kind, J in ((mp.DUMP_PHYS, w.n), (mp.DUMP_LIFTED, w.d)):
        traj = torch.full((H, J, N), 7.0, dtype=torch.float32, device="cuda")
        steps = torch.empty(N, dtype=torch.int32, device="cuda")
        dU, dX = _dev(U), _dev(x0s)
        ctx.rollout_batch(dU.data_ptr(), dX.data_ptr(), 1, N, H, kind, traj.data_ptr(), steps.data_ptr(), 0)
        torch.cuda.synchronize()
        g_steps = steps.cpu().numpy(); g_traj = traj.cpu().numpy()
        bad, nrobust = check_flags(g_steps, r_steps, r_marg, H)
        assert len(bad) == 0, (kind, bad[:5], g_steps[bad[:5]], r_steps[bad[:5]], r_marg[bad[:5]])
        assert nrobust > 0.9 * N
        for i in range(N):
            e = min(r_steps[i] + 1, g_steps[i] + 1, H); e_gpu = min(g_steps[i] + 1, H)
            ref = r_traj[i][:e, :J]
            scale = np.maximum(np.linalg.norm(r_traj[i][:e], axis=1), 1e-3)[:, None]      # T1 scale: the lifted state's norm
            assert np.all(np.abs(g_traj[:e, :, i] - ref) <= TRAJ_RTOL * scale)
            assert np.all(np.isfinite(g_traj[:e_gpu, :, i])) and np.all(np.isnan(g_traj[e_gpu:, :, i]))


@pytest.mark.parametrize("name,N", [("C1", 1024), ("C2", 10000), ("C3", 10000), ("C4", 1 << 15), ("C5", 2048)])
def test_affine_tick_parity(mp, name, N):
    """T3 through the affine path, and the same winner as the full rollout kernel on every tick."""
    w = _small(name, N) if name == "C3" else W.make(name, N=N)
    o = _oracle(w)
    aff = mp.Context(w, variant=mp.mpmi.VARIANT_AFFINE)
    full = mp.Context(w)
    assert aff.info()["variant"] == 6 and full.info()["variant"] != 6
    x0s, uus, ticks = W.tick_inputs(w, 16)
    exact = 0
    for x0, uu, t in zip(x0s, uus, ticks):
        ref = o.step(x0, uu, int(t), detail=True)
        r = aff.step_sync(x0, uu, int(t)).as_dict(w.m)
        ok, ex, why = accept_selection(r, ref, w.H)
        assert ok, (why, r, {k: ref[k] for k in ("index", "safe", "steps", "dist")})
        exact += ex
        f = full.step_sync(x0, uu, int(t)).as_dict(w.m)
        if (ref["margin_all"] > MARGIN).all():
            assert (r["index"], r["safe"], r["steps"], r["n_safe"], r["n_exec"]) == (f["index"], f["safe"], f["steps"], f["n_safe"], f["n_exec"])
    assert exact >= 15


def test_affine_flag_ignored_with_noise_or_relift(mp):
    w = W.make("C2", N=2000); w.noise_sigma = 0.01
    assert mp.Context(w, variant=mp.mpmi.VARIANT_AFFINE).info()["variant"] == 1
    w = W.make("C2", N=2000); w.model_kind = 1
    assert mp.Context(w, variant=mp.mpmi.VARIANT_AFFINE).info()["variant"] == 5


# ------------------------------------------------------------------ the paper's own race-car sample set ------------------
def _paper_grid(relift=False):
    """N = 10,120 = 20 x 22 x 23 equally spaced samples over heading [-1,1] x gas [0,1] x brake [-1,0], horizon 25
    (PAPER.md:222, 242, 270), on the m = 3 model of C5 (the paper's trained race-car model is not available)."""
    w = W.make("C5", N=10120, H=25)
    w.sampler = 1; w.grid_counts = np.array([20, 22, 23], np.int32)
    w.u_lo = np.array([-1, 0, -1], np.float32); w.u_hi = np.array([1, 1, 0], np.float32)
    if relift:
        w = G.scaled_bounds(w, 0.25); w.model_kind = 1
    return w


@pytest.mark.parametrize("variant,kernel", [(0, 4), (128, 2), (256, 6), ("relift", 5)])
def test_paper_race_car_grid_tick(mp, variant, kernel):
    """T3 on the paper's 3-D asymmetric grid through every kernel that serves d = 128: tcgen05, FP32 tile, affine, re-lift."""
    w = _paper_grid(relift=(variant == "relift"))
    ctx = mp.Context(w, variant=0 if variant == "relift" else variant)
    assert ctx.info()["variant"] == kernel and ctx.info()["ncand_local"] == 10121
    o = _oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 10)
    exact = 0; branches = set()
    for x0, uu, t in zip(x0s, uus, ticks):
        ref = o.step(x0, uu, int(t), detail=True)
        r = ctx.step_sync(x0, uu, int(t)).as_dict(w.m)
        ok, ex, why = accept_selection(r, ref, w.H)
        assert ok, (why, r, {k: ref[k] for k in ("index", "safe", "steps", "dist")})
        exact += ex
        assert np.all(np.asarray(r["u"][:3]) >= w.u_lo) and np.all(np.asarray(r["u"][:3]) <= w.u_hi)
        if (ref["margin_all"] > MARGIN).all():
            assert r["n_safe"] == ref["n_safe"] and r["n_exec"] == ref["n_exec"]
        branches.add("user" if (r["safe"] and r["dist"] == 0) else "intervene" if r["safe"] else "fallback")
    assert exact >= 9 and "intervene" in branches, (exact, branches)


# ------------------------------------------------------------------ d = 128: both kernels stay covered ------------------
def test_fp32_tile_kernel_d128_parity(mp):
    """MPMI_VARIANT_NO_TENSOR keeps the FP32 SIMT warp-tile kernel reachable at d = 128: T1 / T2 and the same winner
    as the 3xTF32 tcgen05 kernel (the default there)."""
    w = W.make("C5", N=900)
    o = _oracle(w)
    simt = mp.Context(w, variant=mp.mpmi.VARIANT_NO_TENSOR)
    tens = mp.Context(w, variant=mp.mpmi.VARIANT_TC_UNVERIFIED)          # the bare tcgen05 kernel (caller-supplied inputs below)
    assert simt.info()["variant"] == 2 and tens.info()["variant"] == 4
    rng = np.random.default_rng(3)
    U = rng.uniform(w.u_lo, w.u_hi, (w.N, w.m)).astype(np.float32)
    x0s, _, _ = W.tick_inputs(w, 1)
    r_steps, r_marg, r_traj = o.rollout_batch(U, x0s, want_traj=True)
    worst = {}
    for tag, ctx in (("simt", simt), ("tensor", tens)):
        traj = torch.full((w.H, w.d, w.N), 7.0, dtype=torch.float32, device="cuda")
        steps = torch.empty(w.N, dtype=torch.int32, device="cuda")
        dU, dX = _dev(U), _dev(x0s)
        ctx.rollout_batch(dU.data_ptr(), dX.data_ptr(), 1, w.N, w.H, mp.DUMP_LIFTED, traj.data_ptr(), steps.data_ptr(), 0)
        torch.cuda.synchronize()
        g_steps = steps.cpu().numpy(); g_traj = traj.cpu().numpy()
        bad, _ = check_flags(g_steps, r_steps, r_marg, w.H)
        assert len(bad) == 0
        worst[tag] = max(traj_rel_err(g_traj[:, :, i], r_traj[i], min(r_steps[i] + 1, g_steps[i] + 1, w.H)) for i in range(w.N))
    assert worst["simt"] <= 1e-5 and worst["tensor"] <= TRAJ_RTOL, worst
    x0s, uus, ticks = W.tick_inputs(w, 6)
    for x0, uu, t in zip(x0s, uus, ticks):
        a = simt.step_sync(x0, uu, int(t)).as_dict(w.m); b = tens.step_sync(x0, uu, int(t)).as_dict(w.m)
        ref = o.step(x0, uu, int(t), detail=True)
        if (ref["margin_all"] > MARGIN).all():
            assert (a["index"], a["safe"], a["steps"], a["n_safe"]) == (b["index"], b["safe"], b["steps"], b["n_safe"])


def test_constant_slot_exhaustion_falls_back_to_shared_memory(mp):
    """The register kernels keep the model in one of 8 __constant__ slots per live context; a 9th, 10th ... context must
    fall back to the shared-memory variant and return identical results (and slots are recycled on close)."""
    w = W.make("C4", N=1 << 19)
    x0s, uus, ticks = W.tick_inputs(w, 2)
    NT = mp.mpmi.VARIANT_NO_TENSOR
    ctxs = [mp.Context(w, variant=NT) for _ in range(11)]
    ref = [ctxs[0].step_sync(x0, uu, int(t)).as_dict(w.m) for x0, uu, t in zip(x0s, uus, ticks)]
    for c in ctxs[1:]:
        for r0, (x0, uu, t) in zip(ref, zip(x0s, uus, ticks)):
            r = c.step_sync(x0, uu, int(t)).as_dict(w.m)
            assert (r["index"], r["safe"], r["steps"], r["n_safe"], r["n_exec"], r["key"]) == \
                   (r0["index"], r0["safe"], r0["steps"], r0["n_safe"], r0["n_exec"], r0["key"])
    for c in ctxs:
        c.close()
    again = mp.Context(w, variant=NT)                      # a slot is free again
    r = again.step_sync(x0s[0], uus[0], int(ticks[0])).as_dict(w.m)
    assert r["key"] == ref[0]["key"]


# ------------------------------------------------------------------ N > 1: two ranks over NCCL (needs 2 GPUs) -------------
def _nccl_worker(rank, world, port, name, N, nticks, out):
    import os
    import torch.distributed as dist
    import paper_1906_02318_b200 as mpk
    from paper_1906_02318_b200.shard import shard_plan, gather_partials
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    w = W.make(name, N=N)
    b, c = shard_plan(w.N, 1, world, rank)
    ctx = mpk.Context(w, device=rank, shard=(b, c))
    x0s, uus, ticks = W.tick_inputs(w, nticks)
    s = torch.cuda.current_stream().cuda_stream
    part = torch.zeros(3, dtype=torch.int64, device="cuda")
    res = torch.zeros(56, dtype=torch.uint8, device="cuda")
    got = []
    for x0, uu, t in zip(x0s, uus, ticks):
        dx, du = torch.as_tensor(x0).cuda(), torch.as_tensor(uu).cuda()
        ctx.shard_step(dx.data_ptr(), du.data_ptr(), int(t), s, part.data_ptr())
        parts = gather_partials(part, world)
        ctx.shard_finalize(parts.data_ptr(), world, du.data_ptr(), int(t), s, res.data_ptr())
        torch.cuda.synchronize()
        r = np.frombuffer(res.cpu().numpy().tobytes(), dtype=mpk.mpmi.RESULT_DTYPE)[0]
        got.append((int(r["index"]), int(r["safe"]), int(r["steps"]), int(r["n_safe"]), int(r["n_exec"]), int(r["key"])))
    out[rank] = got
    dist.destroy_process_group()


def test_two_rank_nccl_sharded_tick(mp):
    """Candidates sharded over two GPUs, one 24-byte all-gather over NCCL per tick: every rank decodes
    the result of the single-context tick.  Skipped on a 1-GPU box (the same code path runs there as two shards on one GPU:
    test_device_and_shard_paths_match_host_path, and through a 1-rank NCCL group: MPMI_BENCH_FORCE_SHARD=1 python bench.py)."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs")
    import torch.multiprocessing as tmp
    name, N, nticks = "C4", 1 << 18, 3
    w = W.make(name, N=N)
    one = mp.Context(w)
    x0s, uus, ticks = W.tick_inputs(w, nticks)
    ref = []
    for x0, uu, t in zip(x0s, uus, ticks):
        r = one.step_sync(x0, uu, int(t)).as_dict(w.m)
        ref.append((r["index"], r["safe"], r["steps"], r["n_safe"], r["n_exec"], r["key"]))
    out = tmp.Manager().dict()
    tmp.spawn(_nccl_worker, args=(2, 29500 + os.getpid() % 2000, name, N, nticks, out), nprocs=2, join=True)
    assert out[0] == ref and out[1] == ref


# ------------------------------------------------------------------ measurement entry points ---------------------------
def test_profile_entry_points(mp):
    """mpmi_profile_enable / mpmi_profile_read: event times of the tick kernel and the second pass of plain-launch ticks;
    mpmi_profile_timeline: stage stamps of the latency kernel (monotone per CTA), UNSUPPORTED on the other kernels.  The
    tick's result is not affected by either."""
    s = torch.cuda.current_stream().cuda_stream
    w = W.make("C4", N=1 << 17)                               # verified tensor-core tick: both passes timed
    ctx = mp.Context(w)
    x0s, uus, ticks = W.tick_inputs(w, 5)
    d_res = torch.zeros(56, dtype=torch.uint8, device="cuda")
    ref = [ctx.step_sync(x0, uu, int(t)).as_dict(w.m) for x0, uu, t in zip(x0s, uus, ticks)]
    ctx.profile_enable(True)
    for k, (x0, uu, t) in enumerate(zip(x0s, uus, ticks)):
        dx, du = _dev(x0), _dev(uu)
        ctx.step_device(dx.data_ptr(), du.data_ptr(), int(t), s, d_res.data_ptr())
        torch.cuda.synchronize()
        got = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)[0]
        assert int(got["key"]) == ref[k]["key"] and int(got["n_exec"]) == ref[k]["n_exec"]
    first, second = ctx.profile_read()
    ctx.profile_enable(False)
    assert len(first) == 5 and len(second) == 5 and (first > 0.05).all() and (second > 0.005).all() and (first < 50).all()
    with pytest.raises(mp.MpmiError) as e:
        ctx.profile_timeline(d_res.data_ptr())
    assert e.value.status == mp.mpmi.ERR_UNSUPPORTED
    w2 = W.make("C2")                                         # latency kernel: the stage timeline
    c2 = mp.Context(w2)
    info = c2.info()
    assert info["variant"] == 3
    stamps = torch.zeros((info["blocks"], 8), dtype=torch.int64, device="cuda")
    x0s, uus, ticks = W.tick_inputs(w2, 2)
    want = c2.step_sync(x0s[1], uus[1], int(ticks[1])).as_dict(1)
    c2.profile_timeline(stamps.data_ptr())
    dx, du = _dev(x0s[1]), _dev(uus[1])
    c2.step_device(dx.data_ptr(), du.data_ptr(), int(ticks[1]), s, d_res.data_ptr())
    torch.cuda.synchronize()
    c2.profile_timeline(0)
    got = np.frombuffer(d_res.cpu().numpy().tobytes(), dtype=mp.mpmi.RESULT_DTYPE)[0]
    assert int(got["key"]) == want["key"]
    st = stamps.cpu().numpy()
    assert (st[:, 0] > 0).all() and (np.diff(st[:, :6], axis=1) >= 0).all()
    assert 1e3 < (st[:, 5].max() - st[:, 0].min()) < 1e6      # kernel span between 1 us and 1 ms
