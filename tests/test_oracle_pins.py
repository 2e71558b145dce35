"""Pins for the FP64 oracle: each checks oracle/ against something other than
itself -- published known answers, closed forms, brute force, textbook special cases, invariants."""
import os
import numpy as np
import pytest

import workloads as W
from workloads import generate as G
from oracle import oracle as O
from oracle.oracle import Oracle


def _free(w):
    """copy of w with the safe set = everything"""
    import copy
    v = copy.copy(w)
    v.bidx = np.zeros(0, np.int32); v.blo = np.zeros(0, np.float32); v.bhi = np.zeros(0, np.float32)
    v.annulus = 0
    return v


# ---------------------------------------------------------------- P8: sampler --------------------
def test_philox_known_answers(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")) if not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert O.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def _py_philox(ctr, key):
    """independent pure-Python restatement (Python ints) used to pin counter/key layout"""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    c = list(ctr); k = list(key)
    for r in range(10):
        if r:
            k = [(k[0] + W0) & 0xFFFFFFFF, (k[1] + W1) & 0xFFFFFFFF]
        p0, p1 = M0 * c[0], M1 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
    return c


def test_philox_sampler_layout_and_mapping():
    """counter = (i_lo, i_hi, tick_lo, tick_hi), key = (seed_lo, seed_hi), word j -> dim j,
    r = (w>>8) 2^-24, u = fmaf(r, hi-lo, lo) in fp32 (DESIGN G4)."""
    w = W.make("C5", calibrated=False)
    w.seed = 0x1234_5678_9ABC_DEF0
    w.u_lo = np.array([-1.0, 0.0, -1.0], np.float32); w.u_hi = np.array([1.0, 1.0, 0.0], np.float32)
    o = Oracle(w)
    tick = (7 << 32) | 99
    idx = [0, 1, 2, 12345, w.N - 1]
    got = o.sample(tick, idx)
    for row, i in zip(got, idx):
        words = _py_philox([i, 0, tick & 0xFFFFFFFF, tick >> 32], [w.seed & 0xFFFFFFFF, w.seed >> 32])
        for j in range(3):
            r = np.float32(words[j] >> 8) * np.float32(2.0 ** -24)
            span = np.float32(w.u_hi[j] - w.u_lo[j])
            exact = float(r) * float(span) + float(w.u_lo[j])          # fp64 is exact enough to round once
            assert row[j] == np.float32(exact)
            assert w.u_lo[j] <= row[j] <= w.u_hi[j]


def test_philox_uniform_moments():
    w = W.make("C1", calibrated=False)
    o = Oracle(w, N=20000)
    u = o.sample(3, np.arange(20000))[:, 0].astype(np.float64)
    assert abs(u.mean()) < 0.02 and abs(u.var() - 1.0 / 3.0) < 0.01
    assert u.min() >= -1 and u.max() <= 1
    u2 = o.sample(4, np.arange(100))[:, 0]
    assert not np.array_equal(u2, u[:100].astype(np.float32))        # fresh set each tick


def test_grid_points_exact():
    """endpoint-inclusive grid, row-major, dimension 0 slowest (DESIGN G3)."""
    w = W.make("C3", calibrated=False)
    o = Oracle(w)
    u = o.sample(0, [0, 99, 100, 9999, 50 * 100 + 50])
    assert tuple(u[0]) == (-1.0, -1.0) and tuple(u[1]) == (-1.0, 1.0)
    assert u[2][1] == -1.0 and u[2][0] == np.float32(float(np.float32(1.0) / np.float32(99)) * 2.0 - 1.0)
    assert tuple(u[3]) == (1.0, 1.0)
    assert abs(u[4][0] - (-1 + 50 * 2 / 99)) < 1e-6
    w.grid_counts = np.array([23, 1], np.int32); w.N = 23
    u = Oracle(w).sample(0, np.arange(23))
    assert u[11][0] == 0.0 and np.all(u[:, 1] == 0.0)                 # odd count contains "straight"
    assert not np.array_equal(Oracle(w).sample(0, [5]), Oracle(w).sample(0, [6]))
    assert np.array_equal(Oracle(w).sample(0, [5]), Oracle(w).sample(9, [5]))   # grid ignores tick


def test_paper_race_car_grid_20x22x23(golden_dir):
    """The paper's race-car sample set: N = 10,120 'equally spaced samples in all 3 input dimensions'
     = 20 x 22 x 23 over heading [-1,1] x gas [0,1] x brake [-1,0]:
    an asymmetric box with a different count per dimension.  Pinned against numpy's linspace / meshgrid
    (endpoint-inclusive, dimension 0 slowest: DESIGN G3) and the row the paper prints for Eq. (2)."""
    row = [l.split() for l in open(os.path.join(golden_dir, "eq2_printed.txt")) if l.startswith("race_car")][0]
    counts = np.array([20, 22, 23], np.int32)
    lo = np.array([-1, 0, -1], np.float32); hi = np.array([1, 1, 0], np.float32)
    assert int(row[2]) == int(counts.prod()) == 10120
    assert float(row[1]) == float((hi - lo).sum())                       # lambda* = 4 as printed (G7: a sum of lengths)
    w = W.make("C5", N=10120, H=25)
    w.sampler = 1; w.grid_counts = counts; w.u_lo = lo; w.u_hi = hi
    o = Oracle(w, include_user=0)
    u = o.sample(3, np.arange(10120))
    axes = [np.linspace(float(lo[j]), float(hi[j]), int(counts[j])) for j in range(3)]
    ref = np.stack(np.meshgrid(*axes, indexing="ij"), axis=-1).reshape(-1, 3)
    assert np.abs(u.astype(np.float64) - ref).max() <= 2.0 ** -23        # fp32 rounding of the grid value
    for j in range(3):
        assert len(np.unique(u[:, j])) == counts[j]
        assert u[:, j].min() == lo[j] and u[:, j].max() == hi[j]          # endpoints included, exactly
    assert np.array_equal(u[0], lo) and np.array_equal(u[-1], hi)
    assert u[1][2] > u[0][2] and u[1][0] == u[0][0] and u[23][1] > u[0][1] and u[22 * 23][0] > u[0][0]   # dim 0 slowest
    # a tick on it: the selected input is a grid point (or the injected u_h) and lies in the box
    o = Oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 3)
    for x0, uu, t in zip(x0s, uus, ticks):
        r = o.step(x0, uu, int(t), detail=True)
        assert np.all(r["u"] >= lo) and np.all(r["u"] <= hi)
        assert 0 < r["n_safe"] < 10121                                    # a mixed set on this workload
        if r["index"] < 10120:
            assert np.array_equal(np.asarray(r["u"], np.float32), u[r["index"]])


# ---------------------------------------------------------------- P9: lift -----------------------
def test_lift_hand_values():
    w = W.make("C3", calibrated=False)
    o = Oracle(w)
    assert o.lift(np.zeros(6))[7] == 1.0 and np.count_nonzero(o.lift(np.zeros(6))) == 1   # only cos(0)
    x = np.array([2.0, 3.0, 0.5, 5.0, 7.0, 11.0])
    z = o.lift(x)
    assert np.allclose(z[:6], x)
    assert np.isclose(z[6], np.sin(0.5)) and np.isclose(z[7], np.cos(0.5))
    prods = [x[i] * x[j] for i in range(6) for j in range(i, 6)]
    assert np.allclose(z[8:29], prods)
    assert np.allclose(z[29:], [5 * np.cos(0.5), 5 * np.sin(0.5), 7 * np.cos(0.5)])
    w2 = W.make("C2", calibrated=False)
    e1 = np.zeros(4); e1[1] = 2.0
    z2 = Oracle(w2).lift(e1)
    assert z2[1] == 2.0 and z2[14] == 8.0 and z2[15] == 0.0 and z2[8] == 4.0   # x1, x1^3, x3^3, x1*x1
    assert np.count_nonzero(Oracle(w2).lift(np.zeros(4))) == 0


def test_lift_rff_matches_numpy():
    w = W.make("C5", calibrated=False)
    x = np.linspace(-0.3, 0.4, 8)
    z = Oracle(w).lift(x)
    ref = w.scale * np.cos(w.W.astype(np.float64) @ x + w.b.astype(np.float64))
    assert np.allclose(z[:8], x) and np.allclose(z[8:], ref, rtol=0, atol=1e-14)


# ---------------------------------------------------------------- P1: closed forms ---------------
@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C5"])
def test_rollout_closed_form(name):
    """z_H = K^H z0 + sum_{k<H} K^k B u  (north_star) and (I-K)^-1 (I-K^H) B u  (rho(K) < 1)."""
    w = _free(W.make(name, calibrated=False))
    o = Oracle(w)
    rng = np.random.default_rng(5)
    K = w.K.astype(np.float64); B = w.B.astype(np.float64)
    for _ in range(3):
        z0 = o.lift(w.x_nom.astype(np.float64) + 0.01 * rng.standard_normal(w.n))
        u = rng.uniform(-1, 1, w.m)
        steps, _, traj = o.rollout(z0, u, want_traj=True)
        assert steps == w.H
        H = w.H
        KH = np.linalg.matrix_power(K, H)
        s = sum(np.linalg.matrix_power(K, k) @ B @ u for k in range(H))
        zH = KH @ z0 + s
        scale = max(np.linalg.norm(zH), 1e-12)
        assert np.linalg.norm(traj[H - 1] - zH) / scale < 1e-10
        geo = np.linalg.solve(np.eye(w.d) - K, (np.eye(w.d) - KH) @ B @ u)
        assert np.linalg.norm(traj[H - 1] - (KH @ z0 + geo)) / scale < 1e-8
        k = H // 3                                                   # an interior step too
        zk = np.linalg.matrix_power(K, k + 1) @ z0 + sum(np.linalg.matrix_power(K, q) @ B @ u for q in range(k + 1))
        assert np.linalg.norm(traj[k] - zk) / max(np.linalg.norm(zk), 1e-12) < 1e-10


# ---------------------------------------------------------------- P2: brute force ----------------
def _brute_tick(w, U, z0, u_h, H):
    """un-vectorised Python restatement of Algorithm 2 l.2-13 with explicit sorting of key tuples"""
    K = [[float(v) for v in row] for row in w.K]; B = [[float(v) for v in row] for row in w.B]
    keys, steps_all = [], []
    for i, u in enumerate(U):
        z = [float(v) for v in z0]; steps = H
        for k in range(H):
            zn = []
            for r in range(w.d):
                s = 0.0
                for c in range(w.d):
                    s += K[r][c] * z[c]
                for j in range(w.m):
                    s += B[r][j] * float(u[j])
                zn.append(s)
            z = zn
            ok = True
            for q in range(len(w.bidx)):
                v = z[int(w.bidx[q])]
                ok = ok and (float(w.blo[q]) + float(w.inflate) < v < float(w.bhi[q]) - float(w.inflate))
            if w.annulus:
                r2 = (z[w.ix] - w.cx) ** 2 + (z[w.iy] - w.cy) ** 2
                ok = ok and ((w.rmin + w.inflate) ** 2 <= r2 <= (w.rmax - w.inflate) ** 2)
            if not ok:
                steps = k
                break
        steps_all.append(steps)
        dist = sum((float(u[j]) - float(u_h[j])) ** 2 for j in range(w.m)) ** 0.5
        keys.append((0, dist, i) if steps == H else (1, H - steps, i))
    return sorted(keys)[0], steps_all


@pytest.mark.parametrize("name,shrink", [("C1", 1.0), ("C1", 0.05), ("C3", 1.0), ("C3", 0.02), ("C2", 1.0)])
def test_tick_vs_brute_force(name, shrink):
    w = W.make(name, calibrated=True, N=16, H=5)
    if name == "C3":
        w.grid_counts = np.array([4, 4], np.int32)
    w = G.scaled_bounds(w, shrink)
    w.inflate = 0.01
    o = Oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 6)
    for x0, uu, t in zip(x0s, uus, ticks):
        r = o.step(x0, uu, int(t), detail=True)
        u_h = np.clip(uu, w.u_lo, w.u_hi)
        key, steps_all = _brute_tick(w, r["U"], o.lift(x0.astype(np.float64)), u_h, w.H)
        assert list(r["steps_all"]) == steps_all
        assert r["index"] == key[2] and r["safe"] == (key[0] == 0)
        assert r["n_safe"] == sum(s == w.H for s in steps_all)
        assert r["n_exec"] == sum(min(s + 1, w.H) for s in steps_all)
        if key[0] == 0:
            assert abs(r["dist"] - key[1]) < 1e-15
        else:
            assert r["steps"] == w.H - key[1]
    # the forced-fallback set really falls back, the literal set really has safe candidates
    if shrink < 0.1:
        assert r["safe"] == 0


# ---------------------------------------------------------------- P3 / P4: invariants ------------
@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C5"])
def test_minimal_intervention_and_membership(name):
    """a safe u_user is returned unchanged; the selected input is a sampled one."""
    w = W.make(name, N=512 if name != "C3" else 400)
    if name == "C3":
        w.grid_counts = np.array([20, 20], np.int32)
    o = Oracle(w)
    x0s, uus, ticks = W.tick_inputs(w, 12)
    seen_safe_user = seen_intervention = 0
    for x0, uu, t in zip(x0s, uus, ticks):
        r = o.step(x0, uu, int(t), detail=True)
        assert 0 <= r["index"] <= w.N
        assert np.array_equal(r["u"], r["U"][r["index"]])                       # P4
        u_h = np.clip(uu, w.u_lo, w.u_hi)
        assert np.array_equal(r["U"][w.N], u_h)
        if r["steps_all"][w.N] == w.H:                                          # P3
            seen_safe_user += 1
            assert np.array_equal(r["u"], u_h) and r["dist"] == 0.0 and r["safe"] == 1
            assert r["index"] == w.N or np.array_equal(r["U"][r["index"]], u_h)
        elif r["safe"]:
            seen_intervention += 1
            assert r["dist"] > 0 and r["steps_all"][r["index"]] == w.H          # never an unsafe input
    assert seen_safe_user > 0 and seen_intervention > 0


# ---------------------------------------------------------------- P5: Eq. (2) --------------------
def test_eq2_printed_value(golden_dir):
    """1-D grid of 10,000 samples on [-1,1], everything safe, literal Alg. 2 (u_h not injected):
    max deviation = half the spacing ~ lambda*/(2N) = 0.0001 as printed."""
    row = [l.split() for l in open(os.path.join(golden_dir, "eq2_printed.txt")) if l.startswith("balance")][0]
    lam, N, printed = float(row[1]), int(row[2]), float(row[3])
    assert abs(lam / (2 * N) - printed) < 1e-12
    w = _free(W.make("C1", calibrated=False, N=N, H=1))
    w.sampler = 1; w.grid_counts = np.array([N], np.int32)
    o = Oracle(w, include_user=0)
    spacing = 2.0 / (N - 1)
    worst = 0.0
    rng = np.random.default_rng(0)
    cells = rng.integers(0, N - 1, 40)
    for c in cells:
        for frac in (0.5, 0.25, 0.999):
            u_h = np.float32(-1.0 + (c + frac) * spacing)
            r = o.step(np.zeros(4, np.float32), np.array([u_h]), 0)
            dev = abs(float(r["u"][0]) - float(u_h))
            assert dev <= spacing / 2 + 2.0 ** -23                  # half the spacing (+ fp32 rounding of the grid)
            worst = max(worst, dev)
    assert worst > 0.99 * spacing / 2                                    # attained at cell mid-points
    assert round(worst, 4) == printed


# ---------------------------------------------------------------- P6: textbook special cases -----
def test_special_case_K_zero():
    """K = 0  =>  x_k = C B u for every k: safe iff that one point is in the safe set."""
    w = W.make("C1", N=256, H=7)
    w.K = np.zeros_like(w.K)
    w.B = (w.B * 0 + np.linspace(0.2, 1.0, 8)[:, None]).astype(np.float32)
    o = Oracle(w)
    r = o.step(w.x_nom + 1.0, np.array([0.3], np.float32), 0, detail=True)
    for i in range(w.N + 1):
        x = w.B[:4, 0].astype(np.float64) * float(r["U"][i, 0])
        ok = (-2 < x[0] < 2) and (-0.5 < x[1] < 0.5)
        assert r["steps_all"][i] == (w.H if ok else 0)


def test_special_case_K_rho_identity():
    """K = rho I  =>  z_k = rho^k z0 + (1-rho^k)/(1-rho) B u ; first violation step in closed form."""
    w = W.make("C1", N=300, H=40)
    rho = 0.9
    w.K = (rho * np.eye(8)).astype(np.float32)
    w.B = np.zeros((8, 1), np.float32); w.B[1, 0] = 0.1
    w.bidx = np.array([1], np.int32); w.blo = np.array([-0.5], np.float32); w.bhi = np.array([0.5], np.float32)
    o = Oracle(w)
    x0 = np.array([0.0, 0.2, 0.0, 0.0], np.float32)
    r = o.step(x0, np.array([0.0], np.float32), 0, detail=True)
    rho64 = float(np.float32(rho)); b = float(np.float32(0.1)); x1 = float(x0[1])
    mixed = set()
    for i in range(w.N + 1):
        u = float(r["U"][i, 0])
        expect = w.H
        for k in range(1, w.H + 1):
            xk = rho64 ** k * x1 + (1 - rho64 ** k) / (1 - rho64) * b * u
            if not (-0.5 < xk < 0.5):
                expect = k - 1
                break
        assert r["steps_all"][i] == expect
        mixed.add(expect == w.H)
    assert mixed == {True, False}


def test_special_case_B_zero():
    """B = 0: all candidates share one trajectory => all safe (nearest sample wins) or all unsafe
    with equal steps (index 0 wins)."""
    w = W.make("C1", N=64, H=20)
    w.B = np.zeros_like(w.B)
    o = Oracle(w)
    r = o.step(w.x_nom, np.array([0.123], np.float32), 5, detail=True)
    assert r["n_safe"] == w.N + 1 and r["index"] == w.N and r["dist"] == 0
    o0 = Oracle(w, include_user=0)
    r0 = o0.step(w.x_nom, np.array([0.123], np.float32), 5, detail=True)
    assert r0["index"] == int(np.argmin(np.abs(r0["U"][:, 0].astype(np.float64) - np.float64(np.float32(0.123)))))
    bad = np.array([1.9, 0.49, 3.0, 3.0], np.float32)                   # leaves the box under K alone
    rb = o.step(bad, np.array([0.123], np.float32), 5, detail=True)
    if rb["safe"] == 0:
        assert rb["index"] == 0 and len(set(rb["steps_all"])) == 1


# ---------------------------------------------------------------- P7: structural invariants ------
def test_prefix_and_monotone_invariants():
    w = W.make("C2", N=400)
    x0s, uus, ticks = W.tick_inputs(w, 3)
    for x0, uu, t in zip(x0s, uus, ticks):
        full = Oracle(w).step(x0, uu, int(t), detail=True)
        for Hp in (1, 17, 60):
            part = Oracle(w, H=Hp).step(x0, uu, int(t), detail=True)
            assert np.array_equal(part["steps_all"], np.minimum(full["steps_all"], Hp))   # prefix
        big = Oracle(G.scaled_bounds(w, 1.5)).step(x0, uu, int(t), detail=True)
        assert np.all(big["steps_all"] >= full["steps_all"])                               # monotone
        if full["safe"]:
            assert big["safe"] and big["dist"] <= full["dist"]
        # inflated barrier shrinks the safe set
        import copy
        wi = copy.copy(w); wi.inflate = 0.05
        infl = Oracle(wi).step(x0, uu, int(t), detail=True)
        assert np.all(infl["steps_all"] <= full["steps_all"])


def test_is_safe_conventions():
    """box strict, annulus closed, NaN/Inf => unsafe (DESIGN G9)."""
    w = W.make("C1")
    o = Oracle(w)
    assert o.is_safe([0, 0, 0, 0])[0] and not o.is_safe([2.0, 0, 0, 0])[0] and not o.is_safe([0, -0.5, 0, 0])[0]
    assert not o.is_safe([np.nan, 0, 0, 0])[0] and not o.is_safe([0, np.inf, 0, 0])[0]
    assert abs(o.is_safe([1.5, 0.1, 9, 9])[1] - 0.4) < 1e-12
    w3 = W.make("C3")
    o3 = Oracle(w3)
    assert o3.is_safe([8, 0, 0, 0, 0, 0])[0] and o3.is_safe([0, -12, 0, 0, 0, 0])[0]
    assert not o3.is_safe([7.999, 0, 0, 0, 0, 0])[0] and not o3.is_safe([np.nan, 0, 0, 0, 0, 0])[0]
    assert abs(o3.is_safe([3.0, 4.0 + 5, 0, 0, 0, 0])[1] - min(abs(np.hypot(3, 9) - 8), abs(12 - np.hypot(3, 9)))) < 1e-12


def test_rollout_batch_matches_single():
    w = W.make("C3", N=32)
    o = Oracle(w)
    rng = np.random.default_rng(1)
    U = rng.uniform(-1, 1, (32, 2)).astype(np.float32)
    x0s, _, _ = W.tick_inputs(w, 32)
    steps, marg, traj = o.rollout_batch(U, x0s, want_traj=True)
    for i in (0, 7, 31):
        s, mg, tr = o.rollout(o.lift(x0s[i].astype(np.float64)), U[i].astype(np.float64), want_traj=True)
        assert s == steps[i] and mg == marg[i] and np.array_equal(np.nan_to_num(tr), np.nan_to_num(traj[i]))
        e = min(s + 1, w.H)
        assert np.all(np.isfinite(traj[i, :e])) and np.all(np.isnan(traj[i, e:]))


def test_calibrated_workloads_are_mixed():
    """safe fraction at x_nom inside Table I's band."""
    for name in ("C1", "C2", "C3", "C5"):
        w = W.make(name, N=2048 if name != "C3" else 10000)
        r = Oracle(w, include_user=0).step(w.x_nom, np.zeros(w.m, np.float32), 0)
        assert 0.28 <= r["n_safe"] / w.N <= 0.50, (name, r["n_safe"] / w.N)


# ---------------------------------------------------------------- NEXT-2: prediction noise ---------
def test_noise_is_standard_normal_and_independent():
    """eps of orc_noise: N(0, 1) marginals (moments + Kolmogorov-Smirnov against the normal CDF),
    uncorrelated across dims, steps, candidates and ticks (i.i.d. Gaussian white noise)."""
    from scipy import stats
    w = _free(W.make("C4", calibrated=False)); w.noise_sigma = 1.0
    o = Oracle(w)
    E = np.array([[o.noise(3, i, k) for k in range(40)] for i in range(700)])          # (cand, step, dim)
    v = E.reshape(-1)
    assert abs(v.mean()) < 0.01 and abs(v.var() - 1.0) < 0.02
    assert abs(stats.kurtosis(v, fisher=False) - 3.0) < 0.06 and abs(stats.skew(v)) < 0.03
    assert stats.kstest(v, "norm").pvalue > 1e-3
    for j in range(w.n):                                                              # every dim on its own
        assert stats.kstest(E[:, :, j].reshape(-1), "norm").pvalue > 1e-4
    flat = E.reshape(-1, w.n)
    c = np.corrcoef(flat.T)
    assert np.abs(c - np.eye(w.n)).max() < 0.02                                       # across dims (incl. Box-Muller pairs)
    assert abs(np.corrcoef(E[:, :-1, :].reshape(-1), E[:, 1:, :].reshape(-1))[0, 1]) < 0.02   # across steps
    assert abs(np.corrcoef(E[:-1].reshape(-1), E[1:].reshape(-1))[0, 1]) < 0.02               # across candidates
    other = np.array([[o.noise(4, i, k) for k in range(40)] for i in range(100)])
    assert abs(np.corrcoef(other.reshape(-1), E[:100].reshape(-1))[0, 1]) < 0.05               # across ticks
    uni = np.array([o.sample(3, [i])[0] for i in range(700)])                          # not the sampling stream
    assert abs(np.corrcoef(uni[:, 0], E[:, 0, 0])[0, 1]) < 0.1


@pytest.mark.parametrize("name", ["C1", "C4"])
def test_noise_rollout_closed_form(name):
    """z_H = K^H z0 + sum_k K^(H-1-k) (B u + sigma E eps_k), E = [I_n; 0]: pins WHERE the noise enters
    (physical rows, after the step, kept in the carried state) and which draw belongs to which step."""
    w = _free(W.make(name, N=8)); w.noise_sigma = 0.05
    o = Oracle(w)
    K, B = o.K, o.B
    z0 = o.lift(w.x_nom.astype(np.float64))
    H, tick = 12, 9
    for i in (0, 5):
        u = o.sample(tick, [i])[0].astype(np.float64)
        steps, _, traj = o.rollout(z0, u, H=H, want_traj=True, tick=tick, i=i)
        assert steps == H
        z = z0.copy()
        for k in range(H):
            e = np.zeros(w.d); e[: w.n] = np.float64(np.float32(w.noise_sigma)) * o.noise(tick, i, k)
            z = K @ z + B @ u + e
            assert np.allclose(traj[k], z, rtol=1e-12, atol=1e-12)
        acc = np.linalg.matrix_power(K, H) @ z0
        for k in range(H):
            e = np.zeros(w.d); e[: w.n] = np.float64(np.float32(w.noise_sigma)) * o.noise(tick, i, k)
            acc += np.linalg.matrix_power(K, H - 1 - k) @ (B @ u + e)
        assert np.allclose(traj[H - 1], acc, rtol=1e-9, atol=1e-9)


def test_noise_zero_sigma_and_tick_semantics():
    """sigma = 0 is the noise-free path bit for bit; the noise is tested BEFORE it can be ignored:
    K = 0, B = 0 makes x_1 = sigma eps_0, so candidate i is unsafe iff |sigma eps_0| leaves the box."""
    w = W.make("C1", N=64)
    a = Oracle(w).step(w.x_nom, np.zeros(1, np.float32), 5, detail=True)
    w2 = W.make("C1", N=64); w2.noise_sigma = 0.0
    b = Oracle(w2).step(w2.x_nom, np.zeros(1, np.float32), 5, detail=True)
    assert np.array_equal(a["steps_all"], b["steps_all"]) and a["index"] == b["index"]
    w3 = W.make("C1", N=400); w3.K = np.zeros_like(w3.K); w3.B = np.zeros_like(w3.B); w3.noise_sigma = 0.4; w3.H = 1
    o = Oracle(w3)
    r = o.step(np.zeros(4, np.float32), np.zeros(1, np.float32), 2, detail=True)
    sig = float(np.float32(0.4))
    for i in range(401):
        x1 = sig * o.noise(2, i, 0)
        inside = all(lo < x1[j] < hi for j, lo, hi in zip(w3.bidx, w3.blo, w3.bhi))
        assert (r["steps_all"][i] == 1) == inside
    assert 0.2 < (r["steps_all"] == 1).mean() < 0.95


# ---------------------------------------------------------------- NEXT-3: re-lift model -------------
def _py_lift_mono(terms, x):
    out = []
    for f in range(terms.shape[0]):
        p = 1.0
        for code in terms[f]:
            if code == 0xFF:
                continue
            v = x[code & 0x3F]
            p *= v if code >> 6 == 0 else (np.sin(v) if code >> 6 == 1 else np.cos(v))
        out.append(p)
    return np.array(out)


def test_relift_matches_independent_python_loop():
    """x_{k+1} = C (K Psi(x_k) + B u) (the literal f(x, u) on states): an un-vectorised
    Python restatement on the race-car lift (sin, cos and product features)."""
    w = _free(W.make("C3", N=16)); w.model_kind = 1
    o = Oracle(w)
    x0 = (w.x_nom + 0.01).astype(np.float64)
    u = np.array([0.3, -0.2])
    H = 9
    steps, _, traj = o.rollout(o.lift(x0), u, H=H, want_traj=True)
    assert steps == H
    x = x0.copy()
    for k in range(H):
        z = _py_lift_mono(w.terms, x)
        zn = o.K @ z + o.B @ u
        x = zn[: w.n]
        assert np.allclose(traj[k][: w.n], x, rtol=1e-11, atol=1e-11)
        assert np.allclose(traj[k], _py_lift_mono(w.terms, x), rtol=1e-11, atol=1e-11)     # carried state = Psi(x)
    # and it differs from the linear lifted model on the same inputs (the lifted rows are NOT closed under K)
    w.model_kind = 0
    _, _, lin = Oracle(w).rollout(o.lift(x0), u, H=H, want_traj=True)
    assert not np.allclose(lin[H - 1][: w.n], traj[H - 1][: w.n], rtol=1e-6)


def test_relift_reduces_to_textbook_linear_recursion():
    """If the physical rows of K ignore the lifted features (K[0:n, n:] = 0) the re-lift model is the
    linear system x' = A x + B_x u with A = K[0:n, 0:n]: x_H = A^H x0 + sum A^k B_x u."""
    w = _free(W.make("C2", N=8)); w.model_kind = 1
    w.K = w.K.copy(); w.K[: w.n, w.n:] = 0.0
    o = Oracle(w)
    A, Bx = o.K[: w.n, : w.n], o.B[: w.n]
    x0 = np.array([0.1, -0.05, 0.02, 0.3]); u = np.array([0.7])
    H = 25
    _, _, traj = o.rollout(o.lift(x0), u, H=H, want_traj=True)
    xH = np.linalg.matrix_power(A, H) @ x0 + sum(np.linalg.matrix_power(A, k) @ Bx @ u for k in range(H))
    assert np.allclose(traj[H - 1][: w.n], xH, rtol=1e-10, atol=1e-12)


def test_relift_identity_lift_equals_linear_model():
    w = _free(W.make("C1", N=8))
    n = w.n
    w.d = n; w.K = w.K[:n, :n].copy(); w.B = w.B[:n].copy(); w.terms = w.terms[:n].copy()
    x0 = np.array([0.1, 0.2, -0.1, 0.05]); u = np.array([-0.4])
    w.model_kind = 0
    _, _, a = Oracle(w).rollout(x0, u, H=20, want_traj=True)
    w.model_kind = 1
    _, _, b = Oracle(w).rollout(x0, u, H=20, want_traj=True)
    assert np.array_equal(a, b)
