"""Seeded synthetic workloads C1..C5 (BASELINE.json:configs[0..4]).

The paper's learned Koopman models, simulators and human data are not available, so these
inputs stand in for them and take only the SHAPES and STRUCTURE of the paper's workloads:
N ~ 1e4 candidates, 1-D and multi-D bounded joystick boxes, grid and
uniform sampling, short horizons, 28-50 % safe rollouts
(Table I).

This module contains no arithmetic of the method itself: it draws matrices, tables and
boundary constants with numpy's default_rng and applies the input-gain / scaling constants that
oracle/calibrate.py stored in workloads/calibration.json.
Order of draws is fixed: G, B, [W, b], then tick inputs from a second generator (seed+1000).
"""
import json
import os
from dataclasses import dataclass, field
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
CALIBRATION_JSON = os.path.join(_HERE, "calibration.json")
C2_SEQUENCE = os.path.join(_HERE, "c2_tick_sequence.txt")   # written by oracle/make_c2_sequence.py
CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")
# Extra parity-test workloads (not bench lines): shapes that BASELINE.json's five configs do not reach --
# T48: lifted dim 48 (zero-padded to 64 -> the D = 64 warp-tile kernel), T4: a 4-dimensional input box (M = 4 kernels).
TEST_NAMES = ("T48", "T4")

ONE = 0xFF           # lift factor codes (include/mpmi.h: mpmi_lift_spec.terms)
SIN, COS = 0x40, 0x80


def _X(j):
    return j


@dataclass
class Workload:
    name: str
    n: int
    m: int
    d: int
    N: int
    H: int
    K: np.ndarray
    B: np.ndarray
    u_lo: np.ndarray
    u_hi: np.ndarray
    sampler: int = 0                      # 0 Philox, 1 grid
    grid_counts: np.ndarray = None
    seed: int = 0
    include_user: int = 1
    lift_kind: int = 0                    # 0 MONO (products of x_j, sin x_j, cos x_j), 1 RFF
    terms: np.ndarray = None
    W: np.ndarray = None
    b: np.ndarray = None
    scale: float = 1.0
    bidx: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int32))
    blo: np.ndarray = field(default_factory=lambda: np.zeros(0, np.float32))
    bhi: np.ndarray = field(default_factory=lambda: np.zeros(0, np.float32))
    annulus: int = 0
    ix: int = 0
    iy: int = 1
    cx: float = 0.0
    cy: float = 0.0
    rmin: float = 0.0
    rmax: float = 0.0
    inflate: float = 0.0
    noise_sigma: float = 0.0              # std of the additive prediction noise; 0 = none
    model_kind: int = 0                   # 0 linear lifted model, 1 re-lift every step
    x_nom: np.ndarray = None
    x_pert: np.ndarray = None             # per-dimension perturbation half-width for tick inputs
    rho: float = 0.0
    gamma: float = 1.0
    model_seed: int = 0


def _terms_from_lists(lists):
    t = np.full((len(lists), 4), ONE, dtype=np.uint8)
    for f, fac in enumerate(lists):
        assert len(fac) <= 4
        for q, code in enumerate(fac):
            t[f, q] = code
    return t


def _pairs(n):
    return [(i, j) for i in range(n) for j in range(i, n)]


def lift_terms(name):
    """Factor-code tables for the monomial / trig-polynomial lifts (reading G12)."""
    if name == "C1":      # x0..x3, x0^2, x0x1, x0x2, x0x3
        return _terms_from_lists([[0], [1], [2], [3], [0, 0], [0, 1], [0, 2], [0, 3]])
    if name in ("C2", "T4"):      # x0..x3, the 10 products x_i x_j (i<=j), then x1^3, x3^3
        return _terms_from_lists([[j] for j in range(4)] + [list(p) for p in _pairs(4)] + [[1, 1, 1], [3, 3, 3]])
    if name in ("C3", "C4"):  # (x,y,th,vx,vy,om), sin th, cos th, 21 products, vx cos, vx sin, vy cos
        return _terms_from_lists([[j] for j in range(6)] + [[SIN + 2], [COS + 2]] + [list(p) for p in _pairs(6)]
                                 + [[3, COS + 2], [3, SIN + 2], [4, COS + 2]])
    raise KeyError(name)


_SPEC = {
    #        n  m  d    N        H    rho    sampler
    "C1": (4, 1, 8, 1024, 50, 0.98, 0),
    "C2": (4, 1, 16, 10000, 100, 0.99, 0),
    "C3": (6, 2, 32, 10000, 60, 0.995, 1),
    "C4": (6, 2, 32, 1 << 20, 100, 0.995, 0),
    "C5": (8, 3, 128, 262144, 100, 0.99, 0),
    "T48": (8, 3, 48, 4096, 60, 0.99, 0),
    "T4": (4, 4, 16, 4096, 50, 0.98, 0),
}
_EPS_NEAR_IDENTITY = 1e-4   # C3/C4: K = S (rho (I+eps G)/rho(I+eps G)) S^-1


def load_calibration():
    if os.path.exists(CALIBRATION_JSON):
        with open(CALIBRATION_JSON) as f:
            return json.load(f)
    return {}


def make(name, N=None, H=None, calibrated=True, model_seed=None, gamma=None, S=None):
    """Build workload `name`.  calibrated=False gives the literal config (gamma = 1).
    model_seed / gamma / S override calibration.json (used by oracle/calibrate.py itself)."""
    n, m, d, N0, H0, rho, sampler = _SPEC[name]
    cal = load_calibration().get(name, {}) if calibrated else {}
    if model_seed is None:
        model_seed = int(cal.get("model_seed", 0))
    if gamma is None:
        gamma = float(cal.get("gamma", 1.0))
    if S is None and "S" in cal:
        S = np.asarray(cal["S"], dtype=np.float64)
    rng = np.random.default_rng(model_seed)
    G = rng.standard_normal((d, d))
    Bm = 0.1 * rng.standard_normal((d, m))
    w = dict(lift_kind=0, terms=None, W=None, b=None, scale=1.0)
    if name in ("C5", "T48"):
        W = rng.standard_normal((d - n, n))
        b = rng.uniform(0.0, 2.0 * np.pi, d - n)
        w.update(lift_kind=1, W=W.astype(np.float32), b=b.astype(np.float32),
                 scale=float(np.float32(np.sqrt(2.0 / (d - n)))))
    else:
        w.update(terms=lift_terms(name))
    if name in ("C3", "C4"):
        Kt = np.eye(d) + _EPS_NEAR_IDENTITY * G
        Kt = rho * Kt / np.max(np.abs(np.linalg.eigvals(Kt)))
        if S is None:
            S = np.ones(d)
        K = (S[:, None] * Kt) / S[None, :]
    else:
        K = rho * G / np.max(np.abs(np.linalg.eigvals(G)))
    Bm = gamma * Bm
    kw = dict(name=name, n=n, m=m, d=d, N=int(N or N0), H=int(H or H0),
              K=K.astype(np.float32), B=Bm.astype(np.float32),
              u_lo=-np.ones(m, np.float32), u_hi=np.ones(m, np.float32),
              sampler=sampler, seed=0, rho=rho, gamma=gamma, model_seed=model_seed, **w)
    if name in ("C1", "C2", "T4"):    # safe iff |x1| < 0.5 and |x0| < 2
        kw.update(bidx=np.array([0, 1], np.int32), blo=np.array([-2.0, -0.5], np.float32),
                  bhi=np.array([2.0, 0.5], np.float32), x_nom=np.zeros(4, np.float32),
                  x_pert=np.array([0.5, 0.1, 0.2, 0.2], np.float32))
    elif name in ("C3", "C4"):        # safe iff 8 <= hypot(x, y) <= 12
        kw.update(annulus=1, ix=0, iy=1, cx=0.0, cy=0.0, rmin=8.0, rmax=12.0,
                  x_nom=np.array([11.5, 0.0, np.pi / 2, 0.0, 1.0, 0.1], np.float32),
                  x_pert=np.array([0.2, 0.2, 0.05, 0.05, 0.05, 0.01], np.float32))
        if name == "C3":
            kw.update(grid_counts=np.array([100, 100], np.int32))
    else:                              # C5: |x_j| < 1, j < 8
        kw.update(bidx=np.arange(8, dtype=np.int32), blo=-np.ones(8, np.float32), bhi=np.ones(8, np.float32),
                  x_nom=np.zeros(8, np.float32), x_pert=np.full(8, 0.1, np.float32))
    return Workload(**kw)


def scaled_bounds(w, factor):
    """Copy of w with the safe set shrunk (factor<1) or enlarged (factor>1): the forced-fallback
    and forced-all-safe parity sets of SURVEY 8(d)."""
    import copy
    v = copy.copy(w)
    if len(w.bidx):
        mid = 0.5 * (w.blo + w.bhi); half = 0.5 * (w.bhi - w.blo) * factor
        v.blo = (mid - half).astype(np.float32); v.bhi = (mid + half).astype(np.float32)
    if w.annulus:
        mid = 0.5 * (w.rmin + w.rmax); half = 0.5 * (w.rmax - w.rmin) * factor
        v.rmin = float(np.float32(max(mid - half, 0.0))); v.rmax = float(np.float32(mid + half))
    return v


def rescaled_units(w, s):
    """The same RFF workload (C5, T48) with the physical state measured in units s times smaller, x -> s x: lifted states,
    bounds and input gain grow by s while every trajectory is the same up to that factor -- the stress case in which the
    ABSOLUTE 1e-4 margin of rule T2 becomes relative 1e-4 / s."""
    import copy
    assert w.lift_kind == 1
    v = copy.copy(w)
    v.W = (w.W / s).astype(np.float32); v.scale = float(np.float32(w.scale * s))
    v.B = (w.B * s).astype(np.float32)
    v.blo = (w.blo * s).astype(np.float32); v.bhi = (w.bhi * s).astype(np.float32)
    v.x_nom = (w.x_nom * s).astype(np.float32); v.x_pert = (w.x_pert * s).astype(np.float32)
    return v


def tick_inputs(w, count, seed=None):
    """(x0_t, u_user_t, tick_t) for t < count: x0 = x_nom + seeded perturbation,
    u_user uniform in a box 10 % wider than the input box (so clamping is exercised)."""
    rng = np.random.default_rng((w.model_seed if seed is None else seed) + 1000)
    x0 = w.x_nom[None, :] + rng.uniform(-1.0, 1.0, (count, w.n)) * w.x_pert[None, :]
    mid = 0.5 * (w.u_lo + w.u_hi); half = 0.55 * (w.u_hi - w.u_lo)
    uu = mid[None, :] + rng.uniform(-1.0, 1.0, (count, w.m)) * half[None, :]
    ticks = np.arange(count, dtype=np.uint64)
    return x0.astype(np.float32), uu.astype(np.float32), ticks
