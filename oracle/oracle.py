"""ctypes wrapper around oracle/mpmi_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke(), bench.py (cpu_baseline leg and --impl reference) and
oracle/calibrate.py may import this module.  It imports nothing from paper_1906_02318_b200.
Every numerical step is in mpmi_oracle.c (Algorithm 2); this file only
marshals arrays.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "mpmi_oracle.c")


def build(force=False):
    """Compile the oracle with gcc (plain -O2, OpenMP only for the paper's parallel-for)."""
    hdr = os.path.join(_HERE, "mpmi_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr))):
        return _SO
    subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall",
                           "-o", _SO, _SRC, "-lm"])
    return _SO


class _Cfg(C.Structure):
    _fields_ = [("n", C.c_int32), ("m", C.c_int32), ("d", C.c_int32), ("N", C.c_int32), ("H", C.c_int32),
                ("K", C.c_void_p), ("B", C.c_void_p), ("u_lo", C.c_void_p), ("u_hi", C.c_void_p),
                ("sampler", C.c_int32), ("grid_counts", C.c_void_p), ("seed", C.c_uint64),
                ("include_user", C.c_int32), ("lift_kind", C.c_int32), ("terms", C.c_void_p),
                ("W", C.c_void_p), ("b", C.c_void_p), ("scale", C.c_double),
                ("nbounds", C.c_int32), ("bidx", C.c_void_p), ("blo", C.c_void_p), ("bhi", C.c_void_p),
                ("annulus", C.c_int32), ("ix", C.c_int32), ("iy", C.c_int32),
                ("cx", C.c_double), ("cy", C.c_double), ("rmin", C.c_double), ("rmax", C.c_double),
                ("inflate", C.c_double), ("noise_sigma", C.c_double), ("model_kind", C.c_int32)]


class _Res(C.Structure):
    _fields_ = [("u", C.c_double * 4), ("index", C.c_int32), ("safe", C.c_int32), ("steps", C.c_int32),
                ("n_safe", C.c_int32), ("dist", C.c_double), ("n_exec", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_step.restype = C.c_int
        _lib.orc_rollout_batch.restype = C.c_int
        _lib.orc_rollout.restype = C.c_int
        _lib.orc_is_safe.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    """One problem instance (model, lift, safe set, sampler).  `w` is a workloads.Workload-like
    object or dict with the fields of orc_config (numpy arrays, any float dtype)."""

    def __init__(self, w, N=None, H=None, include_user=None):
        g = (lambda k, dflt=None: w[k] if isinstance(w, dict) and k in w else getattr(w, k, dflt))
        self.n, self.m, self.d = int(g("n")), int(g("m")), int(g("d"))
        self.N = int(N if N is not None else g("N"))
        self.H = int(H if H is not None else g("H"))
        self.include_user = int(g("include_user", 1) if include_user is None else include_user)
        f64 = lambda a: None if a is None else np.ascontiguousarray(np.asarray(a, dtype=np.float32).astype(np.float64))
        self.K = f64(g("K")); self.B = f64(g("B"))
        assert self.K.shape == (self.d, self.d) and self.B.shape == (self.d, self.m)
        self.u_lo = np.ascontiguousarray(g("u_lo"), dtype=np.float32)
        self.u_hi = np.ascontiguousarray(g("u_hi"), dtype=np.float32)
        self.sampler = int(g("sampler", 0))
        gc = g("grid_counts")
        self.grid_counts = None if gc is None else np.ascontiguousarray(gc, dtype=np.int32)
        self.seed = int(g("seed", 0))
        self.lift_kind = int(g("lift_kind", 0))
        t = g("terms")
        self.terms = None if t is None else np.ascontiguousarray(t, dtype=np.uint8)
        self.W = f64(g("W")); self.b = f64(g("b"))
        self.scale = float(np.float32(g("scale", 1.0)))
        bi = g("bidx")
        self.bidx = np.ascontiguousarray(bi if bi is not None else [], dtype=np.int32)
        self.blo = np.ascontiguousarray(np.asarray(g("blo", []), dtype=np.float32).astype(np.float64))
        self.bhi = np.ascontiguousarray(np.asarray(g("bhi", []), dtype=np.float32).astype(np.float64))
        self.annulus = int(g("annulus", 0))
        f32 = lambda v: float(np.float32(v))
        self.ix, self.iy = int(g("ix", 0)), int(g("iy", 1))
        self.cx, self.cy = f32(g("cx", 0.0)), f32(g("cy", 0.0))
        self.rmin, self.rmax = f32(g("rmin", 0.0)), f32(g("rmax", 0.0))
        self.inflate = f32(g("inflate", 0.0))
        self.noise_sigma = f32(g("noise_sigma", 0.0))
        self.model_kind = int(g("model_kind", 0))
        self._cfg = self._make_cfg()

    def _make_cfg(self):
        c = _Cfg()
        c.n, c.m, c.d, c.N, c.H = self.n, self.m, self.d, self.N, self.H
        c.K, c.B, c.u_lo, c.u_hi = _p(self.K), _p(self.B), _p(self.u_lo), _p(self.u_hi)
        c.sampler, c.grid_counts, c.seed = self.sampler, _p(self.grid_counts), self.seed
        c.include_user, c.lift_kind, c.terms = self.include_user, self.lift_kind, _p(self.terms)
        c.W, c.b, c.scale = _p(self.W), _p(self.b), self.scale
        c.nbounds, c.bidx, c.blo, c.bhi = len(self.bidx), _p(self.bidx), _p(self.blo), _p(self.bhi)
        c.annulus, c.ix, c.iy = self.annulus, self.ix, self.iy
        c.cx, c.cy, c.rmin, c.rmax, c.inflate = self.cx, self.cy, self.rmin, self.rmax, self.inflate
        c.noise_sigma, c.model_kind = self.noise_sigma, self.model_kind
        return c

    @property
    def ncand(self):
        return self.N + (1 if self.include_user else 0)

    def sample(self, tick, idx):
        """fp32 candidate inputs u_i for the indices in idx -> (len, m) float32."""
        idx = np.atleast_1d(np.asarray(idx, dtype=np.int64))
        out = np.empty((len(idx), self.m), dtype=np.float32)
        u = (C.c_float * 4)()
        for r, i in enumerate(idx):
            lib().orc_sample(C.byref(self._cfg), C.c_uint64(tick), C.c_int64(int(i)), u)
            out[r] = u[: self.m]
        return out

    def lift(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        z = np.empty(self.d, dtype=np.float64)
        lib().orc_lift(C.byref(self._cfg), _p(x), _p(z))
        return z

    def is_safe(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        mg = C.c_double()
        s = lib().orc_is_safe(C.byref(self._cfg), _p(x), C.byref(mg))
        return bool(s), mg.value

    def noise(self, tick, i, k):
        """The n standard normals added (times noise_sigma) to the physical rows of candidate i at step k."""
        eps = np.empty(self.n, dtype=np.float64)
        lib().orc_noise(C.byref(self._cfg), C.c_uint64(tick), C.c_int64(int(i)), C.c_int(int(k)), _p(eps))
        return eps

    def rollout(self, z0, u, H=None, want_traj=False, tick=0, i=0):
        H = self.H if H is None else H
        z0 = np.ascontiguousarray(z0, dtype=np.float64); u = np.ascontiguousarray(u, dtype=np.float64)
        traj = np.empty((H, self.d), dtype=np.float64) if want_traj else None
        mg = C.c_double()
        steps = lib().orc_rollout(C.byref(self._cfg), _p(z0), _p(u), C.c_int(H), C.c_uint64(tick), C.c_int64(int(i)),
                                  C.byref(mg), _p(traj))
        return steps, mg.value, traj

    def step(self, x0, u_user, tick, detail=False):
        x0 = np.ascontiguousarray(x0, dtype=np.float32); u_user = np.ascontiguousarray(u_user, dtype=np.float32)
        assert x0.shape == (self.n,) and u_user.shape == (self.m,)
        res = _Res()
        NC = self.ncand
        steps = np.empty(NC, dtype=np.int32) if detail else None
        marg = np.empty(NC, dtype=np.float64) if detail else None
        dist = np.empty(NC, dtype=np.float64) if detail else None
        U = np.empty((NC, self.m), dtype=np.float32) if detail else None
        rc = lib().orc_step(C.byref(self._cfg), _p(x0), _p(u_user), C.c_uint64(tick), C.byref(res),
                            _p(steps), _p(marg), _p(dist), _p(U))
        if rc != 0:
            raise ValueError("oracle: non-finite x0 / u_user")
        out = dict(u=np.array(res.u[: self.m], dtype=np.float64).astype(np.float32), index=res.index,
                   safe=res.safe, steps=res.steps, n_safe=res.n_safe, dist=res.dist, n_exec=res.n_exec)
        if detail:
            out.update(steps_all=steps, margin_all=marg, dist_all=dist, U=U)
        return out

    def rollout_batch(self, U, X0, H=None, want_traj=False, tick=0):
        H = self.H if H is None else H
        U = np.ascontiguousarray(U, dtype=np.float32).reshape(-1, self.m)
        X0 = np.ascontiguousarray(X0, dtype=np.float32).reshape(-1, self.n)
        Nc = U.shape[0]
        steps = np.empty(Nc, dtype=np.int32); marg = np.empty(Nc, dtype=np.float64)
        traj = np.empty((Nc, H, self.d), dtype=np.float64) if want_traj else None
        rc = lib().orc_rollout_batch(C.byref(self._cfg), _p(U), _p(X0), C.c_int(X0.shape[0]), C.c_int64(Nc),
                                     C.c_int(H), C.c_uint64(tick), _p(steps), _p(marg), _p(traj))
        if rc != 0:
            raise ValueError("oracle: x0_count must be 1 or N")
        return steps, marg, traj


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) for v in ctr]); k = (C.c_uint32 * 2)(*[int(v) for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def num_threads():
    return int(lib().orc_num_threads())
