"""ctypes binding of include/mpmi.h -- same names as the C entry points, marshalling only.

PyTorch is used by callers for device memory and streams (tensor.data_ptr(),
torch.cuda.current_stream().cuda_stream); nothing here computes.
"""
import ctypes as C
import os
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("MPMI_LIB") or os.path.join(_HERE, "libmpmi.so")     # MPMI_LIB: e.g. a build with MPMI_NVCC_EXTRA=-DMPMI_TC_DEBUG

SAMPLER_PHILOX, SAMPLER_GRID = 0, 1
LIFT_MONO, LIFT_RFF = 0, 1
DUMP_NONE, DUMP_PHYS, DUMP_LIFTED = 0, 1, 2
OK, ERR_INVALID, ERR_UNSUPPORTED, ERR_CUDA, ERR_NOMEM = 0, -1, -2, -3, -4
VARIANT_NARROW, VARIANT_WIDE, VARIANT_NO_BINNING, VARIANT_FORCE_BINNING, VARIANT_LATENCY = 1, 2, 4, 8, 16
VARIANT_LAT_R2, VARIANT_LAT_R4, VARIANT_NO_TENSOR, VARIANT_AFFINE, VARIANT_NO_PREDICT = 32, 64, 128, 256, 512
VARIANT_TENSOR32, VARIANT_SMEM_MODEL, VARIANT_TC_UNVERIFIED = 1024, 2048, 4096

EXPORTS = ("mpmi_create", "mpmi_destroy", "mpmi_step", "mpmi_step_result", "mpmi_step_sync",
           "mpmi_step_device", "mpmi_step_trace", "mpmi_profile_enable", "mpmi_profile_timeline", "mpmi_profile_read", "mpmi_shard_step", "mpmi_shard_finalize", "mpmi_rollout_batch",
           "mpmi_get_info", "mpmi_strerror", "mpmi_last_error", "mpmi_tick_noalloc", "mpmi_noalloc_last_error")


class MpmiError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"mpmi status {status}: {text}")
        self.status = status


class _Lift(C.Structure):
    _fields_ = [("kind", C.c_int32), ("terms", C.c_void_p), ("W", C.c_void_p), ("b", C.c_void_p),
                ("scale", C.c_float)]


class _Safe(C.Structure):
    _fields_ = [("nbounds", C.c_int32), ("idx", C.c_void_p), ("lo", C.c_void_p), ("hi", C.c_void_p),
                ("annulus", C.c_int32), ("ix", C.c_int32), ("iy", C.c_int32),
                ("cx", C.c_float), ("cy", C.c_float), ("rmin", C.c_float), ("rmax", C.c_float),
                ("inflate", C.c_float)]


class _Config(C.Structure):
    _fields_ = [("n", C.c_int32), ("m", C.c_int32), ("d", C.c_int32), ("N", C.c_int32), ("H", C.c_int32),
                ("K", C.c_void_p), ("B", C.c_void_p), ("u_lo", C.c_void_p), ("u_hi", C.c_void_p),
                ("sampler", C.c_int32), ("grid_counts", C.c_void_p), ("seed", C.c_uint64),
                ("include_user", C.c_int32), ("lift", _Lift), ("safe", _Safe), ("device", C.c_int32),
                ("shard_begin", C.c_int64), ("shard_count", C.c_int64), ("variant", C.c_int32),
                ("noise_sigma", C.c_float), ("model", C.c_int32), ("reserved", C.c_int32)]


class Result(C.Structure):
    """mpmi_result (include/mpmi.h); identical layout on host and device."""
    _fields_ = [("u", C.c_float * 4), ("index", C.c_int32), ("safe", C.c_int32), ("steps", C.c_int32),
                ("n_safe", C.c_int32), ("dist", C.c_float), ("reserved", C.c_int32),
                ("n_exec", C.c_int64), ("key", C.c_uint64)]

    def as_dict(self, m=4):
        return dict(u=np.array(self.u[:m], dtype=np.float32), index=self.index, safe=self.safe,
                    steps=self.steps, n_safe=self.n_safe, dist=self.dist, n_exec=self.n_exec, key=self.key)


RESULT_DTYPE = np.dtype([("u", np.float32, 4), ("index", np.int32), ("safe", np.int32), ("steps", np.int32),
                         ("n_safe", np.int32), ("dist", np.float32), ("reserved", np.int32),
                         ("n_exec", np.int64), ("key", np.uint64)])
PARTIAL_DTYPE = np.dtype([("key", np.uint64), ("n_safe", np.int64), ("n_exec", np.int64)])
assert RESULT_DTYPE.itemsize == C.sizeof(Result) == 56 and PARTIAL_DTYPE.itemsize == 24


class Info(C.Structure):
    _fields_ = [("d_pad", C.c_int32), ("variant", C.c_int32), ("cand_per_block", C.c_int32),
                ("threads_per_block", C.c_int32), ("blocks", C.c_int32), ("smem_bytes", C.c_int32),
                ("regs_per_thread", C.c_int32), ("sm_count", C.c_int32), ("launches_per_tick", C.c_int32),
                ("uses_graph", C.c_int32), ("binning_cells", C.c_int32), ("reserved", C.c_int32),
                ("ncand_local", C.c_int64)]


_lib = None


def library_path():
    return _LIB_PATH


def load_library():
    """dlopen libmpmi.so; raises (never falls back) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_1906_02318_b200.build` "
                          "(the product has no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, i32, i64, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
    lib.mpmi_create.argtypes = [C.POINTER(_Config), C.POINTER(vp)]
    lib.mpmi_destroy.argtypes = [vp]; lib.mpmi_destroy.restype = None
    lib.mpmi_step.argtypes = [vp, vp, vp, u64, vp]
    lib.mpmi_step_result.argtypes = [vp, C.POINTER(Result)]
    lib.mpmi_step_sync.argtypes = [vp, vp, vp, u64, vp, C.POINTER(Result)]
    lib.mpmi_step_device.argtypes = [vp, vp, vp, u64, vp, vp]
    lib.mpmi_step_trace.argtypes = [vp, vp, vp, u64, vp, vp, vp]
    lib.mpmi_profile_enable.argtypes = [vp, i32]
    lib.mpmi_profile_timeline.argtypes = [vp, vp]
    lib.mpmi_profile_read.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(C.c_float), C.POINTER(C.c_float)]
    lib.mpmi_shard_step.argtypes = [vp, vp, vp, u64, vp, vp]
    lib.mpmi_shard_finalize.argtypes = [vp, vp, i32, vp, u64, vp, vp]
    lib.mpmi_rollout_batch.argtypes = [vp, vp, vp, i64, i64, i32, i32, vp, vp, vp, u64, vp]
    lib.mpmi_get_info.argtypes = [vp, C.POINTER(Info)]
    lib.mpmi_strerror.argtypes = [C.c_int]; lib.mpmi_strerror.restype = C.c_char_p
    lib.mpmi_last_error.argtypes = [vp]; lib.mpmi_last_error.restype = C.c_char_p
    lib.mpmi_tick_noalloc.argtypes = [C.POINTER(_Config), vp, vp, u64, vp, vp]
    lib.mpmi_noalloc_last_error.argtypes = []; lib.mpmi_noalloc_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if getattr(lib, name).restype is C.c_int and name not in ("mpmi_destroy",):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


class Context:
    """mpmi_ctx.  `w` is any object / dict with the fields of mpmi_config (e.g. workloads.Workload)."""

    def __init__(self, w, N=None, H=None, include_user=None, device=-1, shard=(0, 0), variant=0):
        self._lib = load_library()
        g = (lambda k, dflt=None: w[k] if isinstance(w, dict) and k in w else getattr(w, k, dflt))
        self.n, self.m, self.d = int(g("n")), int(g("m")), int(g("d"))
        self.N = int(N if N is not None else g("N"))
        self.H = int(H if H is not None else g("H"))
        self.include_user = int(g("include_user", 1) if include_user is None else include_user)
        keep = self._keep = dict(
            K=_f32(g("K")), B=_f32(g("B")), u_lo=_f32(g("u_lo")), u_hi=_f32(g("u_hi")),
            grid=None if g("grid_counts") is None else np.ascontiguousarray(g("grid_counts"), dtype=np.int32),
            terms=None if g("terms") is None else np.ascontiguousarray(g("terms"), dtype=np.uint8),
            W=_f32(g("W")), b=_f32(g("b")),
            bidx=np.ascontiguousarray(g("bidx") if g("bidx") is not None else [], dtype=np.int32),
            blo=_f32(g("blo", [])), bhi=_f32(g("bhi", [])))
        c = _Config()
        c.n, c.m, c.d, c.N, c.H = self.n, self.m, self.d, self.N, self.H
        c.K, c.B, c.u_lo, c.u_hi = _p(keep["K"]), _p(keep["B"]), _p(keep["u_lo"]), _p(keep["u_hi"])
        c.sampler, c.grid_counts, c.seed = int(g("sampler", 0)), _p(keep["grid"]), int(g("seed", 0))
        c.include_user = self.include_user
        c.lift = _Lift(int(g("lift_kind", 0)), _p(keep["terms"]), _p(keep["W"]), _p(keep["b"]), float(g("scale", 1.0)))
        c.safe = _Safe(len(keep["bidx"]), _p(keep["bidx"]), _p(keep["blo"]), _p(keep["bhi"]),
                       int(g("annulus", 0)), int(g("ix", 0)), int(g("iy", 1)), float(g("cx", 0.0)), float(g("cy", 0.0)),
                       float(g("rmin", 0.0)), float(g("rmax", 0.0)), float(g("inflate", 0.0)))
        c.device, c.shard_begin, c.shard_count, c.variant = device, int(shard[0]), int(shard[1]), variant
        c.noise_sigma, c.model = float(g("noise_sigma", 0.0)), int(g("model_kind", 0))
        h = C.c_void_p()
        rc = self._lib.mpmi_create(C.byref(c), C.byref(h))
        if rc != OK:
            raise MpmiError(rc, self._lib.mpmi_last_error(None).decode() or self._lib.mpmi_strerror(rc).decode())
        self._h = h

    # -- plumbing ---------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != OK:
            raise MpmiError(rc, self._lib.mpmi_last_error(self._h).decode() or self._lib.mpmi_strerror(rc).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.mpmi_destroy(self._h)
            self._h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    @property
    def ncand(self):
        return self.N + (1 if self.include_user else 0)

    def info(self):
        i = Info()
        self._check(self._lib.mpmi_get_info(self._h, C.byref(i)))
        return {k: getattr(i, k) for k, _ in Info._fields_}

    # -- entry points (same names as include/mpmi.h) --------------------------------------------------
    def step(self, x0, u_user, tick, stream=0):
        x0 = _f32(x0); u_user = _f32(u_user)
        self._check(self._lib.mpmi_step(self._h, _p(x0), _p(u_user), int(tick), stream))

    def step_result(self):
        r = Result()
        self._check(self._lib.mpmi_step_result(self._h, C.byref(r)))
        return r

    def step_sync(self, x0, u_user, tick, stream=0):
        x0 = _f32(x0); u_user = _f32(u_user)
        if x0.shape != (self.n,) or u_user.shape != (self.m,):
            raise ValueError("x0 must have n and u_user m entries")
        r = Result()
        self._check(self._lib.mpmi_step_sync(self._h, _p(x0), _p(u_user), int(tick), stream, C.byref(r)))
        return r

    def step_sync_raw(self, x0_ptr, u_ptr, tick, stream, res):
        """no marshalling at all: host pointers in, ctypes Result out (latency harness)"""
        return self._lib.mpmi_step_sync(self._h, x0_ptr, u_ptr, tick, stream, C.byref(res))

    def step_device(self, d_x0, d_u_user, tick, stream, d_out):
        """device pointers (ints, e.g. tensor.data_ptr())"""
        self._check(self._lib.mpmi_step_device(self._h, d_x0, d_u_user, int(tick), stream, d_out))

    def step_trace(self, d_x0, d_u_user, tick, stream, d_out, d_steps):
        self._check(self._lib.mpmi_step_trace(self._h, d_x0, d_u_user, int(tick), stream, d_out, d_steps))

    def profile_enable(self, enable=True):
        self._check(self._lib.mpmi_profile_enable(self._h, 1 if enable else 0))

    def profile_timeline(self, d_stamps):
        self._check(self._lib.mpmi_profile_timeline(self._h, d_stamps))

    def profile_read(self, capacity=64):
        """(ms of the tick kernel, ms of the second pass) per recorded plain-launch tick, oldest first"""
        n = C.c_int32(0)
        a = (C.c_float * capacity)(); b = (C.c_float * capacity)()
        self._check(self._lib.mpmi_profile_read(self._h, capacity, C.byref(n), a, b))
        return np.array(a[: n.value], dtype=np.float64), np.array(b[: n.value], dtype=np.float64)

    def shard_step(self, d_x0, d_u_user, tick, stream, d_partial):
        self._check(self._lib.mpmi_shard_step(self._h, d_x0, d_u_user, int(tick), stream, d_partial))

    def shard_finalize(self, d_partials, G, d_u_user, tick, stream, d_out):
        self._check(self._lib.mpmi_shard_finalize(self._h, d_partials, int(G), d_u_user, int(tick), stream, d_out))

    def rollout_batch(self, d_U, d_X0, x0_count, ncand, H, dump_kind, d_traj, d_steps, d_safe, tick=0, stream=0):
        self._check(self._lib.mpmi_rollout_batch(self._h, d_U, d_X0, int(x0_count), int(ncand), int(H), int(dump_kind),
                                                 d_traj, d_steps, d_safe, int(tick), stream))


def tick_noalloc(w, d_K, d_B, d_x0, d_u_user, tick, stream, d_out, d_terms=None, d_W=None, d_b=None, N=None, H=None,
                 include_user=None, device=-1):
    """mpmi_tick_noalloc: one tick without a context and without any allocation in the library.  `w` carries the small
    host-side fields of mpmi_config (as for Context); the tables are DEVICE pointers (ints): d_K (d*d), d_B (d*m),
    d_terms (d*4 bytes, MONO lift) or d_W / d_b (RFF lift)."""
    lib = load_library()
    g = (lambda k, dflt=None: w[k] if isinstance(w, dict) and k in w else getattr(w, k, dflt))
    keep = dict(u_lo=_f32(g("u_lo")), u_hi=_f32(g("u_hi")),
                grid=None if g("grid_counts") is None else np.ascontiguousarray(g("grid_counts"), dtype=np.int32),
                bidx=np.ascontiguousarray(g("bidx") if g("bidx") is not None else [], dtype=np.int32),
                blo=_f32(g("blo", [])), bhi=_f32(g("bhi", [])))
    c = _Config()
    c.n, c.m, c.d = int(g("n")), int(g("m")), int(g("d"))
    c.N, c.H = int(N if N is not None else g("N")), int(H if H is not None else g("H"))
    c.K, c.B, c.u_lo, c.u_hi = d_K, d_B, _p(keep["u_lo"]), _p(keep["u_hi"])
    c.sampler, c.grid_counts, c.seed = int(g("sampler", 0)), _p(keep["grid"]), int(g("seed", 0))
    c.include_user = int(g("include_user", 1) if include_user is None else include_user)
    c.lift = _Lift(int(g("lift_kind", 0)), d_terms, d_W, d_b, float(g("scale", 1.0)))
    c.safe = _Safe(len(keep["bidx"]), _p(keep["bidx"]), _p(keep["blo"]), _p(keep["bhi"]),
                   int(g("annulus", 0)), int(g("ix", 0)), int(g("iy", 1)), float(g("cx", 0.0)), float(g("cy", 0.0)),
                   float(g("rmin", 0.0)), float(g("rmax", 0.0)), float(g("inflate", 0.0)))
    c.device, c.shard_begin, c.shard_count, c.variant = device, 0, 0, 0
    c.noise_sigma, c.model = float(g("noise_sigma", 0.0)), int(g("model_kind", 0))
    rc = lib.mpmi_tick_noalloc(C.byref(c), d_x0, d_u_user, int(tick), stream, d_out)
    if rc != OK:
        raise MpmiError(rc, lib.mpmi_noalloc_last_error().decode() or lib.mpmi_strerror(rc).decode())
