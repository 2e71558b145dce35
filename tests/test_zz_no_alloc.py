"""mpmi_tick_noalloc (include/mpmi.h, csrc/noalloc.cu): the tick for callers that may not allocate.  Its scratch (packed
model + cross-CTA selection state) is one static __device__ array, so there is no oracle-side meaning to test here: the
entry point must give, call after call, exactly what the existing register-kernel path (mpmi_create + mpmi_step_device)
gives for the same configuration -- every field of mpmi_result bit for bit (tolerance 0, as in test_parity_gpu.py's
kernel-vs-kernel comparisons).  Collected last on purpose (pytest -x)."""
import copy
import ctypes

import numpy as np
import pytest

import workloads as W
from workloads import generate as G

FIELDS = ("index", "safe", "steps", "n_safe", "n_exec", "key")


def _rff24():
    """RFF lift within the entry point's limit: the first 24 lifted dims of T48 (d = 48)"""
    w = copy.copy(W.make("T48", N=20000))
    d = 24
    w.K = np.ascontiguousarray(w.K[:d, :d]); w.B = np.ascontiguousarray(w.B[:d])
    w.W = np.ascontiguousarray(w.W[: d - w.n]); w.b = np.ascontiguousarray(w.b[: d - w.n]); w.d = d
    return w


def _cases():
    c3 = W.make("C3")
    return [("C1", W.make("C1", N=10000)), ("C2", W.make("C2", N=10000)), ("C3_grid", c3), ("C4", W.make("C4", N=50000 + 37)),
            ("C4_all_unsafe", G.scaled_bounds(W.make("C4", N=3000), 0.01)), ("rff24", _rff24())]


def _row(t):
    return np.frombuffer(t.cpu().numpy().tobytes(), dtype=_mp().mpmi.RESULT_DTYPE)[0]


def _mp():
    import paper_1906_02318_b200 as mp
    return mp


@pytest.mark.gpu
@pytest.mark.parametrize("name", [c[0] for c in _cases()])
def test_no_alloc_tick_equals_context_tick_call_after_call(name):
    import torch
    mp = _mp()
    mp.load_library()
    w = dict(_cases())[name]
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    dev = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a, dtype=dt)).cuda()
    dK, dB = dev(w.K, np.float32), dev(w.B, np.float32)
    dterms = dev(w.terms, np.uint8) if w.lift_kind == 0 else None
    dW = dev(w.W, np.float32) if w.lift_kind == 1 else None
    db = dev(w.b, np.float32) if w.lift_kind == 1 else None
    ptr = lambda t: None if t is None else t.data_ptr()
    x0s, uus, ticks = W.tick_inputs(w, 3)
    # the existing path: the register kernel of a context (NARROW keeps small N off the latency kernel, whose row sums are
    # associated differently -- rollout_lat.cuh -- so that a candidate within rounding of the boundary may differ there)
    ctx = mp.Context(w, variant=mp.mpmi.VARIANT_NO_TENSOR | mp.mpmi.VARIANT_NARROW)
    assert ctx.info()["variant"] == 1
    ref = torch.zeros(56, dtype=torch.uint8, device="cuda")
    out = torch.zeros(56, dtype=torch.uint8, device="cuda")
    rows = []
    # two different ticks in a row, then the first one again: the shared scratch array keeps nothing a later call trips over
    for i in (0, 1, 0):
        dx, du = dev(x0s[i], np.float32), dev(uus[i], np.float32)
        ctx.step_device(dx.data_ptr(), du.data_ptr(), int(ticks[i]), stream, ref.data_ptr())
        out.fill_(0xAB)
        mp.mpmi.tick_noalloc(w, dK.data_ptr(), dB.data_ptr(), dx.data_ptr(), du.data_ptr(), int(ticks[i]), stream, out.data_ptr(),
                             d_terms=ptr(dterms), d_W=ptr(dW), d_b=ptr(db))
        torch.cuda.synchronize()
        g, r = _row(out), _row(ref)
        for f in FIELDS:
            assert int(g[f]) == int(r[f]), (name, i, f, g, r)
        assert g["u"].tobytes() == r["u"].tobytes() and g["dist"].tobytes() == r["dist"].tobytes(), (name, i, g, r)
        assert 0 <= int(g["index"]) <= w.N
        rows.append(g.copy())
    assert rows[0].tobytes() == rows[2].tobytes()
    if name == "C4_all_unsafe":
        assert rows[0]["safe"] == 0 and rows[0]["n_safe"] == 0
    elif name != "rff24":
        assert any(r["n_safe"] > 0 for r in rows)
    ctx.close()


@pytest.mark.gpu
def test_no_alloc_non_finite_input_gives_index_minus_one():
    import torch
    mp = _mp()
    w = W.make("C2", N=4000)
    stream = torch.cuda.current_stream().cuda_stream
    dK, dB, dt = torch.as_tensor(w.K).cuda(), torch.as_tensor(w.B).cuda(), torch.as_tensor(w.terms).cuda()
    x0s, uus, ticks = W.tick_inputs(w, 1)
    x = x0s[0].copy(); x[1] = np.nan
    dx, du = torch.as_tensor(x).cuda(), torch.as_tensor(uus[0]).cuda()
    out = torch.zeros(56, dtype=torch.uint8, device="cuda")
    for _ in range(2):          # the aborted-looking tick must leave the scratch usable
        mp.mpmi.tick_noalloc(w, dK.data_ptr(), dB.data_ptr(), dx.data_ptr(), du.data_ptr(), 0, stream, out.data_ptr(), d_terms=dt.data_ptr())
        torch.cuda.synchronize()
        assert int(_row(out)["index"]) == -1


def test_no_alloc_rejects_sizes_beyond_the_static_scratch():
    """the size check comes before any CUDA call: it runs without a GPU"""
    mp = _mp()
    w = W.make("C5", N=1000)                                          # d = 128 > 32
    with pytest.raises(mp.MpmiError) as e:
        mp.mpmi.tick_noalloc(w, 1 << 20, 1 << 20, 1 << 20, 1 << 20, 0, None, 1 << 20, d_W=1 << 20, d_b=1 << 20)
    assert e.value.status == mp.mpmi.ERR_UNSUPPORTED and "maximum of 32" in str(e.value)
    w = copy.copy(W.make("C4", N=1000)); w.noise_sigma = 0.1
    with pytest.raises(mp.MpmiError) as e:
        mp.mpmi.tick_noalloc(w, 1 << 20, 1 << 20, 1 << 20, 1 << 20, 0, None, 1 << 20, d_terms=1 << 20)
    assert e.value.status == mp.mpmi.ERR_UNSUPPORTED and "noise" in str(e.value)
    lib = mp.load_library()
    assert lib.mpmi_tick_noalloc(None, None, None, 0, None, None) == mp.mpmi.ERR_INVALID
    assert b"null" in lib.mpmi_noalloc_last_error()
    assert ctypes.sizeof(mp.mpmi.Result) == 56
