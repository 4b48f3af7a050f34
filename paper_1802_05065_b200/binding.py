"""ctypes binding of libfpt_b200.so -- same names as include/fpt.h, argument marshalling only.

torch is used for device memory and streams (``tensor.data_ptr()``, ``torch.cuda.current_stream().cuda_stream``); every
step of the path runs in the library's kernels.  The library is loaded on first use; a missing library is an error
(build it with ``python -m paper_1802_05065_b200.build``) -- there is no fallback of any kind.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_HERE = Path(__file__).resolve().parent
_LIB_PATH = _HERE / "libfpt_b200.so"

MODEL = {"overdamped": 0, "underdamped": 1}
SCHEME = {"em": 0, "heun": 1, "paper": 2}
PRECISION = {"fp64": 0, "fp32": 1, "fp32_fast": 2}
HIST_OF = {"gamma": 0, "fpt": 1}
SCHEDULE = {"dynamic": 0, "static": 1}


class FptError(RuntimeError):
    pass


class FptParams(C.Structure):
    """struct fpt_params of include/fpt.h (96 bytes)."""
    _fields_ = [("model", C.c_int32), ("scheme", C.c_int32), ("precision", C.c_int32), ("check_every", C.c_int32),
                ("alpha", C.c_double), ("temperature", C.c_double), ("amp", C.c_double), ("gamma0", C.c_double),
                ("nu", C.c_double), ("phi0", C.c_double), ("v0", C.c_double), ("threshold", C.c_double),
                ("dt", C.c_double), ("first_id", C.c_uint64)]


class FptStats(C.Structure):
    """struct fpt_stats of include/fpt.h."""
    _fields_ = [("n_traj", C.c_uint64), ("n_escaped", C.c_uint64), ("n_censored", C.c_uint64), ("n_nan", C.c_uint64),
                ("useful_steps", C.c_uint64), ("issued_lane_steps", C.c_uint64), ("refill_atomics", C.c_uint64),
                ("n_cap", C.c_uint64), ("grid", C.c_int32), ("block", C.c_int32), ("check_every", C.c_int32),
                ("kernel", C.c_int32), ("migrations", C.c_uint64), ("helper_lane_steps", C.c_uint64),
                ("time_slices", C.c_uint64)]

    def as_dict(self):
        d = {k: int(getattr(self, k)) for k, _ in self._fields_}
        d["lane_efficiency"] = d["useful_steps"] / d["issued_lane_steps"] if d["issued_lane_steps"] else None
        return d


class FptLaunchOpts(C.Structure):
    """struct fpt_launch_opts of include/fpt.h (40 bytes); all zero = the library's defaults."""
    _fields_ = [("block", C.c_int32), ("blocks_per_sm", C.c_int32), ("max_blocks", C.c_int32), ("schedule", C.c_int32),
                ("tail_helper", C.c_int32), ("specialise", C.c_int32), ("consumers", C.c_int32), ("producers", C.c_int32),
                ("time_slice", C.c_int32), ("reserved", C.c_int32)]


class FptHist(C.Structure):
    """struct fpt_hist of include/fpt.h."""
    _fields_ = [("of", C.c_int32), ("nbins", C.c_int32), ("lo", C.c_double), ("hi", C.c_double), ("out_counts", C.c_void_p)]


KERNEL = {0: "fill", 1: "persistent", 2: "specialised"}

_lib = None

_SIGNATURES = {
    "fpt_simulate": [C.POINTER(FptParams), C.c_int64, C.c_uint64, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p],
    "fpt_simulate_hist": [C.POINTER(FptParams), C.c_int64, C.c_uint64, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p,
                          C.c_int32, C.c_double, C.c_double, C.c_int32, C.c_void_p, C.c_void_p],
    "fpt_simulate_ex": [C.POINTER(FptParams), C.c_int64, C.c_uint64, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p,
                        C.POINTER(FptHist), C.POINTER(FptLaunchOpts), C.c_void_p, C.c_void_p],
    "fpt_simulate_noalloc": [C.POINTER(FptParams), C.c_int64, C.c_uint64, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p,
                             C.c_void_p, C.c_void_p],
    "fpt_histogram": [C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_double, C.c_int32, C.c_void_p, C.c_void_p],
    "fpt_simulate_host": [C.POINTER(FptParams), C.c_int64, C.c_uint64, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p,
                          C.c_int32, C.c_double, C.c_double, C.c_int32, C.c_void_p],
    "fpt_simulate_sweep": [C.POINTER(FptParams), C.c_int32, C.c_int64, C.c_uint64, C.POINTER(C.c_double), C.c_void_p,
                           C.c_void_p, C.c_void_p, C.c_void_p],
    "fpt_set_launch": [C.c_int32, C.c_int32, C.c_int32],
    "fpt_set_schedule": [C.c_int32],
    "fpt_set_tail_helper": [C.c_int32],
    "fpt_set_specialise": [C.c_int32, C.c_int32, C.c_int32],
    "fpt_last_stats": [C.POINTER(FptStats)],
    "fpt_fp64_peak": [C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)],
    "fpt_fp32_peak": [C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)],
    "fpt_strerror": [C.c_int],
    "fpt_version": [],
    "fpt_dbg_philox": [C.c_uint64, C.c_uint64, C.c_int64, C.c_uint64, C.c_void_p, C.c_void_p],
    "fpt_dbg_normals_f64": [C.c_uint64, C.c_uint64, C.c_uint64, C.c_int64, C.c_void_p, C.c_void_p],
    "fpt_dbg_normals_f32": [C.c_uint64, C.c_uint64, C.c_uint64, C.c_int64, C.c_void_p, C.c_void_p],
    "fpt_dbg_unary_f64": [C.c_int32, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p],
    "fpt_dbg_unary_f32": [C.c_int32, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p],
    "fpt_dbg_sincos_f64": [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p],
    "fpt_dbg_sincos_f32": [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p],
    "fpt_dbg_selfcheck": [C.c_uint64, C.c_uint64, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p],
    "fpt_dbg_set_helper_seq0": [C.c_uint64],
    "fpt_dbg_set_slice_quantum": [C.c_uint64],
    "fpt_dbg_trace": [C.POINTER(FptParams), C.c_uint64, C.c_uint64, C.c_double, C.c_int64, C.c_void_p, C.c_void_p,
                      C.c_void_p, C.c_void_p, C.c_void_p],
}
EXPORTS = tuple(_SIGNATURES)


def lib():
    """Load libfpt_b200.so (once).  Raises FptError if it has not been built -- there is no fallback."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise FptError(f"{_LIB_PATH} is missing: build it with `python -m paper_1802_05065_b200.build` "
                           "(nvcc, sm_100a).  This package has no CPU fallback.")
        L = C.CDLL(str(_LIB_PATH))
        for name, argtypes in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.argtypes = argtypes
            fn.restype = C.c_char_p if name == "fpt_strerror" else C.c_int
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise FptError(f"{what}: {lib().fpt_strerror(rc).decode()} (code {rc})")


def _stream(stream=None):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def make_params(model="underdamped", scheme="heun", precision="fp64", check_every=0, alpha=0.0, temperature=0.0, amp=1.0,
                gamma0=0.0, nu=0.0, phi0=0.0, v0=0.0, threshold=0.0, dt=0.0, first_id=0, **_ignored) -> FptParams:
    m = MODEL[model] if isinstance(model, str) else int(model)
    s = SCHEME[scheme] if isinstance(scheme, str) else int(scheme)
    pr = PRECISION[precision] if isinstance(precision, str) else int(precision)
    return FptParams(m, s, pr, check_every, alpha, temperature, amp, gamma0, nu, phi0, v0, threshold, dt, first_id)


def _alloc_outputs(n, want_gamma=True, device=None):
    import torch
    device = device or torch.device("cuda", torch.cuda.current_device())
    fpt = torch.empty(n, dtype=torch.float64, device=device)
    gam = torch.empty(n, dtype=torch.float64, device=device) if want_gamma else None
    st = torch.empty(n, dtype=torch.int32, device=device)
    return fpt, gam, st


def simulate(params: FptParams, n_traj: int, seed: int, t_max: float, out=None, stream=None):
    """fpt_simulate.  `out` = (fpt, gamma|None, status) CUDA tensors, allocated when None.  Asynchronous."""
    fpt, gam, st = out if out is not None else _alloc_outputs(n_traj)
    _check(lib().fpt_simulate(C.byref(params), n_traj, seed, t_max, _ptr(fpt), _ptr(gam), _ptr(st), _stream(stream)),
           "fpt_simulate")
    return fpt, gam, st


def launch_opts(block=0, blocks_per_sm=0, max_blocks=0, schedule="dynamic", tail_helper=None, specialise=None, consumers=0,
                producers=0, time_slice=None) -> FptLaunchOpts:
    """fpt_launch_opts.  tail_helper / specialise / time_slice: None = the library's default, True = on / always, False = off /
    never."""
    tri = lambda v: 0 if v is None else (1 if v else -1)
    sch = SCHEDULE[schedule] if isinstance(schedule, str) else int(schedule)
    return FptLaunchOpts(block, blocks_per_sm, max_blocks, sch, tri(tail_helper), tri(specialise), consumers, producers,
                         tri(time_slice), 0)


def alloc_stats(n=1):
    """Device memory for n fpt_stats blocks (the d_stats argument of simulate_ex)."""
    import torch
    return torch.zeros(n * C.sizeof(FptStats), dtype=torch.uint8, device=torch.device("cuda", torch.cuda.current_device()))


def read_stats(d_stats, i=0) -> dict:
    """The i-th fpt_stats block of `d_stats` as a dict (synchronises through the device-to-host copy)."""
    raw = d_stats[i * C.sizeof(FptStats):(i + 1) * C.sizeof(FptStats)].cpu().numpy().tobytes()
    return FptStats.from_buffer_copy(raw).as_dict()


def simulate_ex(params: FptParams, n_traj: int, seed: int, t_max: float, hist=None, opts=None, stats=None, out=None,
                stream=None):
    """fpt_simulate_ex.  hist = (hist_of, lo, hi, nbins, counts CUDA tensor) or None; opts = FptLaunchOpts or None; stats =
    a uint8 CUDA tensor from alloc_stats() (or a (tensor, index) pair) that receives this call's fpt_stats, or None.
    Returns (fpt, gamma, status).  Asynchronous."""
    fpt, gam, st = out if out is not None else _alloc_outputs(n_traj)
    h = None
    if hist is not None:
        of, lo, hi, nb, counts = hist
        h = FptHist(HIST_OF[of] if isinstance(of, str) else int(of), nb, lo, hi, counts.data_ptr())
    sp = C.c_void_p(0)
    if stats is not None:
        t, i = stats if isinstance(stats, tuple) else (stats, 0)
        sp = C.c_void_p(t.data_ptr() + i * C.sizeof(FptStats))
    _check(lib().fpt_simulate_ex(C.byref(params), n_traj, seed, t_max, _ptr(fpt), _ptr(gam), _ptr(st),
                                 C.byref(h) if h is not None else None, C.byref(opts) if opts is not None else None, sp,
                                 _stream(stream)), "fpt_simulate_ex")
    return fpt, gam, st


NOALLOC_MAX_TRAJ = 131072       # FPT_NOALLOC_MAX_TRAJ


def simulate_noalloc(params: FptParams, n_traj: int, seed: int, t_max: float, out, stats=None, stream=None):
    """fpt_simulate_noalloc: `out` = (fpt f64, gamma f64 or None, status i32) CUDA tensors the CALLER allocated; stats as in
    simulate_ex.  The library allocates nothing; calls that overlap on the GPU race on its one scratch array.  Returns out."""
    fpt, gam, st = out
    sp = C.c_void_p(0)
    if stats is not None:
        t, i = stats if isinstance(stats, tuple) else (stats, 0)
        sp = C.c_void_p(t.data_ptr() + i * C.sizeof(FptStats))
    _check(lib().fpt_simulate_noalloc(C.byref(params), n_traj, seed, t_max, _ptr(fpt), _ptr(gam), _ptr(st), sp, _stream(stream)),
           "fpt_simulate_noalloc")
    return out


def simulate_hist(params: FptParams, n_traj: int, seed: int, t_max: float, lo: float, hi: float, nbins: int,
                  hist_of="gamma", counts=None, out=None, stream=None):
    """fpt_simulate_hist.  `counts` (uint64-as-int64 CUDA tensor of nbins+2) is accumulated into; zeros when None."""
    import torch
    fpt, gam, st = out if out is not None else _alloc_outputs(n_traj)
    if counts is None:
        counts = torch.zeros(nbins + 2, dtype=torch.int64, device=fpt.device)
    h = HIST_OF[hist_of] if isinstance(hist_of, str) else int(hist_of)
    _check(lib().fpt_simulate_hist(C.byref(params), n_traj, seed, t_max, _ptr(fpt), _ptr(gam), _ptr(st), h, lo, hi, nbins,
                                   _ptr(counts), _stream(stream)), "fpt_simulate_hist")
    return fpt, gam, st, counts


def histogram(values, status, lo: float, hi: float, nbins: int, counts=None, stream=None):
    import torch
    if counts is None:
        counts = torch.zeros(nbins + 2, dtype=torch.int64, device=values.device)
    _check(lib().fpt_histogram(_ptr(values), _ptr(status), values.numel(), lo, hi, nbins, _ptr(counts), _stream(stream)),
           "fpt_histogram")
    return counts


def simulate_host(params: FptParams, n_traj: int, seed: int, t_max: float, fpt, gamma, status, hist=None):
    """fpt_simulate_host: `fpt`, `gamma` (or None), `status` are HOST buffers (numpy arrays or CPU torch tensors, pinned
    or not); hist = (hist_of, lo, hi, nbins, counts_host) or None.  Synchronous."""
    def hp(a):
        if a is None:
            return C.c_void_p(0)
        return C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)
    if hist is None:
        h, lo, hi, nb, cnt = 0, 0.0, 1.0, 0, None
    else:
        h, lo, hi, nb, cnt = hist
        h = HIST_OF[h] if isinstance(h, str) else int(h)
    _check(lib().fpt_simulate_host(C.byref(params), n_traj, seed, t_max, hp(fpt), hp(gamma), hp(status), h, lo, hi, nb,
                                   hp(cnt)), "fpt_simulate_host")


def simulate_sweep(param_sets, n_per_set: int, seed: int, t_max, out=None, stream=None):
    """fpt_simulate_sweep.  param_sets: sequence of FptParams; t_max: one cap or one per set.  Returns (fpt, gamma,
    status) CUDA tensors of shape (n_sets, n_per_set).  Asynchronous."""
    n_sets = len(param_sets)
    arr = (FptParams * max(1, n_sets))(*param_sets)
    caps = [float(t_max)] * n_sets if not hasattr(t_max, "__len__") else [float(x) for x in t_max]
    if len(caps) != n_sets:
        raise ValueError("t_max must be a scalar or have one entry per parameter set")
    tm = (C.c_double * max(1, n_sets))(*caps)
    fpt, gam, st = out if out is not None else _alloc_outputs(n_sets * n_per_set)
    _check(lib().fpt_simulate_sweep(arr, n_sets, n_per_set, seed, tm, _ptr(fpt), _ptr(gam), _ptr(st), _stream(stream)),
           "fpt_simulate_sweep")
    shape = (n_sets, n_per_set)
    return fpt.view(shape), (gam.view(shape) if gam is not None else None), st.view(shape)


def set_launch(block=0, blocks_per_sm=0, max_blocks=0):
    _check(lib().fpt_set_launch(block, blocks_per_sm, max_blocks), "fpt_set_launch")


def set_schedule(schedule="dynamic"):
    """fpt_set_schedule: "dynamic" (refill + drain compaction, default) or "static" (Appendix A's split, for the A/B)."""
    v = SCHEDULE[schedule] if isinstance(schedule, str) else int(schedule)
    _check(lib().fpt_set_schedule(v), "fpt_set_schedule")


def set_tail_helper(on=True):
    _check(lib().fpt_set_tail_helper(1 if on else 0), "fpt_set_tail_helper")


def set_specialise(specialise=None, consumers=0, producers=0):
    """fpt_set_specialise: None = automatic, True = always, False = never (thread-local default of the plain calls)."""
    v = 0 if specialise is None else (1 if specialise else -1)
    _check(lib().fpt_set_specialise(v, consumers, producers), "fpt_set_specialise")


def last_stats() -> dict:
    s = FptStats()
    _check(lib().fpt_last_stats(C.byref(s)), "fpt_last_stats")
    return s.as_dict()


def fp64_peak(seconds=0.5):
    r, c = C.c_double(), C.c_double()
    _check(lib().fpt_fp64_peak(seconds, C.byref(r), C.byref(c)), "fpt_fp64_peak")
    return r.value, c.value


def fp32_peak(seconds=0.5):
    r, c = C.c_double(), C.c_double()
    _check(lib().fpt_fp32_peak(seconds, C.byref(r), C.byref(c)), "fpt_fp32_peak")
    return r.value, c.value


def version() -> int:
    return lib().fpt_version()


# ---- test hooks ---------------------------------------------------------------------------------------------------
def dbg_philox(seed, id0, n_ids, block, stream=None):
    import torch
    out = torch.empty(4 * n_ids, dtype=torch.int32, device="cuda")
    _check(lib().fpt_dbg_philox(seed, id0, n_ids, block, _ptr(out), _stream(stream)), "fpt_dbg_philox")
    return out


def dbg_normals_f64(seed, tid, b0, nblocks, stream=None):
    import torch
    out = torch.empty(2 * nblocks, dtype=torch.float64, device="cuda")
    _check(lib().fpt_dbg_normals_f64(seed, tid, b0, nblocks, _ptr(out), _stream(stream)), "fpt_dbg_normals_f64")
    return out


def dbg_normals_f32(seed, tid, b0, nblocks, stream=None):
    import torch
    out = torch.empty(4 * nblocks, dtype=torch.float32, device="cuda")
    _check(lib().fpt_dbg_normals_f32(seed, tid, b0, nblocks, _ptr(out), _stream(stream)), "fpt_dbg_normals_f32")
    return out


def dbg_unary_f64(which, x, stream=None):
    import torch
    y = torch.empty_like(x)
    _check(lib().fpt_dbg_unary_f64(which, _ptr(x), _ptr(y), x.numel(), _stream(stream)), "fpt_dbg_unary_f64")
    return y


def dbg_unary_f32(which, x, stream=None):
    import torch
    y = torch.empty_like(x)
    _check(lib().fpt_dbg_unary_f32(which, _ptr(x), _ptr(y), x.numel(), _stream(stream)), "fpt_dbg_unary_f32")
    return y


def dbg_sincos_f64(Y, stream=None):
    import torch
    c = torch.empty(Y.numel(), dtype=torch.float64, device=Y.device)
    s = torch.empty_like(c)
    _check(lib().fpt_dbg_sincos_f64(_ptr(Y), _ptr(c), _ptr(s), Y.numel(), _stream(stream)), "fpt_dbg_sincos_f64")
    return c, s


def dbg_sincos_f32(o, stream=None):
    import torch
    c = torch.empty(o.numel(), dtype=torch.float32, device=o.device)
    s = torch.empty_like(c)
    _check(lib().fpt_dbg_sincos_f32(_ptr(o), _ptr(c), _ptr(s), o.numel(), _stream(stream)), "fpt_dbg_sincos_f32")
    return c, s


def dbg_selfcheck(seed, id0, n_threads, blocks_per_thread, stream=None):
    import torch
    out = torch.zeros(4, dtype=torch.int64, device="cuda")
    _check(lib().fpt_dbg_selfcheck(seed, id0, n_threads, blocks_per_thread, _ptr(out), _stream(stream)), "fpt_dbg_selfcheck")
    return out


def dbg_set_helper_seq0(seq0=0):
    _check(lib().fpt_dbg_set_helper_seq0(seq0), "fpt_dbg_set_helper_seq0")


def dbg_set_slice_quantum(steps=0):
    _check(lib().fpt_dbg_set_slice_quantum(steps), "fpt_dbg_set_slice_quantum")


def dbg_trace(params: FptParams, seed, tid, t_max, trace_len, stream=None):
    import torch
    phi = torch.full((trace_len,), float("nan"), dtype=torch.float64, device="cuda")
    v = torch.full((trace_len,), float("nan"), dtype=torch.float64, device="cuda")
    st = torch.zeros(1, dtype=torch.int32, device="cuda")
    ke = torch.zeros(1, dtype=torch.int64, device="cuda")
    _check(lib().fpt_dbg_trace(C.byref(params), seed, tid, t_max, trace_len, _ptr(phi), _ptr(v), _ptr(st), _ptr(ke),
                               _stream(stream)), "fpt_dbg_trace")
    return phi, v, st, ke
