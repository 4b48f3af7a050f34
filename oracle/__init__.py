"""ctypes loader for the CPU oracle (oracle/fpt_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, by ``__graft_entry__.smoke()`` and by ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs.  Nothing under ``paper_1802_05065_b200/`` imports it, and it
imports nothing from there.  Holds argument marshalling only; all arithmetic is in fpt_oracle.cpp.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "fpt_oracle.cpp"
_LIB = _HERE / "libfpt_oracle.so"

MODEL = {"overdamped": 0, "underdamped": 1}
SCHEME = {"em": 0, "heun": 1, "paper": 2}    # "paper": Alg. 1 / Alg. 3 as printed (gamma_k before the step, strict >)
PRECISION = {"fp64": 0, "fp32": 1}


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags"):
                    return " fma " in (line + " ")
    except OSError:
        pass
    return False


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (no contraction, no fast-math; the only fused ops are explicit std::fma)."""
    if _LIB.exists() and not force and _LIB.stat().st_mtime >= _SRC.stat().st_mtime:
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC"]
    if _cpu_has_fma():
        cmd.append("-mfma")
    tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd += ["-o", str(tmp), str(_SRC)]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


class OracleParams(C.Structure):
    _fields_ = [("model", C.c_int32), ("scheme", C.c_int32), ("precision", C.c_int32), ("reserved", C.c_int32),
                ("alpha", C.c_double), ("temperature", C.c_double), ("amp", C.c_double), ("gamma0", C.c_double),
                ("nu", C.c_double), ("phi0", C.c_double), ("v0", C.c_double), ("threshold", C.c_double),
                ("dt", C.c_double), ("first_id", C.c_uint64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        p_u32, p_u64, p_f64, p_f32, p_i32 = (C.POINTER(t) for t in (C.c_uint32, C.c_uint64, C.c_double, C.c_float, C.c_int32))
        L.oracle_philox4x32_10.argtypes = [p_u32, p_u32, p_u32]
        L.oracle_philox_block.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, p_u32]
        L.oracle_sin_drift.argtypes = [C.c_double]; L.oracle_sin_drift.restype = C.c_double
        L.oracle_uniform_open.argtypes = [C.c_uint64]; L.oracle_uniform_open.restype = C.c_double
        L.oracle_neg2log.argtypes = [C.c_double]; L.oracle_neg2log.restype = C.c_double
        L.oracle_sincos_turns.argtypes = [C.c_uint64, p_f64, p_f64]
        L.oracle_sin_drift_f.argtypes = [C.c_float]; L.oracle_sin_drift_f.restype = C.c_float
        L.oracle_uniform_open_f.argtypes = [C.c_uint32]; L.oracle_uniform_open_f.restype = C.c_float
        L.oracle_neg2log_f.argtypes = [C.c_float]; L.oracle_neg2log_f.restype = C.c_float
        L.oracle_sincos_turns_f.argtypes = [C.c_uint32, p_f32, p_f32]
        L.oracle_sin_drift_v.argtypes = [p_f64, p_f64, C.c_int64]
        L.oracle_neg2log_v.argtypes = [p_f64, p_f64, C.c_int64]
        L.oracle_sincos_turns_v.argtypes = [p_u64, p_f64, p_f64, C.c_int64]
        L.oracle_sin_drift_fv.argtypes = [p_f32, p_f32, C.c_int64]
        L.oracle_neg2log_fv.argtypes = [p_f32, p_f32, C.c_int64]
        L.oracle_sincos_turns_fv.argtypes = [p_u32, p_f32, p_f32, C.c_int64]
        L.oracle_normals_f64.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_int64, p_f64, p_f64, p_f64]
        L.oracle_normals_f32.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_int64, p_f32]
        L.oracle_normals_ids_f64.argtypes = [C.c_uint64, C.c_uint64, C.c_int64, C.c_uint64, p_f64]
        L.oracle_n_cap.argtypes = [C.POINTER(OracleParams), C.c_double]; L.oracle_n_cap.restype = C.c_uint64
        L.oracle_simulate.argtypes = [C.POINTER(OracleParams), C.c_int64, C.c_uint64, C.c_double, p_f64, p_f64, p_i32,
                                      p_u64, p_f64, p_f64, C.c_int]
        L.oracle_simulate.restype = C.c_int
        L.oracle_trace.argtypes = [C.POINTER(OracleParams), C.c_uint64, C.c_uint64, C.c_double, p_f64, C.c_uint64,
                                   C.c_uint64, p_f64, p_f64, p_i32, p_u64]
        L.oracle_trace.restype = C.c_int
        L.oracle_histogram.argtypes = [p_f64, p_i32, C.c_int64, C.c_double, C.c_double, C.c_int32, p_u64]
        L.oracle_histogram.restype = C.c_int
        L.oracle_omp_threads.restype = C.c_int
        _lib = L
    return _lib


def _ptr(a, ctype):
    return a.ctypes.data_as(C.POINTER(ctype))


def make_params(model="underdamped", scheme="heun", precision="fp64", alpha=0.0, temperature=0.0, amp=1.0,
                gamma0=0.0, nu=0.0, phi0=0.0, v0=0.0, threshold=0.0, dt=0.0, first_id=0, **_ignored) -> OracleParams:
    """Build the oracle's parameter block from plain values (strings or ints for the enums)."""
    m = MODEL[model] if isinstance(model, str) else int(model)
    s = SCHEME[scheme] if isinstance(scheme, str) else int(scheme)
    pr = PRECISION[precision] if isinstance(precision, str) else int(precision)
    return OracleParams(m, s, pr, 0, alpha, temperature, amp, gamma0, nu, phi0, v0, threshold, dt, first_id)


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def philox_block(seed, tid, block):
    o = (C.c_uint32 * 4)()
    lib().oracle_philox_block(seed, tid, block, o)
    return tuple(int(x) for x in o)


def sin_drift(x):
    x = np.ascontiguousarray(x, dtype=np.float64); y = np.empty_like(x)
    lib().oracle_sin_drift_v(_ptr(x, C.c_double), _ptr(y, C.c_double), x.size)
    return y


def neg2log(u):
    u = np.ascontiguousarray(u, dtype=np.float64); y = np.empty_like(u)
    lib().oracle_neg2log_v(_ptr(u, C.c_double), _ptr(y, C.c_double), u.size)
    return y


def uniform_open(X):
    return lib().oracle_uniform_open(int(X))


def sincos_turns(Y):
    Y = np.ascontiguousarray(Y, dtype=np.uint64); c = np.empty(Y.shape, np.float64); s = np.empty(Y.shape, np.float64)
    lib().oracle_sincos_turns_v(_ptr(Y, C.c_uint64), _ptr(c, C.c_double), _ptr(s, C.c_double), Y.size)
    return c, s


def sin_drift_f(x):
    x = np.ascontiguousarray(x, dtype=np.float32); y = np.empty_like(x)
    lib().oracle_sin_drift_fv(_ptr(x, C.c_float), _ptr(y, C.c_float), x.size)
    return y


def neg2log_f(u):
    u = np.ascontiguousarray(u, dtype=np.float32); y = np.empty_like(u)
    lib().oracle_neg2log_fv(_ptr(u, C.c_float), _ptr(y, C.c_float), u.size)
    return y


def uniform_open_f(o):
    return lib().oracle_uniform_open_f(int(o))


def sincos_turns_f(o):
    o = np.ascontiguousarray(o, dtype=np.uint32); c = np.empty(o.shape, np.float32); s = np.empty(o.shape, np.float32)
    lib().oracle_sincos_turns_fv(_ptr(o, C.c_uint32), _ptr(c, C.c_float), _ptr(s, C.c_float), o.size)
    return c, s


def normals_f64(seed, tid, b0, nblocks, with_uniforms=False):
    z = np.empty(2 * nblocks, np.float64)
    if with_uniforms:
        u = np.empty(nblocks, np.float64); f = np.empty(nblocks, np.float64)
        lib().oracle_normals_f64(seed, tid, b0, nblocks, _ptr(z, C.c_double), _ptr(u, C.c_double), _ptr(f, C.c_double))
        return z, u, f
    lib().oracle_normals_f64(seed, tid, b0, nblocks, _ptr(z, C.c_double), None, None)
    return z


def normals_f32(seed, tid, b0, nblocks):
    z = np.empty(4 * nblocks, np.float32)
    lib().oracle_normals_f32(seed, tid, b0, nblocks, _ptr(z, C.c_float))
    return z


def normals_ids_f64(seed, id0, nids, block=0):
    z = np.empty(2 * nids, np.float64)
    lib().oracle_normals_ids_f64(seed, id0, nids, block, _ptr(z, C.c_double))
    return z


def n_cap(params: OracleParams, t_max: float) -> int:
    return int(lib().oracle_n_cap(C.byref(params), t_max))


def simulate(params: OracleParams, n_traj: int, seed: int, t_max: float, nthreads: int = 0, with_state: bool = False):
    """Run ids first_id .. first_id+n_traj-1.  Returns dict(fpt, gamma, status, k[, phi_end, v_end])."""
    fpt = np.empty(n_traj, np.float64); gam = np.empty(n_traj, np.float64)
    st = np.empty(n_traj, np.int32); k = np.empty(n_traj, np.uint64)
    pe = np.empty(n_traj, np.float64) if with_state else None
    ve = np.empty(n_traj, np.float64) if with_state else None
    rc = lib().oracle_simulate(C.byref(params), n_traj, seed, t_max, _ptr(fpt, C.c_double), _ptr(gam, C.c_double),
                               _ptr(st, C.c_int32), _ptr(k, C.c_uint64),
                               _ptr(pe, C.c_double) if with_state else None,
                               _ptr(ve, C.c_double) if with_state else None, nthreads)
    if rc != 0:
        raise ValueError("oracle_simulate: invalid parameters")
    out = {"fpt": fpt, "gamma": gam, "status": st, "k": k}
    if with_state:
        out["phi_end"] = pe; out["v_end"] = ve
    return out


def trace(params: OracleParams, seed: int, tid: int, t_max: float, trace_len: int, normals=None):
    """One trajectory with recorded states.  Returns (phi[0..], v[0..], status, k_end); entries past k_end are NaN."""
    phi = np.full(trace_len, np.nan); v = np.full(trace_len, np.nan)
    st = C.c_int32(); ke = C.c_uint64()
    if normals is not None:
        nz = np.ascontiguousarray(normals, dtype=np.float64)
        rc = lib().oracle_trace(C.byref(params), seed, tid, t_max, _ptr(nz, C.c_double), nz.size, trace_len,
                                _ptr(phi, C.c_double), _ptr(v, C.c_double), C.byref(st), C.byref(ke))
    else:
        rc = lib().oracle_trace(C.byref(params), seed, tid, t_max, None, 0, trace_len,
                                _ptr(phi, C.c_double), _ptr(v, C.c_double), C.byref(st), C.byref(ke))
    if rc != 0:
        raise ValueError("oracle_trace: invalid parameters")
    return phi, v, int(st.value), int(ke.value)


def histogram(values, status, lo, hi, nbins, counts=None):
    values = np.ascontiguousarray(values, dtype=np.float64)
    if counts is None:
        counts = np.zeros(nbins + 2, np.uint64)
    st_p = None
    if status is not None:
        status = np.ascontiguousarray(status, dtype=np.int32); st_p = _ptr(status, C.c_int32)
    rc = lib().oracle_histogram(_ptr(values, C.c_double), st_p, values.size, lo, hi, nbins, _ptr(counts, C.c_uint64))
    if rc != 0:
        raise ValueError("oracle_histogram: invalid arguments")
    return counts


def omp_threads() -> int:
    return int(lib().oracle_omp_threads())
