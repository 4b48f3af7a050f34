"""Boundary checks that need no GPU: the C-ABI library builds, loads and exports every symbol include/fpt.h declares,
the struct layouts match the header, and argument validation (FPT_E_INVALID) happens before any CUDA work."""
import ctypes as C
import math
import re
from pathlib import Path

import pytest

import paper_1802_05065_b200 as fpt
from paper_1802_05065_b200 import binding, build

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    build.build()
    return fpt.lib()


def test_exports_every_declared_symbol(lib):
    declared = set()
    for name in ("fpt.h", "fpt_dbg.h"):               # product API + test hooks / microbenchmarks
        header = (ROOT / "include" / name).read_text()
        code = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
        declared |= set(re.findall(r"\b(fpt_[a-z0-9_]+)\s*\(", code))
    assert len(declared) >= 25
    product = re.sub(r"/\*.*?\*/", "", (ROOT / "include" / "fpt.h").read_text(), flags=re.S)
    assert "fpt_dbg_" not in product and "_peak" not in product      # hooks live in fpt_dbg.h only
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(binding.EXPORTS)          # the binding covers the whole header, and nothing else


def test_struct_layouts(lib):
    assert C.sizeof(fpt.FptParams) == 96              # 4 x int32, 9 x double, 1 x uint64, no padding
    assert fpt.FptParams.first_id.offset == 88
    assert C.sizeof(fpt.FptStats) == 104 and fpt.FptStats.time_slices.offset == 96
    assert fpt.FptStats.migrations.offset == 80 and fpt.FptStats.kernel.offset == 76
    assert C.sizeof(fpt.FptLaunchOpts) == 40 and fpt.FptLaunchOpts.producers.offset == 28 and fpt.FptLaunchOpts.time_slice.offset == 32
    assert C.sizeof(fpt.FptHist) == 32 and fpt.FptHist.out_counts.offset == 24
    assert fpt.version() >= 200


def test_strerror(lib):
    assert lib.fpt_strerror(0) == b"ok"
    assert lib.fpt_strerror(-1) == b"invalid argument"
    assert lib.fpt_strerror(-99) == b"unknown error code"
    assert b"beyond the fixed maximum" in lib.fpt_strerror(-3)


def _good():
    return dict(fpt.workload("c2")["params"])


def test_hardware_sine_precision_only_with_the_paper_scheme_and_a_sine(lib):
    base = dict(_good(), precision="fp32_fast")
    call = lambda kw: lib.fpt_simulate(C.byref(fpt.make_params(**kw)), 10, 1, 1.0, C.c_void_p(8), None, C.c_void_p(8), None)
    assert call(dict(base, scheme="heun")) == -1 and call(dict(base, scheme="em")) == -1
    assert call(dict(base, scheme="paper", amp=0.0)) == -1
    assert call(dict(base, scheme=3)) == -1 and call(dict(_good(), precision=3)) == -1
    import torch
    if not torch.cuda.is_available():
        assert call(dict(base, scheme="paper")) == -2          # valid: gets as far as the (absent) device


@pytest.mark.parametrize("field,value", [("dt", 0.0), ("dt", -1.0), ("dt", math.nan), ("temperature", -0.1), ("alpha", -1.0),
                                         ("model", 2), ("scheme", -1), ("precision", 3), ("check_every", -1),
                                         ("gamma0", math.inf), ("threshold", math.nan)])
def test_invalid_params_rejected_before_any_cuda_work(lib, field, value):
    kw = _good()
    kw[field] = value
    p = fpt.make_params(**kw)
    # non-null dummy pointers: validation must reject before touching them (there is no GPU here)
    rc = lib.fpt_simulate(C.byref(p), 10, 1, 1.0, C.c_void_p(8), C.c_void_p(8), C.c_void_p(8), None)
    assert rc == -1


def test_invalid_call_arguments(lib):
    p = fpt.make_params(**_good())
    assert lib.fpt_simulate(None, 10, 1, 1.0, C.c_void_p(8), None, C.c_void_p(8), None) == -1
    assert lib.fpt_simulate(C.byref(p), -1, 1, 1.0, C.c_void_p(8), None, C.c_void_p(8), None) == -1
    assert lib.fpt_simulate(C.byref(p), 10, 1, 0.0, C.c_void_p(8), None, C.c_void_p(8), None) == -1
    assert lib.fpt_simulate(C.byref(p), 10, 1, 1e300, C.c_void_p(8), None, C.c_void_p(8), None) == -1     # t_max/dt >= 2^53
    assert lib.fpt_simulate(C.byref(p), 10, 1, 1.0, None, None, C.c_void_p(8), None) == -1
    assert lib.fpt_simulate(C.byref(p), 10, 1, 1.0, C.c_void_p(8), None, None, None) == -1
    assert lib.fpt_simulate(C.byref(p), 0, 1, 1.0, C.c_void_p(8), None, C.c_void_p(8), None) == 0          # n_traj == 0: no-op
    h = lambda nb, lo, hi, cnt: lib.fpt_simulate_hist(C.byref(p), 10, 1, 1.0, C.c_void_p(8), None, C.c_void_p(8), 0, lo, hi,
                                                      nb, cnt, None)
    assert h(0, 0.0, 1.0, C.c_void_p(8)) == -1
    assert h(8193, 0.0, 1.0, C.c_void_p(8)) == -1
    assert h(10, 1.0, 1.0, C.c_void_p(8)) == -1
    assert h(10, 0.0, 1.0, None) == -1
    assert lib.fpt_histogram(None, None, 5, 0.0, 1.0, 4, C.c_void_p(8), None) == -1
    assert lib.fpt_histogram(C.c_void_p(8), None, 5, 1.0, 0.0, 4, C.c_void_p(8), None) == -1
    assert lib.fpt_histogram(C.c_void_p(8), None, 0, 0.0, 1.0, 4, C.c_void_p(8), None) == 0
    # fpt_simulate_ex: bad launch options / histogram request are rejected before any CUDA work
    ex = lambda opts=None, hist=None: lib.fpt_simulate_ex(C.byref(p), 10, 1, 1.0, C.c_void_p(8), None, C.c_void_p(8),
                                                          C.byref(hist) if hist else None, C.byref(opts) if opts else None, None, None)
    assert ex(fpt.FptLaunchOpts(block=48)) == -1
    assert ex(fpt.FptLaunchOpts(block=512)) == -1
    assert ex(fpt.FptLaunchOpts(schedule=2)) == -1
    assert ex(fpt.FptLaunchOpts(tail_helper=2)) == -1
    assert ex(fpt.FptLaunchOpts(specialise=-2)) == -1
    assert ex(fpt.FptLaunchOpts(consumers=5)) == -1
    assert ex(fpt.FptLaunchOpts(producers=4)) == -1
    assert ex(fpt.FptLaunchOpts(max_blocks=-1)) == -1
    assert ex(fpt.FptLaunchOpts(time_slice=2)) == -1 and ex(fpt.FptLaunchOpts(reserved=1)) == -1
    assert ex(None, fpt.FptHist(0, 0, 0.0, 1.0, 8)) == -1
    assert ex(None, fpt.FptHist(2, 10, 0.0, 1.0, 8)) == -1
    assert ex(None, fpt.FptHist(0, 10, 0.0, 1.0, None)) == -1
    assert lib.fpt_simulate_ex(C.byref(p), 0, 1, 1.0, None, None, None, None, None, None, None) == 0
    assert lib.fpt_set_specialise(2, 0, 0) == -1 and lib.fpt_set_specialise(0, 0, 0) == 0
    # fpt_simulate_noalloc: the fixed maximum and the argument checks come before any CUDA work
    na = lambda n, f=C.c_void_p(8), st=C.c_void_p(8), pp=C.byref(p): lib.fpt_simulate_noalloc(pp, n, 1, 1.0, f, None, st, None, None)
    assert na(binding.NOALLOC_MAX_TRAJ + 1) == -3 and na(1 << 40) == -3
    assert na(-1) == -1 and na(10, None) == -1 and na(10, C.c_void_p(8), None) == -1 and na(10, pp=None) == -1
    assert na(0, None, None) == 0
    header = (ROOT / "include" / "fpt.h").read_text()
    assert f"#define FPT_NOALLOC_MAX_TRAJ {binding.NOALLOC_MAX_TRAJ}\n" in header
    assert lib.fpt_dbg_set_slice_quantum(96) == -1 and lib.fpt_dbg_set_slice_quantum(64) == 0 and lib.fpt_dbg_set_slice_quantum(0) == 0
    assert lib.fpt_set_launch(48, 0, 0) == -1
    assert lib.fpt_set_launch(512, 0, 0) == -1
    assert lib.fpt_set_launch(128, 2, 0) == 0
    assert lib.fpt_set_launch(0, 0, 0) == 0


def test_no_cpu_fallback(lib):
    """Without a CUDA device a compute call fails loudly (FPT_E_CUDA); it never computes on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    p = fpt.make_params(**_good())
    buf = (C.c_double * 16)()
    st = (C.c_int32 * 16)()
    rc = lib.fpt_simulate(C.byref(p), 4, 1, 1.0, buf, None, st, None)
    assert rc == -2
    assert lib.fpt_strerror(rc) not in (b"ok", b"")
    rc = lib.fpt_simulate_host(C.byref(p), 4, 1, 1.0, buf, None, st, 0, 0.0, 1.0, 0, None)
    assert rc == -2


def test_product_does_not_import_oracle():
    for path in (ROOT / "paper_1802_05065_b200").rglob("*"):
        if path.suffix in (".py", ".cu", ".cuh", ".h"):
            text = path.read_text()
            assert "import oracle" not in text and "from oracle" not in text, path
            assert "fpt_oracle" not in text, path


def test_noalloc_entry_point_has_no_allocating_call_and_takes_its_scratch_address_from_the_symbol():
    """fpt_simulate_noalloc and its set-up (the last section of fpt_api.cu): no cudaMalloc / cudaFree / pool call, no use of
    device_ctx() (whose first call per device allocates), the scratch is one static __device__ __align__(256) array, and host
    code reaches it through cudaGetSymbolAddress only."""
    src = (ROOT / "paper_1802_05065_b200" / "csrc" / "fpt_api.cu").read_text()
    sec = src[src.index("// fpt_simulate_noalloc (fpt.h)"):]
    code = re.sub(r"//[^\n]*", "", re.sub(r"/\*.*?\*/", "", sec, flags=re.S))
    for banned in ("cudaMalloc", "cudaFree", "cudaMemPool", "device_ctx(", "WsGuard", "cudaHostAlloc", "cudaStreamCreate", "cudaEventCreate"):
        assert banned not in code, banned
    assert re.search(r"static __device__ __align__\(256\) unsigned char g_noalloc_scratch\[kNoAllocBytes\];", code)
    assert code.count("g_noalloc_scratch") == 2 and "cudaGetSymbolAddress(&ptr, g_noalloc_scratch)" in code
