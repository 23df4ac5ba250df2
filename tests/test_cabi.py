"""Host-side checks of the C-ABI library that need no GPU: it builds, loads, exports every symbol
include/fstat.h declares, validates arguments, and fails loudly (never falls back) without a device."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fs():
    from paper_2407_10797_b200 import build
    build.build()
    import paper_2407_10797_b200 as fs
    fs.load_library()
    return fs


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "fstat.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"FSTAT_API[^;(]*?\b(fstat_\w+)\s*\(", txt)))


def test_header_declares_the_boundary_calls():
    names = _declared_symbols()
    for must in ("fstat_plan_create", "fstat_eval_batch", "fstat_plan_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(fs):
    lib = C.CDLL(fs.library_path())
    names = _declared_symbols()
    assert sorted(fs.EXPORTED_SYMBOLS) == names
    for n in names:
        assert getattr(lib, n) is not None
    out = subprocess.run(["nm", "-D", "--defined-only", fs.library_path()], capture_output=True, text=True).stdout
    exported = sorted(set(re.findall(r" T (fstat_\w+)", out)))
    assert exported == names          # nothing else leaks out of the library under the fstat_ prefix


def test_library_is_sm100a_and_uses_tma_bulk_copy(fs):
    out = subprocess.run(["cuobjdump", "-lelf", fs.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", fs.library_path()], capture_output=True, text=True).stdout
    main = sass[sass.index("fstat_main_kernel"):]
    assert "UBLKCP" in main          # cp.async.bulk (TMA 1-D bulk copy) staging of the per-bin table
    assert "DFMA" in main
    fast = sass[sass.index("fstat_fast_kernel"):]
    fast = fast[:fast.index("Function :", 10)] if "Function :" in fast[10:] else fast
    assert "UBLKCP" in fast and "DFMA" in fast and "DADD" in fast


def test_default_options(fs):
    o = fs.fstat_default_options()
    assert o.f_ref_e0 == 0.01 and o.arm_length_m == 2.5e9
    assert o.orbit_kappa == 0.0 and o.orbit_lambda == 0.0
    assert o.device == -1 and o.inputs_on_device == 0 and o.max_segment_bins == 0
    assert o.force_level == -2 and o.interp_tol == 1.0 and o.tdi_channel == fs.TDI_CHANNELS["X"]


def test_status_strings(fs):
    assert [fs.fstat_status_str(i) for i in range(5)] == [fs.STATUS[i] for i in range(5)]


def test_edges_equal_bins(fs):
    import synthetic as syn
    for n, k in ((2096, 4), (1577880, 1024), (7100460, 16), (5, 5), (7, 1)):
        np.testing.assert_array_equal(fs.fstat_edges_equal_bins(n, k), syn.equal_bin_edges(n, k))
    with pytest.raises(fs.FstatError):
        fs.fstat_edges_equal_bins(3, 4)
    with pytest.raises(fs.FstatError):
        fs.fstat_edges_equal_bins(3, 0)


def test_plan_create_rejects_bad_arguments_before_touching_a_device(fs):
    f = np.arange(1, 9) * 1e-3
    dw = np.zeros(8, dtype=np.complex128)
    w = np.ones(8)
    for edges in ([0, 4, 4, 8], [1, 8], [0, 7], [0, 5, 3, 8]):
        with pytest.raises(fs.FstatError) as ei:
            fs.fstat_plan_create(f, dw, w, edges)
        assert ei.value.status == 1
    lib = fs.load_library()
    out = C.c_void_p(123)
    e = np.array([0, 8], dtype=np.int64)
    st = lib.fstat_plan_create(C.byref(out), 8, None, dw.ctypes.data, w.ctypes.data, 1,
                               e.ctypes.data_as(C.POINTER(C.c_int64)), None)
    assert st == 1 and out.value is None
    st = lib.fstat_plan_create(C.byref(out), 0, f.ctypes.data, dw.ctypes.data, w.ctypes.data, 1,
                               e.ctypes.data_as(C.POINTER(C.c_int64)), None)
    assert st == 1
    assert "n_bins" in fs.fstat_last_error(None)


def test_null_plan_calls_are_safe(fs):
    lib = fs.load_library()
    lib.fstat_plan_destroy(None)
    assert lib.fstat_plan_n_bins(None) == 0
    assert lib.fstat_plan_device(None) == -1
    assert lib.fstat_eval_batch(None, 1, None, None, None, None) == 1
    assert lib.fstat_plan_launch_count(None) == 0
    assert lib.fstat_plan_table_bytes(None) == 0
    assert lib.fstat_plan_band_stats(None, None) == 1
    assert lib.fstat_extrinsic_from_amplitudes(None, 0.0, None) == 1
    assert lib.fstat_amplitudes_from_extrinsic(1.0, 0.0, 0.0, 0.0, None) == 1
    # the rows built on top of the path (f2, f2 x f3, f4) answer FSTAT_EINVAL too
    assert lib.fstat_eval_batch_bands(None, 1, None, 4, 1, None, None, None, None) == 1
    assert lib.fstat_eval_batch_bands_host(None, 1, None, 4, 1, None, None, None, None) == 1
    assert lib.fstat_eval_amplitudes_bands(None, 1, None, 4, 1, None, None) == 1
    assert lib.fstat_eval_batch_channels(None, 2, 1, None, None, None, None) == 1
    import ctypes
    two_nulls = (ctypes.c_void_p * 2)(None, None)
    assert lib.fstat_eval_batch_channels(two_nulls, 2, 1, None, None, None, None) == 1


def test_no_cpu_fallback_without_a_device(fs):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    f = np.arange(1, 9) * 1e-3
    with pytest.raises(fs.FstatError) as ei:
        fs.fstat_plan_create(f, np.zeros(8, dtype=np.complex128), np.ones(8), [0, 8])
    assert ei.value.status == 3          # FSTAT_ECUDA: the product path refuses to run on the CPU
    with pytest.raises(fs.FstatError):
        fs.fstat_probe_pipe_peak(0)


def test_product_and_oracle_share_no_code():
    """The CUDA package never imports / includes anything of oracle/ and the oracle nothing of the package."""
    pkg = os.path.join(ROOT, "paper_2407_10797_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), fn
                assert "fstat_oracle" not in txt and "oracle/" not in txt.replace("shares nothing with oracle/", ""), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2407_10797_b200\b", txt, flags=re.M), fn
            assert '#include "../paper' not in txt and "fstat.h" not in txt, fn


def test_bench_fp64_instruction_model_matches_the_sass(fs):
    """bench.py's roofline counts FP64-pipe instructions per template-bin; the same numbers re-derived here
    from the SASS of the built library (tests/sass_util.py).  Per node interval / work item the constants are
    ncu-measured executed counts (profiles/r1_v6.md)."""
    import importlib.util
    import sass_util
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    fast = sass_util.fast_kernel_counts(fs.library_path())
    direct = sass_util.direct_kernel_counts(fs.library_path())
    # every variant of the per-bin loop (4-bin runs, tail) issues the same FP64 work per bin, +1/4 of the
    # Q <- Q C^4 update in the 4-bin runs
    assert bench.FAST_FP64_PER_BIN in fast["per_bin"]
    assert all(bench.FAST_FP64_PER_BIN - 1.0 <= v <= bench.FAST_FP64_PER_BIN for v in fast["per_bin"])
    # the direct kernel's loop body also holds the once-per-work-item choice of the basis constant c (a division,
    # ~20 FP64 instructions behind a branch): executed per bin = the static count minus that
    assert bench.DIRECT_FP64_PER_BIN <= direct["per_bin"] <= bench.DIRECT_FP64_PER_BIN + 24
    # the per-bin loop of the interpolating kernel is almost pure FP64: the pipe that bounds it
    assert bench.FAST_FP64_PER_BIN / fast["per_bin_all_pipes"] > 0.8
    # what bench.py itself reads from the SASS at run time (its constants are only the fallback)
    mix = bench.sass_fp64_mix(fs.library_path())
    assert mix is not None and mix["per_bin"] == bench.FAST_FP64_PER_BIN
    assert mix["dfma"] + mix["dadd"] + mix["dmul"] + mix["dsetp"] == pytest.approx(mix["per_bin"])
    assert mix["dfma"] >= 8.0 and mix["all_per_bin"] < 23.0
