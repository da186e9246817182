"""The C-ABI boundary without a GPU: libgamma_b200.so builds, loads and exports every symbol that
include/gamma_b200.h declares; argument errors are reported before anything touches the device; and
without a CUDA device a compute call fails loudly (there is no CPU fallback).  No compute happens here."""
import ctypes
import os
import re

import pytest
import torch

from paper_1012_1900_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gamma_b200.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gamma_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    return binding.load_library()


def test_library_is_built_in_tree_for_sm100a():
    path = build.build()
    assert os.path.dirname(path) == os.path.join(ROOT, "paper_1012_1900_b200")
    assert "arch=compute_100a,code=sm_100a" in " ".join(build.NVCC_FLAGS) and "-lineinfo" in build.NVCC_FLAGS


def test_every_declared_symbol_is_exported_and_bound(lib):
    names = declared_functions()
    assert "gamma_eval" in names and len(names) >= 10
    for n in names:
        assert hasattr(lib, n), f"{n} declared in gamma_b200.h but not exported"
    assert sorted(binding.exported_symbols) == names
    assert b"sm_100a" in lib.gamma_version()


def test_struct_layouts_match_the_compiled_library(lib):
    sizes = (ctypes.c_int * 4)()
    lib.gamma_abi_sizes(sizes)
    assert list(sizes) == [ctypes.sizeof(c) for c in (binding._COpts, binding._CSummary, binding._CCounters,
                                                      binding._CStageTimes)]
    assert sizes[1] == 48                       # stated in the header


def _call(lib, dims=(4, 4, 4), sp=(1.0, 1.0, 1.0), dd=0.03, dta=3.0, mode=0, cutoff=0.1, ref=1, ev=1, out=1):
    cd = (ctypes.c_int * 3)(*dims)
    cs = (ctypes.c_float * 3)(*sp)
    # fake non-null pointers: argument checks must reject before anything is dereferenced or launched
    return lib.gamma_eval(ctypes.c_void_p(0x1000 if ref else 0), ctypes.c_void_p(0x2000 if ev else 0), cd, cs,
                          dd, dta, mode, cutoff, ctypes.c_void_p(0x3000 if out else 0), None)


@pytest.mark.parametrize("kw,msg", [
    (dict(ref=0), "NULL"), (dict(out=0), "NULL"), (dict(dims=(0, 4, 4)), "dims"), (dict(dims=(1, 1, 1)), "axis"),
    (dict(sp=(1.0, -1.0, 1.0)), "spacing"), (dict(dd=0.0), "DD"), (dict(dta=0.0), "DTA"),
    (dict(dta=float("nan")), "DTA"), (dict(mode=2), "mode"), (dict(cutoff=1.0), "cutoff"),
    (dict(cutoff=-0.1), "cutoff"), (dict(dims=(2048, 2048, 1024)), "2^31"),
])
def test_argument_errors_are_reported_without_touching_the_device(lib, kw, msg):
    assert _call(lib, **kw) == 1                                      # GAMMA_ERR_INVALID_ARGUMENT
    assert msg in lib.gamma_last_error_string().decode()


def test_bad_options_and_aux_entry_points(lib):
    cd, cs = (ctypes.c_int * 3)(4, 4, 4), (ctypes.c_float * 3)(1, 1, 1)
    for bad in (dict(presort=5), dict(star_phase=-1), dict(lanes_per_voxel=4), dict(sort_key_bits=12),
                dict(table_cap=-5), dict(norm_dose=float("inf")), dict(graph=3), dict(table_radius=3), dict(interpolation=4)):
        o = binding.GammaOpts(**bad)._c()
        rc = lib.gamma_eval_ex(0x1000, 0x2000, cd, cs, 0.03, 3.0, 0, 0.1, ctypes.byref(o), 0x3000, None)
        assert rc == 1, bad
    assert lib.gamma_stats(0x1000, 10, 0, 4.0, 0x2000, 0x3000, None) == 1          # nbins
    assert lib.gamma_stats(0x1000, 10, 8, 0.0, 0x2000, 0x3000, None) == 1          # hist_max
    assert lib.gamma_sort_pairs(0x1000, 0x2000, 10, 4, 32, None) == 1              # begin_bit % 8
    assert lib.gamma_sort_pairs(None, None, 0, 0, 32, None) == 0                   # empty sort is a no-op
    assert lib.gamma_offset_table(cd, cs, 3.0, -1.0, 100, 0x1000, 0x2000, None) == 1
    assert lib.gamma_get_counters(None) == 1
    assert lib.gamma_launch_count() >= 0
    lib.gamma_release()


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_no_device_means_loud_failure_not_a_cpu_fallback(lib):
    assert _call(lib) == 3                                            # GAMMA_ERR_CUDA
    assert lib.gamma_last_error_string().decode() != ""
    with pytest.raises(binding.GammaError):
        binding.gamma_eval(torch.zeros(8), torch.zeros(8), (2, 2, 2), (1, 1, 1), 0.03, 3.0)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1012_1900_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower() or f == "phantoms.py", f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_1012_1900_b200" not in re.sub(r'""".*?"""|/\*.*?\*/', "", open(os.path.join(ROOT, "oracle", f)).read(), flags=re.S), f


def test_stats_options_are_refused_where_they_cannot_be_honoured(lib):
    """gamma_eval_batch / gamma_eval_host_batch / gamma_eval_general cannot write opts.stats_* (one pair of buffers for n
    cases; no fused statistics in the general kernels): INVALID_ARGUMENT, not silently unwritten buffers."""
    from paper_1012_1900_b200.binding import _COpts
    o = _COpts()
    o.stats_nbins, o.stats_hist, o.stats_summary, o.stats_hist_max = 16, 0x7000, 0x8000, 4.0
    one = (ctypes.c_void_p * 1)(0x1000)
    dims, sp = (ctypes.c_int * 3)(8, 8, 8), (ctypes.c_float * 3)(1.0, 1.0, 1.0)
    org = (ctypes.c_float * 3)(0.0, 0.0, 0.0)
    assert lib.gamma_eval_batch(1, one, one, dims, sp, 0.03, 3.0, 0, 0.1, ctypes.byref(o), one, None) == 1
    assert b"stats" in lib.gamma_last_error_string()
    assert lib.gamma_eval_host_batch(1, one, one, dims, sp, 0.03, 3.0, 0, 0.1, ctypes.byref(o), one, None) == 1
    assert b"stats" in lib.gamma_last_error_string()
    assert lib.gamma_eval_general(0x1000, dims, sp, org, 0x2000, dims, sp, org, 0.03, 3.0, 0, 0.1, ctypes.byref(o), 0x3000, None,
                                  None) == 1
    assert b"stats" in lib.gamma_last_error_string()
