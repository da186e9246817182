"""Thin ctypes binding of libgamma_b200.so: same names as include/gamma_b200.h, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device memory and
streams (``tensor.data_ptr()``, ``torch.cuda.current_stream().cuda_stream``).  There is no CPU fallback:
if the library cannot be loaded, or a call fails, a ``GammaError`` is raised.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

from . import build as _build

__all__ = [
    "GammaError", "GammaOpts", "load_library", "exported_symbols", "gamma_eval", "gamma_eval_ex",
    "gamma_eval_batch", "gamma_eval_general", "gamma_eval_host", "gamma_eval_host_batch", "gamma_stats", "gamma_stats_async", "decode_summary", "gamma_sort_pairs", "gamma_sort_pairs_noalloc", "gamma_offset_table", "gamma_get_counters",
    "gamma_get_stage_times", "gamma_launch_count", "gamma_workspace_bytes", "gamma_fp32_probe", "gamma_trace_reset", "gamma_trace_read", "gamma_trace_read_warps", "gamma_release", "gamma_version",
    "GAMMA_MODE_GLOBAL", "GAMMA_MODE_LOCAL",
]

GAMMA_MODE_GLOBAL, GAMMA_MODE_LOCAL = 0, 1

# every symbol include/gamma_b200.h declares
exported_symbols = (
    "gamma_eval", "gamma_eval_ex", "gamma_eval_batch", "gamma_eval_general", "gamma_eval_host", "gamma_eval_host_batch", "gamma_stats",
    "gamma_sort_pairs", "gamma_sort_pairs_noalloc", "gamma_offset_table", "gamma_get_counters", "gamma_get_stage_times", "gamma_launch_count", "gamma_workspace_bytes", "gamma_fp32_probe",
    "gamma_trace_reset", "gamma_trace_read", "gamma_trace_read_warps", "gamma_release", "gamma_abi_sizes", "gamma_last_error_string", "gamma_version",
)


class GammaError(RuntimeError):
    pass


class _COpts(ctypes.Structure):
    _fields_ = [("norm_dose", ctypes.c_float), ("presort", ctypes.c_int), ("star_phase", ctypes.c_int),
                ("lanes_per_voxel", ctypes.c_int), ("sort_key_bits", ctypes.c_int), ("table_cap", ctypes.c_longlong),
                ("profile_stages", ctypes.c_int), ("graph", ctypes.c_int), ("table_radius", ctypes.c_int),
                ("interpolation", ctypes.c_int), ("back_to_back", ctypes.c_int), ("star_load", ctypes.c_int), ("stats_nbins", ctypes.c_int),
                ("stats_hist", ctypes.c_void_p), ("stats_summary", ctypes.c_void_p), ("stats_hist_max", ctypes.c_float)]


class _CStageTimes(ctypes.Structure):
    _fields_ = [("prep_ms", ctypes.c_float), ("star_ms", ctypes.c_float), ("table_ms", ctypes.c_float),
                ("sort_ms", ctypes.c_float), ("search_ms", ctypes.c_float), ("total_ms", ctypes.c_float)]


class _CSummary(ctypes.Structure):
    _fields_ = [("n_eval", ctypes.c_ulonglong), ("n_pass", ctypes.c_ulonglong), ("sum_gamma", ctypes.c_double),
                ("sum_gamma3", ctypes.c_double), ("max_gamma", ctypes.c_float), ("n_nan", ctypes.c_uint),
                ("pad_", ctypes.c_ulonglong)]


class _CCounters(ctypes.Structure):
    _fields_ = [("n_voxels", ctypes.c_longlong), ("n_evaluated", ctypes.c_longlong),
                ("n_table_search", ctypes.c_longlong), ("table_entries", ctypes.c_longlong),
                ("vertex_visits", ctypes.c_longlong), ("max_key", ctypes.c_float), ("norm_dose", ctypes.c_float),
                ("table_truncated", ctypes.c_int), ("n_ring_search", ctypes.c_int), ("pipelined", ctypes.c_int),
                ("pad_", ctypes.c_int), ("calls_pipelined", ctypes.c_longlong)]


@dataclass
class GammaOpts:
    """Mirror of ``gamma_opts`` (include/gamma_b200.h); 0 means "library default"."""
    norm_dose: float = 0.0
    presort: int = 0          # 1 bucket presort, 2 no sort, 3 full LSD radix sort, 4 depth classes (default)
    star_phase: int = 0       # 1 on, 2 off
    lanes_per_voxel: int = 0  # 1, 8, 32
    sort_key_bits: int = 0    # presort=3: 8, 16, 24, 32
    table_cap: int = 0
    profile_stages: int = 0   # 1: record per-stage CUDA events (gamma_get_stage_times)
    interpolation: int = 0    # 1 Kuhn simplices (default), 2 grid vertices only (classical discrete gamma)
    table_radius: int = 0     # 1 data-independent prefix table (default), 2 the paper's radius max|DD|/dD
    graph: int = 0            # 1 replay a cached CUDA graph for repeated arguments, 2 plain launches (default)
    back_to_back: int = 0     # 1: caller asserts nothing else was enqueued on the stream since the previous call
    star_load: int = 0        # 1 compacted list + __ldg (default), 2 TMA-staged tiles, 3 tiles by cooperative loads
    stats_hist: object = None     # int64 CUDA tensor [nbins]: a6 fused into the call (with stats_summary)
    stats_summary: object = None  # uint8 CUDA tensor [48]: gamma_summary bytes, decode with decode_summary
    stats_hist_max: float = 0.0

    def __setattr__(self, name, value):
        # any field change drops the cached ctypes struct (argument marshalling only)
        self.__dict__[name] = value
        self.__dict__["_cached"] = None

    def _c(self):
        c = self.__dict__.get("_cached")
        if c is not None and self.stats_hist is not None and (
                c.stats_hist != self.stats_hist.data_ptr() or c.stats_nbins != self.stats_hist.numel()
                or c.stats_summary != self.stats_summary.data_ptr()):
            c = None                                   # the tensors were resized or moved in place
        if c is None:
            c = self._build()
            self.__dict__["_cached"] = c
        return c

    def _build(self):
        nb = int(self.stats_hist.numel()) if self.stats_hist is not None else 0
        if (self.stats_hist is None) != (self.stats_summary is None):
            raise GammaError("stats_hist and stats_summary must be given together")
        if self.stats_hist is not None:
            if not (self.stats_hist.is_cuda and self.stats_hist.dtype == torch.int64 and self.stats_hist.is_contiguous()):
                raise GammaError("stats_hist must be a contiguous int64 CUDA tensor")
            if not (self.stats_summary.is_cuda and self.stats_summary.is_contiguous()
                    and self.stats_summary.numel() * self.stats_summary.element_size() >= ctypes.sizeof(_CSummary)):
                raise GammaError("stats_summary must be a contiguous CUDA tensor of at least 48 bytes")
        return _COpts(float(self.norm_dose), int(self.presort), int(self.star_phase), int(self.lanes_per_voxel),
                      int(self.sort_key_bits), int(self.table_cap), int(self.profile_stages), int(self.graph),
                      int(self.table_radius), int(self.interpolation), int(self.back_to_back), int(self.star_load), nb,
                      self.stats_hist.data_ptr() if self.stats_hist is not None else None,
                      self.stats_summary.data_ptr() if self.stats_summary is not None else None,
                      float(self.stats_hist_max))


_lib = None


def load_library(build_if_needed: bool = True):
    """dlopen libgamma_b200.so (building it with nvcc first if missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if build_if_needed:
        path = _build.build()
    if not os.path.exists(path):
        raise GammaError(f"{path} is missing and there is no CPU fallback; run python -m paper_1012_1900_b200.build")
    lib = ctypes.CDLL(path)
    vp, ci, cf, cll = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_longlong
    i3, f3 = ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_float)
    lib.gamma_eval.argtypes = [vp, vp, i3, f3, cf, cf, ci, cf, vp, vp]
    lib.gamma_eval_ex.argtypes = [vp, vp, i3, f3, cf, cf, ci, cf, ctypes.POINTER(_COpts), vp, vp]
    lib.gamma_eval_batch.argtypes = [ci, vp, vp, vp, vp, cf, cf, ci, cf, ctypes.POINTER(_COpts), vp, vp]
    lib.gamma_eval_host.argtypes = [vp, vp, i3, f3, cf, cf, ci, cf, ctypes.POINTER(_COpts), vp, vp]
    lib.gamma_eval_host_batch.argtypes = [ci, vp, vp, vp, vp, cf, cf, ci, cf, ctypes.POINTER(_COpts), vp, vp]
    lib.gamma_eval_host_batch.restype = ci
    lib.gamma_eval_general.argtypes = [vp, i3, f3, f3, vp, i3, f3, f3, cf, cf, ci, cf, ctypes.POINTER(_COpts), vp, vp, vp]
    lib.gamma_eval_general.restype = ci
    lib.gamma_stats.argtypes = [vp, cll, ci, cf, vp, vp, vp]
    lib.gamma_sort_pairs.argtypes = [vp, vp, cll, ci, ci, vp]
    lib.gamma_sort_pairs_noalloc.argtypes = [vp, vp, cll, ci, ci, vp]
    lib.gamma_offset_table.argtypes = [i3, f3, cf, cf, cll, vp, vp, vp]
    lib.gamma_get_counters.argtypes = [ctypes.POINTER(_CCounters)]
    lib.gamma_fp32_probe.argtypes = [ci, ctypes.POINTER(ctypes.c_double), vp]
    lib.gamma_get_stage_times.argtypes = [ctypes.POINTER(_CStageTimes)]
    lib.gamma_launch_count.argtypes = []
    lib.gamma_launch_count.restype = cll
    lib.gamma_trace_reset.argtypes = []
    lib.gamma_trace_reset.restype = ci
    lib.gamma_trace_read.argtypes = [vp, ctypes.POINTER(cll)]
    lib.gamma_trace_read.restype = ci
    lib.gamma_trace_read_warps.argtypes = [vp, ci]
    lib.gamma_trace_read_warps.restype = ci
    lib.gamma_workspace_bytes.argtypes = []
    lib.gamma_workspace_bytes.restype = cll
    for name in ("gamma_eval", "gamma_eval_ex", "gamma_eval_batch", "gamma_eval_general", "gamma_eval_host", "gamma_eval_host_batch", "gamma_stats", "gamma_sort_pairs",
                 "gamma_sort_pairs_noalloc", "gamma_offset_table", "gamma_get_counters", "gamma_get_stage_times", "gamma_fp32_probe"):
        getattr(lib, name).restype = ci
    lib.gamma_release.restype = None
    lib.gamma_abi_sizes.restype = None
    lib.gamma_abi_sizes.argtypes = [ctypes.POINTER(ctypes.c_int)]
    sizes = (ctypes.c_int * 4)()
    lib.gamma_abi_sizes(sizes)
    mine = [ctypes.sizeof(c) for c in (_COpts, _CSummary, _CCounters, _CStageTimes)]
    if list(sizes) != mine:
        raise GammaError(f"struct layout mismatch between binding.py {mine} and libgamma_b200.so {list(sizes)}")
    lib.gamma_last_error_string.restype = ctypes.c_char_p
    lib.gamma_version.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _check(rc: int):
    if rc != 0:
        msg = load_library().gamma_last_error_string().decode()
        raise GammaError(f"libgamma_b200 error {rc}: {msg}")


def _stream(stream):
    if stream is None:
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _dev_f32(t: torch.Tensor, name: str) -> torch.Tensor:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise GammaError(f"{name} must be a contiguous float32 CUDA tensor")
    return t


_geom_cache = {}


def _geom(dims, spacing_mm):
    """(int[3], float[3]) ctypes arrays; the last few geometries are kept (argument marshalling only)."""
    key = (tuple(dims), tuple(spacing_mm))
    hit = _geom_cache.get(key)
    if hit is None:
        if len(_geom_cache) > 64:
            _geom_cache.clear()
        hit = ((ctypes.c_int * 3)(*[int(d) for d in dims]), (ctypes.c_float * 3)(*[float(s) for s in spacing_mm]))
        _geom_cache[key] = hit
    return hit


def _numel(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2])


def gamma_eval(ref, eval, dims, spacing_mm, DD, DTA_mm, mode=GAMMA_MODE_GLOBAL, low_dose_cutoff=0.1,
               out_gamma=None, stream=None):
    """``gamma_eval`` of include/gamma_b200.h.  Returns ``out_gamma`` (float32 CUDA tensor, N elements)."""
    return gamma_eval_ex(ref, eval, dims, spacing_mm, DD, DTA_mm, mode, low_dose_cutoff, None, out_gamma, stream,
                         _plain=True)


def gamma_eval_ex(ref, eval, dims, spacing_mm, DD, DTA_mm, mode=GAMMA_MODE_GLOBAL, low_dose_cutoff=0.1, opts=None,
                  out_gamma=None, stream=None, _plain=False):
    lib = load_library()
    ref, eval = _dev_f32(ref, "ref"), _dev_f32(eval, "eval")
    n = _numel(dims)
    if ref.numel() != n or eval.numel() != n:
        raise GammaError("ref / eval size does not match dims")
    if out_gamma is None:
        out_gamma = torch.empty(n, dtype=torch.float32, device=ref.device)
    _dev_f32(out_gamma, "out_gamma")
    if out_gamma.numel() != n:
        raise GammaError("out_gamma size does not match dims")
    cd, cs = _geom(dims, spacing_mm)
    if _plain:
        rc = lib.gamma_eval(ref.data_ptr(), eval.data_ptr(), cd, cs, float(DD), float(DTA_mm), int(mode),
                            float(low_dose_cutoff), out_gamma.data_ptr(), _stream(stream))
    else:
        co = opts._c() if opts is not None else None
        rc = lib.gamma_eval_ex(ref.data_ptr(), eval.data_ptr(), cd, cs, float(DD), float(DTA_mm), int(mode),
                               float(low_dose_cutoff), ctypes.byref(co) if co is not None else None,
                               out_gamma.data_ptr(), _stream(stream))
    _check(rc)
    return out_gamma


def gamma_eval_batch(refs, evals, dims_list, spacing_list, DD, DTA_mm, mode=GAMMA_MODE_GLOBAL, low_dose_cutoff=0.1,
                     opts=None, outs=None, stream=None):
    """``gamma_eval_batch``: independent cases (lists of CUDA float32 tensors with their dims / spacings) in one
    call; the cases overlap on the device.  Returns the list of gamma tensors; asynchronous."""
    lib = load_library()
    n = len(refs)
    if not (len(evals) == len(dims_list) == len(spacing_list) == n):
        raise ValueError("refs, evals, dims_list and spacing_list must have the same length")
    if outs is None:
        outs = [torch.empty(_numel(d), dtype=torch.float32, device=r.device) for r, d in zip(refs, dims_list)]
    for i in range(n):
        _dev_f32(refs[i], "ref")
        _dev_f32(evals[i], "eval")
        _dev_f32(outs[i], "out_gamma")
        if not (refs[i].numel() == evals[i].numel() == outs[i].numel() == _numel(dims_list[i])):
            raise ValueError(f"case {i}: ref / eval / out_gamma must have nx*ny*nz elements")
    ptr = ctypes.c_void_p * max(n, 1)
    pr = ptr(*[t.data_ptr() for t in refs])
    pe = ptr(*[t.data_ptr() for t in evals])
    po = ptr(*[t.data_ptr() for t in outs])
    cd = (ctypes.c_int * (3 * max(n, 1)))(*[int(x) for d in dims_list for x in d])
    cs = (ctypes.c_float * (3 * max(n, 1)))(*[float(x) for sp in spacing_list for x in sp])
    o = opts._c() if opts is not None else None
    _check(lib.gamma_eval_batch(n, pr, pe, cd, cs, float(DD), float(DTA_mm), int(mode), float(low_dose_cutoff),
                                ctypes.byref(o) if o is not None else None, po, _stream(stream)))
    return outs


def gamma_eval_general(ref, ref_dims, ref_spacing_mm, ref_origin_mm, eval, eval_dims, eval_spacing_mm, eval_origin_mm, DD,
                       DTA_mm, mode=GAMMA_MODE_GLOBAL, low_dose_cutoff=0.1, opts=None, out_gamma=None, want_closest=False,
                       out_closest=None, stream=None):
    """``gamma_eval_general``: evaluation dose on its own grid.  Returns gamma (float32 CUDA tensor, Nr elements), or
    (gamma, closest [Nr, 4] = x, y, z in mm and evaluation dose of the closest surface point) with ``want_closest``."""
    lib = load_library()
    ref, eval = _dev_f32(ref, "ref"), _dev_f32(eval, "eval")
    nr, ne = _numel(ref_dims), _numel(eval_dims)
    if ref.numel() != nr or eval.numel() != ne:
        raise GammaError("ref / eval size does not match its dims")
    if out_gamma is None:
        out_gamma = torch.empty(nr, dtype=torch.float32, device=ref.device)
    _dev_f32(out_gamma, "out_gamma")
    if want_closest and out_closest is None:
        out_closest = torch.empty((nr, 4), dtype=torch.float32, device=ref.device)
    if out_closest is not None:
        _dev_f32(out_closest, "out_closest")
        if out_closest.numel() != 4 * nr:
            raise GammaError("out_closest must hold Nr x 4 values")
    if out_gamma.numel() != nr:
        raise GammaError("out_gamma size does not match ref_dims")
    rd, rs = _geom(ref_dims, ref_spacing_mm)
    ed, es = _geom(eval_dims, eval_spacing_mm)
    ro = (ctypes.c_float * 3)(*[float(x) for x in ref_origin_mm])
    eo = (ctypes.c_float * 3)(*[float(x) for x in eval_origin_mm])
    co = opts._c() if opts is not None else None
    _check(lib.gamma_eval_general(ref.data_ptr(), rd, rs, ro, eval.data_ptr(), ed, es, eo, float(DD), float(DTA_mm), int(mode),
                                  float(low_dose_cutoff), ctypes.byref(co) if co is not None else None, out_gamma.data_ptr(),
                                  out_closest.data_ptr() if out_closest is not None else None, _stream(stream)))
    return (out_gamma, out_closest) if out_closest is not None else out_gamma


def gamma_eval_host(ref_host, eval_host, dims, spacing_mm, DD, DTA_mm, mode=GAMMA_MODE_GLOBAL, low_dose_cutoff=0.1,
                    opts=None, out_gamma_host=None, stream=None):
    """``gamma_eval_host``: CPU float32 tensors in (pinned for speed), CPU float32 tensor out; synchronises."""
    lib = load_library()
    n = _numel(dims)
    for t, name in ((ref_host, "ref_host"), (eval_host, "eval_host")):
        if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
                and t.numel() == n):
            raise GammaError(f"{name} must be a contiguous float32 CPU tensor with nx*ny*nz elements")
    if out_gamma_host is None:
        out_gamma_host = torch.empty(n, dtype=torch.float32).pin_memory()
    if out_gamma_host.is_cuda or out_gamma_host.dtype != torch.float32 or out_gamma_host.numel() != n:
        raise GammaError("out_gamma_host must be a float32 CPU tensor with nx*ny*nz elements")
    cd, cs = _geom(dims, spacing_mm)
    co = opts._c() if opts is not None else None
    rc = lib.gamma_eval_host(ref_host.data_ptr(), eval_host.data_ptr(), cd, cs, float(DD), float(DTA_mm), int(mode),
                             float(low_dose_cutoff), ctypes.byref(co) if co is not None else None,
                             out_gamma_host.data_ptr(), _stream(stream))
    _check(rc)
    return out_gamma_host


def gamma_eval_host_batch(refs_host, evals_host, dims_list, spacing_list, DD, DTA_mm, mode=GAMMA_MODE_GLOBAL,
                          low_dose_cutoff=0.1, opts=None, outs_host=None, stream=None):
    """``gamma_eval_host_batch``: lists of CPU float32 tensors in (pinned for speed), list of CPU float32 tensors out;
    copies and kernels of consecutive cases overlap; synchronises."""
    lib = load_library()
    n = len(refs_host)
    if not (len(evals_host) == len(dims_list) == len(spacing_list) == n):
        raise ValueError("refs_host, evals_host, dims_list and spacing_list must have the same length")
    if outs_host is None:
        outs_host = [torch.empty(_numel(d), dtype=torch.float32).pin_memory() for d in dims_list]
    for i in range(n):
        for t, name in ((refs_host[i], "ref_host"), (evals_host[i], "eval_host"), (outs_host[i], "out_gamma_host")):
            if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
                    and t.numel() == _numel(dims_list[i])):
                raise GammaError(f"case {i}: {name} must be a contiguous float32 CPU tensor with nx*ny*nz elements")
    ptr = ctypes.c_void_p * max(n, 1)
    pr = ptr(*[t.data_ptr() for t in refs_host])
    pe = ptr(*[t.data_ptr() for t in evals_host])
    po = ptr(*[t.data_ptr() for t in outs_host])
    cd = (ctypes.c_int * (3 * max(n, 1)))(*[int(x) for d in dims_list for x in d])
    cs = (ctypes.c_float * (3 * max(n, 1)))(*[float(x) for sp in spacing_list for x in sp])
    o = opts._c() if opts is not None else None
    _check(lib.gamma_eval_host_batch(n, pr, pe, cd, cs, float(DD), float(DTA_mm), int(mode), float(low_dose_cutoff),
                                     ctypes.byref(o) if o is not None else None, po, _stream(stream)))
    return outs_host


def gamma_stats_async(gamma, nbins=64, hist_max=4.0, hist=None, summary_buf=None, stream=None):
    """``gamma_stats`` without reading anything back: enqueues a6 and returns (hist int64 CUDA tensor [nbins],
    summary bytes CUDA tensor) -- decode the latter with ``decode_summary`` (which synchronises)."""
    lib = load_library()
    _dev_f32(gamma, "gamma")
    if hist is None:
        hist = torch.empty(int(nbins), dtype=torch.int64, device=gamma.device)
    if summary_buf is None:
        summary_buf = torch.empty(ctypes.sizeof(_CSummary), dtype=torch.uint8, device=gamma.device)
    _check(lib.gamma_stats(gamma.data_ptr(), gamma.numel(), int(nbins), float(hist_max), hist.data_ptr(),
                           summary_buf.data_ptr(), _stream(stream)))
    return hist, summary_buf


def decode_summary(summary_buf) -> dict:
    s = _CSummary.from_buffer_copy(bytes(summary_buf.cpu().numpy().tobytes()))
    return {"n_eval": s.n_eval, "n_pass": s.n_pass, "sum_gamma": s.sum_gamma, "sum_gamma3": s.sum_gamma3,
            "max_gamma": s.max_gamma, "n_nan": s.n_nan}


def gamma_stats(gamma, nbins=64, hist_max=4.0, stream=None):
    """``gamma_stats``: returns (hist int64 CUDA tensor [nbins], summary dict) -- reading the dict synchronises."""
    hist, buf = gamma_stats_async(gamma, nbins, hist_max, stream=stream)
    return hist, decode_summary(buf)


def gamma_sort_pairs(keys, vals, begin_bit=0, end_bit=32, stream=None):
    """``gamma_sort_pairs``: in-place stable sort of int32/uint32-typed CUDA tensors (bit patterns)."""
    lib = load_library()
    for t in (keys, vals):
        if not (t.is_cuda and t.is_contiguous() and t.element_size() == 4):
            raise GammaError("keys / vals must be contiguous 4-byte CUDA tensors")
    if keys.numel() != vals.numel():
        raise GammaError("keys and vals differ in length")
    _check(lib.gamma_sort_pairs(keys.data_ptr(), vals.data_ptr(), keys.numel(), int(begin_bit), int(end_bit),
                                _stream(stream)))
    return keys, vals


SORT_NOALLOC_MAX_PAIRS = 1 << 20      # GAMMA_SORT_NOALLOC_MAX_PAIRS of include/gamma_b200.h


def gamma_sort_pairs_noalloc(keys, vals, begin_bit=0, end_bit=32, stream=None):
    """``gamma_sort_pairs_noalloc``: ``gamma_sort_pairs`` without any device allocation by the library.

    For code that must not call cudaMalloc -- it runs beside a global-mode stream capture, inside a latency-bound loop,
    or in a process whose device memory belongs to one pool.  The sort's scratch is an array built into the library
    (about 8.3 MB of every GPU that loads it), which limits it to ``SORT_NOALLOC_MAX_PAIRS`` pairs: a longer input raises
    ``GammaError`` and nothing runs.  All calls on a device share that array, so calls that could overlap on the GPU
    (different streams with no event between them) race; calls on one stream are safe.  Make the first call on a device
    outside stream capture (it looks up the array's device address).  Same result as ``gamma_sort_pairs``, bit for bit.
    """
    lib = load_library()
    for t in (keys, vals):
        if not (t.is_cuda and t.is_contiguous() and t.element_size() == 4):
            raise GammaError("keys / vals must be contiguous 4-byte CUDA tensors")
    if keys.numel() != vals.numel():
        raise GammaError("keys and vals differ in length")
    _check(lib.gamma_sort_pairs_noalloc(keys.data_ptr(), vals.data_ptr(), keys.numel(), int(begin_bit), int(end_bit),
                                        _stream(stream)))
    return keys, vals


def gamma_offset_table(dims, spacing_mm, DTA_mm, radius, max_entries=1 << 20, device="cuda", stream=None):
    """``gamma_offset_table``: returns (entries int32 [count, 4], truncated flag, covered radius^2)."""
    lib = load_library()
    ent = torch.empty((int(max_entries), 4), dtype=torch.int32, device=device)
    cnt = torch.zeros(3, dtype=torch.int32, device=device)
    cd, cs = _geom(dims, spacing_mm)
    _check(lib.gamma_offset_table(cd, cs, float(DTA_mm), float(radius), int(max_entries), ent.data_ptr(),
                                  cnt.data_ptr(), _stream(stream)))
    c = cnt.cpu()
    r2 = c[2:3].view(torch.float32).item()
    return ent[: int(c[0])], bool(c[1]), r2


def gamma_get_counters() -> dict:
    lib = load_library()
    c = _CCounters()
    _check(lib.gamma_get_counters(ctypes.byref(c)))
    return {k: getattr(c, k) for k, _ in _CCounters._fields_ if k != "pad_"}


def gamma_get_stage_times() -> dict:
    lib = load_library()
    t = _CStageTimes()
    _check(lib.gamma_get_stage_times(ctypes.byref(t)))
    return {k: getattr(t, k) for k, _ in _CStageTimes._fields_}


def gamma_launch_count() -> int:
    return int(load_library().gamma_launch_count())


def gamma_trace_reset():
    """Clear the device timeline and switch the stamps on (library built with -DGAMMA_TRACE only)."""
    _check(load_library().gamma_trace_reset())


def gamma_trace_read():
    """(records uint64 numpy [256, 4, 4] = call x kernel x (first, waited, last, 0) in ns, number of the next call)."""
    import numpy as np
    buf = np.zeros((256, 4, 4), dtype=np.uint64)
    nxt = ctypes.c_longlong(0)
    _check(load_library().gamma_trace_read(buf.ctypes.data_as(ctypes.c_void_p), ctypes.byref(nxt)))
    return buf, int(nxt.value)


def gamma_trace_read_warps(max_warps=8192):
    """uint64 numpy [max_warps, 8] = warp x (started, wait passed, first unit finished, ended, units taken, 0, 0, 0) of
    the last k_table_search launch, ns (library built with -DGAMMA_TRACE only)."""
    import numpy as np
    buf = np.zeros((int(max_warps), 8), dtype=np.uint64)
    _check(load_library().gamma_trace_read_warps(buf.ctypes.data_as(ctypes.c_void_p), int(max_warps)))
    return buf


def gamma_workspace_bytes() -> int:
    return int(load_library().gamma_workspace_bytes())


def gamma_fp32_probe(repeats=5, stream=None) -> float:
    lib = load_library()
    v = ctypes.c_double(0.0)
    _check(lib.gamma_fp32_probe(int(repeats), ctypes.byref(v), _stream(stream)))
    return v.value


def gamma_release():
    load_library().gamma_release()


def gamma_version() -> str:
    return load_library().gamma_version().decode()
