#!/usr/bin/env python3
"""bench_suite.py -- the per-config measurements SURVEY.md section 8(d) lists, beside bench.py's headline line.

    python bench_suite.py [--suite configs|criteria|all] [--reps 30] [--oracle-seconds 8] [--md out.md]

configs   every BASELINE.json config (cfg1, cfg2, cfg3, cfg4 coarse/fine, cfg5): grid voxels N, evaluated voxels M,
          ms per case (t_total), stage times t_p / t_gamma, M/t_gamma, N/t_total, sum gamma^3, pass rate,
          the resolution exponent of cfg4 (Fig. 2) and cfg5 with the voxel pre-sort on / off and
          with the paper's thread-per-voxel mapping (Table 2)
batch     independent cfg3 cases per call through gamma_eval_batch against the same cases one by one
sort      subsystem (3) stand-alone: gamma_sort_pairs on 2^20 / 2^24 (key, value) pairs, 16 and 32 key bits, GB/s against
          the algorithmic 20 B per pair per 8-bit pass and the measured HBM copy rate
general   gamma_eval_general on the cfg3 reference against a 2 mm evaluation grid: ms per case, with / without closest point
trace     device timeline of consecutive calls (library built with -DGAMMA_TRACE: GAMMA_NVCC_EXTRA=-DGAMMA_TRACE python -m
          paper_1012_1900_b200.build --force): when each kernel of a call starts, passes its dependency wait and ends,
          relative to the call's first kernel, one call after the other with and without opts.back_to_back
criteria  the 9 DD x DTA combinations of Table 3 on the cfg3 phantom: time against sum gamma^3
          (Fig. 1) and the exact law gamma(k DD, k DTA) = gamma(DD, DTA) / k checked on the device maps

Timing: one gamma_eval per repetition on device-resident inputs, rotating input/output sets larger than L2, CUDA
events per repetition, median.  The CPU oracle is timed on a bounded seeded sample of each workload (--oracle-seconds
of host time per config; 0 skips it).  One JSON line per measurement on stdout; --md also writes a table.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

L2_BYTES = 126e6


def f32(x):
    return float(np.float32(x))


def measure(case, opts_kw, reps, dd=None, dta=None, keep_map=False, mode=None):
    import torch
    from paper_1012_1900_b200 import binding
    from paper_1012_1900_b200.binding import GammaOpts

    dd = case.dd if dd is None else dd
    dta = case.dta_mm if dta is None else dta
    dev = torch.device("cuda", 0)
    N = case.ref.size
    nsets = max(2, min(24, int(np.ceil(2.0 * L2_BYTES / (12.0 * N))) + 1))
    ref_h = torch.from_numpy(case.ref.ravel().copy())
    ev_h = torch.from_numpy(case.eval.ravel().copy())
    refs = [ref_h.to(dev) for _ in range(nsets)]
    evs = [ev_h.to(dev) for _ in range(nsets)]
    outs = [torch.empty(N, dtype=torch.float32, device=dev) for _ in range(nsets)]
    stream = torch.cuda.current_stream()
    a = (case.dims, case.spacing_mm, dd, dta, case.mode if mode is None else mode, case.cutoff)
    opts = GammaOpts(**opts_kw)
    popts = GammaOpts(profile_stages=1, **opts_kw)
    for i in range(4):
        binding.gamma_eval_ex(refs[i % nsets], evs[i % nsets], *a, opts, outs[i % nsets], stream)
    torch.cuda.synchronize()
    times = []
    for i in range(reps):
        k = i % nsets
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        binding.gamma_eval_ex(refs[k], evs[k], *a, opts, outs[k], stream)
        e1.record(stream)
        e1.synchronize()
        times.append(e0.elapsed_time(e1))
    # back-to-back rate (what bench.py reports): consecutive calls pipelined (opts.back_to_back: nothing else is
    # enqueued on the stream between them)
    torch.cuda.synchronize()
    bopts = GammaOpts(back_to_back=1, **opts_kw)
    for i in range(12):                       # every lane has seen this geometry: workspaces allocated, graphs built
        binding.gamma_eval_ex(refs[i % nsets], evs[i % nsets], *a, bopts, outs[i % nsets], stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(reps):
        k = i % nsets
        binding.gamma_eval_ex(refs[k], evs[k], *a, bopts, outs[k], stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_stream = e0.elapsed_time(e1) / reps
    cnt = binding.gamma_get_counters()
    acc = {}
    for i in range(min(reps, 20)):
        k = i % nsets
        binding.gamma_eval_ex(refs[k], evs[k], *a, popts, outs[k], stream)
        for kk, v in binding.gamma_get_stage_times().items():
            acc.setdefault(kk, []).append(v)
    stages = {k: float(np.median(v)) for k, v in acc.items()}
    hist, summ = binding.gamma_stats(outs[0], 64, 4.0)
    torch.cuda.synchronize()
    res = {"N": N, "M": int(cnt["n_evaluated"]), "ms_case_median": float(np.median(times)),
           "ms_case_min": float(np.min(times)), "ms_case_back_to_back": ms_stream, "stages_ms": stages,
           "n_table_search": int(cnt["n_table_search"]), "vertex_visits": int(cnt["vertex_visits"]),
           "table_entries": int(cnt["table_entries"]), "max_key": float(cnt["max_key"]),
           "sum_gamma3": float(summ["sum_gamma3"]), "pass_rate": summ["n_pass"] / max(1, summ["n_eval"]),
           "max_gamma": float(summ["max_gamma"]), "options": opts_kw, "criteria": f"{dd * 100:g}%/{dta:g}mm"}
    t_gamma = stages.get("star_ms", 0.0) + stages.get("search_ms", 0.0)
    res["t_gamma_ms"] = t_gamma
    res["t_p_ms"] = max(0.0, stages.get("total_ms", 0.0) - t_gamma)
    res["evaluated_voxels_per_s"] = res["M"] / (ms_stream * 1e-3)
    res["grid_voxels_per_s"] = N / (ms_stream * 1e-3)
    if keep_map:
        res["_map"] = outs[0].clone()
    del refs, evs, outs
    torch.cuda.empty_cache()
    return res


def oracle_sample(case, seconds, dd=None, dta=None, nthreads=0):
    """The oracle as it stands on a bounded seeded sample of the evaluated voxels (all host cores, or `nthreads`)."""
    if seconds <= 0:
        return None
    import oracle
    oracle.build()
    dd = case.dd if dd is None else dd
    dta = case.dta_mm if dta is None else dta
    ref = case.ref.ravel().astype(np.float64)
    keep = np.flatnonzero(ref >= f32(case.cutoff) * ref.max())
    rng = np.random.default_rng([0, 77])
    sp = [f32(s) for s in case.spacing_mm]

    def run(vox):
        t0 = time.perf_counter()
        # explicit thread count: the oracle keeps the last OpenMP setting, and a one-core run may have come before
        oracle.gamma(case.ref, case.eval, case.dims, sp, f32(dd), f32(dta), case.mode, f32(case.cutoff), voxels=vox,
                     nthreads=nthreads if nthreads else (os.cpu_count() or 1))
        return time.perf_counter() - t0

    probe = np.sort(rng.choice(keep, size=min(keep.size, 2000), replace=False))
    tp = run(probe)
    n = int(min(keep.size, max(probe.size, seconds / (tp / probe.size))))
    vox = np.sort(rng.choice(keep, size=n, replace=False))
    t = run(vox)
    return {"voxels": n, "of": int(keep.size), "seconds": t, "voxels_per_s": n / t,
            "cores": nthreads if nthreads else (os.cpu_count() or 1),
            "seconds_per_case_extrapolated": t / n * keep.size}


def suite_configs(args, emit):
    from paper_1012_1900_b200 import phantoms
    rows = []
    for name in ("cfg1", "cfg2", "cfg3", "cfg4_coarse", "cfg4_fine", "cfg5"):
        case = phantoms.make_case(name)
        variants = [("default", {})]
        if name == "cfg3":       # kernel variants of SURVEY.md 8(f) 2: the paper's routine on whole cells; grid vertices only
            variants += [("graph replay (opts.graph = 1)", {"graph": 1}),
                         ("recursion variant (PAPER.md:209)", {"interpolation": 3}),
                         ("vertices only (no interpolation)", {"interpolation": 2})]
        if name == "cfg5":
            variants += [("presort off", {"presort": 2}), ("full radix sort", {"presort": 3}),
                         ("thread per voxel, presort on", {"lanes_per_voxel": 1, "star_phase": 2, "presort": 3}),
                         ("thread per voxel, presort off", {"lanes_per_voxel": 1, "star_phase": 2, "presort": 2})]
        orc = oracle_sample(case, args.oracle_seconds)
        if name in ("cfg1", "cfg2") and orc is not None:     # per-core figure; the paper's CPU threading is unstated
            orc["one_core"] = oracle_sample(case, args.oracle_seconds, nthreads=1)
        if name in ("cfg3", "cfg5"):     # the local criterion (dD_v = DD * D_r[v], reading 9): a reciprocal per voxel in double
            variants.append(("local criterion (mode 1)", {}))
        for label, kw in variants:
            reps = args.reps if "thread per voxel" not in label else max(3, args.reps // 6)
            r = measure(case, kw, reps, mode=1 if label.startswith("local criterion") else None)
            r.update({"suite": "configs", "case": name, "variant": label, "cpu_oracle": orc if label == "default" else None})
            emit(r)
            rows.append(r)
    fine = next(r for r in rows if r["case"] == "cfg4_fine")
    mid = next(r for r in rows if r["case"] == "cfg2")
    coarse = next(r for r in rows if r["case"] == "cfg4_coarse")
    xs = np.log([coarse["N"], mid["N"], fine["N"]])
    ys = np.log([coarse["ms_case_median"], mid["ms_case_median"], fine["ms_case_median"]])
    yg = np.log([coarse["t_gamma_ms"], mid["t_gamma_ms"], fine["t_gamma_ms"]])
    emit({"suite": "configs", "resolution_exponent_t_total": float(np.polyfit(xs, ys, 1)[0]),
          "resolution_exponent_t_gamma": float(np.polyfit(xs, yg, 1)[0]),
          "paper": "T_gamma^C ~ N^1.90, T_gamma^G ~ N^1.68 (PAPER.md:382-388); same phantom at 5 / 2.5 / 1.25 mm"})
    return rows


def suite_batch(args, emit):
    """independent cases per call (gamma_eval_batch) against the same cases one by one."""
    import torch
    from paper_1012_1900_b200 import binding, phantoms
    case = phantoms.make_case("cfg3")
    dev = torch.device("cuda", 0)
    N = case.ref.size
    for nb in (4, 16, 32):
        refs = [torch.from_numpy(case.ref.ravel().copy()).to(dev) for _ in range(nb)]
        evs = [torch.from_numpy(case.eval.ravel().copy()).to(dev) for _ in range(nb)]
        outs = [torch.empty(N, dtype=torch.float32, device=dev) for _ in range(nb)]
        dims, sps = [case.dims] * nb, [case.spacing_mm] * nb
        a = (case.dd, case.dta_mm, case.mode, case.cutoff)
        stream = torch.cuda.current_stream()
        res = {}
        gopts = binding.GammaOpts(graph=1)
        for label, fn in (("batch", lambda: binding.gamma_eval_batch(refs, evs, dims, sps, *a, None, outs, stream)),
                          ("batch, graph replay", lambda: binding.gamma_eval_batch(refs, evs, dims, sps, *a, gopts, outs,
                                                                                   stream)),
                          ("one by one", lambda: [binding.gamma_eval_ex(refs[i], evs[i], case.dims, case.spacing_mm, *a,
                                                                        binding.GammaOpts(back_to_back=1), outs[i], stream)
                                                  for i in range(nb)])):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            reps = max(5, args.reps // 2)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                fn()
            e1.record(stream)
            torch.cuda.synchronize()
            res[label] = e0.elapsed_time(e1) / reps / nb
        cnt_m = int((~torch.isnan(outs[0])).sum().item())
        emit({"suite": "batch", "case": "cfg3", "cases_per_call": nb, "working_set_MB": nb * 12 * N / 1e6,
              "ms_per_case_batch": res["batch"], "ms_per_case_batch_graph_replay": res["batch, graph replay"],
              "ms_per_case_one_by_one": res["one by one"],
              "evaluated_voxels_per_s_batch": cnt_m / (res["batch"] * 1e-3), "speedup": res["one by one"] / res["batch"]})
        del refs, evs, outs
        torch.cuda.empty_cache()


def suite_criteria(args, emit):
    import torch
    from paper_1012_1900_b200 import phantoms
    case = phantoms.make_case("cfg3")
    rows, maps = [], {}
    for dd in (0.01, 0.02, 0.03):
        for dta in (1.0, 2.0, 3.0):
            r = measure(case, {}, args.reps, dd=dd, dta=dta, keep_map=True)
            maps[(dd, dta)] = r.pop("_map")
            r.update({"suite": "criteria", "case": "cfg3 phantom", "variant": f"{dd * 100:g}%/{dta:g}mm"})
            emit(r)
            rows.append(r)
    # gamma(k DD, k DTA) = gamma(DD, DTA) / k: exact in real arithmetic
    base = maps[(0.01, 1.0)]
    m = ~torch.isnan(base)
    law = {}
    for k in (2, 3):
        other = maps[(0.01 * k, 1.0 * k)]
        assert bool((torch.isnan(other) == ~m).all())
        law[f"k={k}"] = float((other[m] * k - base[m]).abs().max().item())
    mono_dd = all(bool((maps[(0.02, t)][m] <= maps[(0.01, t)][m] + 1e-5).all()) for t in (1.0, 2.0, 3.0))
    mono_dta = all(bool((maps[(d, 2.0)][m] <= maps[(d, 1.0)][m] + 1e-5).all()) for d in (0.01, 0.02, 0.03))
    t = np.array([r["t_gamma_ms"] for r in rows])
    s3 = np.array([r["sum_gamma3"] for r in rows])
    emit({"suite": "criteria", "scaling_law_max_abs_dev": law, "monotone_in_DD": mono_dd, "monotone_in_DTA": mono_dta,
          "corr_t_gamma_vs_sum_gamma3": float(np.corrcoef(t, s3)[0, 1]),
          "corr_log_t_gamma_vs_log_sum_gamma3": float(np.corrcoef(np.log(t), np.log(s3))[0, 1])})
    return rows


def suite_sort(args, emit):
    """Hand-written LSD radix sort (csrc/radix_sort.cuh): per 8-bit pass it reads the keys twice and the values once and
    writes both (20 B per pair); an odd number of passes costs one more copy back (16 B per pair)."""
    import torch
    from paper_1012_1900_b200 import binding
    hbm = 6551.4
    try:
        hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:  # noqa: BLE001
        pass
    stream = torch.cuda.current_stream()
    for n in (1 << 20, 1 << 24):
        rng = np.random.default_rng([n, 3])
        keys0 = torch.from_numpy(np.abs(rng.normal(0, 3, size=n)).astype(np.float32).view(np.int32)).cuda()
        vals0 = torch.arange(n, dtype=torch.int32, device="cuda")
        for bits in ((16, 32), (0, 32)):
            passes = (bits[1] - bits[0]) // 8
            k, v = keys0.clone(), vals0.clone()
            binding.gamma_sort_pairs(k, v, *bits)
            torch.cuda.synchronize()
            ok = bool((k[1:].view(torch.int32) >> bits[0] >= k[:-1].view(torch.int32) >> bits[0]).all())
            times = []
            for _ in range(max(5, args.reps // 3)):
                k.copy_(keys0); v.copy_(vals0)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                binding.gamma_sort_pairs(k, v, *bits)
                e1.record(stream)
                e1.synchronize()
                times.append(e0.elapsed_time(e1))
            ms = float(np.median(times))
            alg = passes * 20.0 * n
            emit({"suite": "sort", "pairs": n, "key_bits": bits[1] - bits[0], "passes": passes, "ms": ms, "sorted": ok,
                  "pairs_per_s": n / (ms * 1e-3), "algorithmic_GBs": alg / (ms * 1e-3) / 1e9,
                  "frac_of_hbm_copy_peak": alg / (ms * 1e-3) / 1e9 / hbm, "hbm_peak_GBs": hbm})


def suite_general(args, emit):
    import torch
    from paper_1012_1900_b200 import binding, phantoms
    c = phantoms.make_general_case("cfg3_general")
    r = torch.from_numpy(c.ref.ravel().copy()).cuda()
    e = torch.from_numpy(c.eval.ravel().copy()).cuda()
    a = (c.ref_dims, c.ref_spacing_mm, c.ref_origin_mm)
    b = (c.eval_dims, c.eval_spacing_mm, c.eval_origin_mm, c.dd, c.dta_mm, c.mode, c.cutoff)
    stream = torch.cuda.current_stream()
    out = torch.empty(r.numel(), device="cuda")
    clo = torch.empty((r.numel(), 4), device="cuda")
    res = {}
    for label, oc in (("gamma only", None), ("gamma + closest point", clo)):
        for _ in range(3):
            binding.gamma_eval_general(r, *a, e, *b, None, out, False, oc, stream)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.reps):
            binding.gamma_eval_general(r, *a, e, *b, None, out, False, oc, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        res[label] = e0.elapsed_time(e1) / args.reps
    m = int((~torch.isnan(out)).sum().item())
    emit({"suite": "general", "case": "cfg3_general: cfg3 reference (128x128x64 at 2.5 mm) against a 160x160x80 evaluation grid "
          "at 2 mm, fractional origin offset", "M": m, "ms_per_case": res,
          "evaluated_voxels_per_s": m / (res["gamma only"] * 1e-3)})


def suite_trace(args, emit):
    """Where the time of a call goes: %globaltimer stamps of every kernel (first thread in, dependency wait passed,
    last block out), median over the calls of a back-to-back run; needs a -DGAMMA_TRACE build of the library."""
    import torch
    from paper_1012_1900_b200 import binding, phantoms
    from paper_1012_1900_b200.binding import GammaOpts
    case = phantoms.make_case(args.trace_case)
    dev = torch.device("cuda", 0)
    N = case.ref.size
    nsets = max(2, min(24, int(np.ceil(2.0 * L2_BYTES / (12.0 * N))) + 1))
    refs = [torch.from_numpy(case.ref.ravel().copy()).to(dev) for _ in range(nsets)]
    evs = [torch.from_numpy(case.eval.ravel().copy()).to(dev) for _ in range(nsets)]
    outs = [torch.empty(N, dtype=torch.float32, device=dev) for _ in range(nsets)]
    a = (case.dims, case.spacing_mm, case.dd, case.dta_mm, case.mode, case.cutoff)
    stream = torch.cuda.current_stream()
    names = ("k_norm", "k_classify", "k_star", "k_table_search")
    for label, opts in (("back_to_back", GammaOpts(back_to_back=1)), ("serial (default)", GammaOpts())):
        for i in range(8):
            binding.gamma_eval_ex(refs[i % nsets], evs[i % nsets], *a, opts, outs[i % nsets], stream)
        torch.cuda.synchronize()
        binding.gamma_trace_reset()
        _, first_call = binding.gamma_trace_read()
        ncalls = 120
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(ncalls):
            binding.gamma_eval_ex(refs[i % nsets], evs[i % nsets], *a, opts, outs[i % nsets], stream)
        e1.record(stream)
        torch.cuda.synchronize()
        rec, nxt = binding.gamma_trace_read()
        assert nxt - first_call == ncalls
        idx = [(first_call + i) % 256 for i in range(20, ncalls)]          # steady state
        t = rec[idx].astype(np.float64)                                      # [call, kernel, (first, waited, last, 0)]
        origin = t[:, 0, 0][:, None, None]
        rel = (t[:, :, :3] - origin) / 1e3                                   # us after the call's k_norm started
        med = np.median(rel, axis=0)
        period = np.median(np.diff(t[:, 0, 0])) / 1e3
        prev_search_end = np.median((t[:-1, 3, 2] - t[1:, 0, 0]) / 1e3)      # previous call's search end after this norm start
        # eight consecutive calls as they were: [first thread in, last block passed its wait, last block out] per kernel,
        # us after the first of them started -- shows which kernels of which calls are on the device together
        w0 = 40
        raw = (t[w0:w0 + 8, :, :3] - t[w0, 0, 0]) / 1e3
        emit({"suite": "trace", "case": args.trace_case, "mode": label, "ms_per_case_events": e0.elapsed_time(e1) / ncalls,
              "consecutive_calls_us": [{n: [round(float(v), 1) for v in raw[c, k]] for k, n in enumerate(names)}
                                       for c in range(raw.shape[0])],
              "period_us": float(period), "previous_search_ends_after_this_norm_starts_us": float(prev_search_end),
              "kernels_us_after_norm_start": {n: {"first": float(med[k, 0]), "waited": float(med[k, 1]),
                                                 "last": float(med[k, 2])} for k, n in enumerate(names)},
              "pipelined_calls": binding.gamma_get_counters()["calls_pipelined"]})
    # the warps of one k_table_search launch (a call on its own, full-size grid): how long a work unit takes
    torch.cuda.synchronize()
    binding.gamma_eval_ex(refs[0], evs[0], *a, GammaOpts(), outs[0], stream)
    torch.cuda.synchronize()
    w = binding.gamma_trace_read_warps().astype(np.float64)
    w = w[w[:, 3] > 0]
    if len(w):
        t0 = w[:, 0].min()
        pct = lambda x: [round(float(v), 2) for v in np.percentile(x, [0, 10, 50, 90, 100])]
        units = w[:, 4]
        busy = (w[:, 3] - w[:, 1]) / 1e3
        emit({"suite": "trace", "case": args.trace_case, "mode": "warps of one k_table_search (us after the first warp started; percentiles 0 / 10 / 50 / 90 / 100)",
              "warps": int(len(w)), "warp_started": pct((w[:, 0] - t0) / 1e3), "wait_passed": pct((w[:, 1] - t0) / 1e3),
              "first_unit_finished": pct((w[units > 0, 2] - t0) / 1e3), "warp_ended": pct((w[:, 3] - t0) / 1e3),
              "first_unit_us": pct((w[units > 0, 2] - w[units > 0, 1]) / 1e3),
              "warps_by_units_taken": {str(int(k)): int((units == k).sum()) for k in np.unique(units)},
              "median_busy_us_by_units_taken": {str(int(k)): round(float(np.median(busy[units == k])), 2) for k in np.unique(units)}})


def write_md(path, rows):
    with open(path, "w") as f:
        f.write("| suite | case | variant | criteria | N | M | ms/case (median) | ms/case (back to back) | t_p ms | "
                "t_gamma ms | M/t_gamma (1/s) | N/t_total (1/s) | table search items | vertex visits | sum gamma^3 | "
                "pass rate | max gamma | oracle s/case (cores) |\n")
        f.write("|" + "---|" * 18 + "\n")
        for r in rows:
            if "variant" not in r:
                continue
            o = r.get("cpu_oracle")
            f.write(f"| {r['suite']} | {r['case']} | {r['variant']} | {r['criteria']} | {r['N']} | {r['M']} | "
                    f"{r['ms_case_median']:.4f} | {r['ms_case_back_to_back']:.4f} | {r['t_p_ms']:.4f} | "
                    f"{r['t_gamma_ms']:.4f} | {r['M'] / (r['t_gamma_ms'] * 1e-3):.3e} | {r['grid_voxels_per_s']:.3e} | "
                    f"{r['n_table_search']} | {r['vertex_visits']} | {r['sum_gamma3']:.4g} | {r['pass_rate']:.4f} | "
                    f"{r['max_gamma']:.3f} | "
                    + (f"{o['seconds_per_case_extrapolated']:.2f} ({o['cores']})" if o else "-") + " |\n")
        for r in rows:
            if "variant" not in r:
                f.write("\n`" + json.dumps(r) + "`\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--suite", default="all", choices=["configs", "criteria", "batch", "sort", "general", "trace", "all"])
    ap.add_argument("--trace-case", default="cfg3")
    ap.add_argument("--reps", type=int, default=30)
    ap.add_argument("--oracle-seconds", type=float, default=8.0)
    ap.add_argument("--md", default=None)
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench_suite.py needs a CUDA device: libgamma_b200 has no CPU path")
    torch.cuda.set_device(0)
    rows = []

    def emit(r):
        rows.append(r)
        print(json.dumps({k: v for k, v in r.items() if not k.startswith("_")}), flush=True)

    if args.suite in ("configs", "all"):
        suite_configs(args, emit)
    if args.suite in ("criteria", "all"):
        suite_criteria(args, emit)
    if args.suite in ("batch", "all"):
        suite_batch(args, emit)
    if args.suite in ("sort", "all"):
        suite_sort(args, emit)
    if args.suite in ("general", "all"):
        suite_general(args, emit)
    if args.suite == "trace":
        suite_trace(args, emit)
    if args.md:
        write_md(args.md, rows)


if __name__ == "__main__":
    main()
