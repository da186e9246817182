#!/usr/bin/env python3
"""bench.py -- times the gamma-index hot path (one `gamma_eval` = one step) on the headline workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--case cfg3] [--no-cpu-baseline]
                    [--no-configs] [--serial-calls]

Workload (config.workload): BASELINE.json configs[2], the "3D 2%/2 mm case" that north_star and SURVEY.md
section 8(d) name as the headline roofline case: 128x128x64 beam phantom at 2.5 mm, (2.0, 1.5, -1.0) mm shift,
scale 0.97, noise 2 %, criteria 2 %/2 mm global, 10 % cutoff.  Synthetic, seeded (paper_1012_1900_b200/phantoms.py).

value     evaluated reference voxels per second (gamma evaluations/s) over all ranks, inputs resident in HBM
e2e       the same through gamma_eval_host: pinned HOST buffers in, HOST gamma out, copies inside the timed region
roofline  dominant kernel, bound "alu": algorithmic FLOPs / its CUDA-event duration,
          against the plain FP32 FMA peak 148 SM x 128 lanes x 2 x 1.965 GHz; the FFMA-chain rate measured on
          the box is reported beside it
cpu_baseline / --impl reference: the CPU oracle (oracle/) as it stands, on the host cores
parity    the map the last timed step wrote against the oracle's map of the cpu_baseline leg, element by element
ms_per_step is the PIPELINED rate (opts.back_to_back = 1, about six calls in flight); ms_per_step_serial / serial_calls is
the library default (one call after the other on the caller's stream, the plain gamma_eval signature), ms_per_call_isolated
a single call; configs = the other BASELINE.json configs and cfg5 without the voxel pre-sort, same loop

N > 1: replicas only: every rank runs the same case on its own GPU, no data-path
collective; timing = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

SM_COUNT, FP32_LANES, SM_MAX_MHZ_NOMINAL = 148, 128, 1965.0
F_CELL_3D, F_CELL_2D = 1911.0, 190.0       # canonical flops per visited cell, frozen in BASELINE.md
L2_BYTES = 126e6
# executed FP32 flops per unit (ncu smsp__sass_thread_inst_executed_op_{fadd,fmul,ffma}_pred_on, FFMA counted twice),
# measured on the final round-2 kernels (profiles/r2_mix_<case>.csv, profiles/r2_profile.md): k_star 451 per evaluated
# voxel (450.6 / 451.5 / 450.6 / 451.0 on cfg2 / cfg3 / cfg5 / cfg4_fine); k_table_search = 380 per owner-vertex visit +
# 1 212 per ring item (solved from the cfg2 and cfg3 launches, reproduces cfg5 and cfg4_fine to 0.1 %)
FLOP_PER_STAR_VOXEL, FLOP_PER_VISIT, FLOP_PER_RING_ITEM = 451.0, 380.0, 1212.0
# executed WARP instructions (smsp__inst_executed.sum of the same captures) as unit costs plus a fixed part per launch:
# k_norm and k_classify per grid voxel, k_star per evaluated voxel, k_table_search per owner-vertex visit and per ring
# item (least squares over the four cases; reproduces each launch to a few per cent; k_classify's fixed part after its
# constants moved to one thread per block: 1.634 M on cfg3 instead of the 1.823 M of that capture)
WINST = {"norm_per_voxel": 0.0567, "norm_fixed": 0.474e6, "classify_per_voxel": 1.096, "classify_fixed": 0.47e6,
         "star_per_voxel": 27.3, "star_fixed": 0.70e6, "visit": 19.84, "ring_item": 30.4, "search_fixed": 0.288e6}
SCHEDULERS = 4 * SM_COUNT                   # one warp instruction per scheduler per cycle
# dram__bytes_read.sum + dram__bytes_write.sum per launch on cfg3 from the ncu --set full capture (profiles/r2_full_summary.csv)
TRAFFIC_BYTES = {"k_star": 2.69e6, "k_table_search": 1.83e6}


def f32(x):
    return float(np.float32(x))


def work_model(case_name):
    p = os.path.join(ROOT, "tests", "golden", "work_model.json")
    if os.path.exists(p):
        return json.load(open(p)).get(case_name)
    return None


# ------------------------------------------------------------------------------------------------------
# clocks: sampled DURING the timed regions through NVML
# ------------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index):
        self.samples, self.mask, self.ok, self.max_mhz = [], 0, False, None
        self._stop, self._active = threading.Event(), threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and all(t.strip().isdigit() for t in vis.split(",")) else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)
        self.t = threading.Thread(target=self._run, daemon=True)
        if self.ok:
            self.t.start()

    def _run(self):
        while not self._stop.is_set():
            if self._active.is_set():
                try:
                    self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                    self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:  # noqa: BLE001
                    try:
                        self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                    except Exception:  # noqa: BLE001
                        pass
                time.sleep(0.002)
            else:
                time.sleep(0.0005)

    def __enter__(self):
        self._active.set()
        return self

    def __exit__(self, *a):
        self._active.clear()

    def report(self):
        self._stop.set()
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable: " + getattr(self, "err", "")]}
        reasons = [n for b, n in self.REASONS.items() if self.mask & b and n != "gpu_idle"]
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------------
# the CPU oracle legs (the only places this file touches oracle/)
# ------------------------------------------------------------------------------------------------------
_last_oracle_gamma = None      # the map of the last oracle_time() call (the parity record of the bench line uses it)


def oracle_time(case, voxels, reps):
    global _last_oracle_gamma
    import oracle
    oracle.build()
    best = float("inf")
    sp = [f32(s) for s in case.spacing_mm]
    for _ in range(reps):
        t0 = time.perf_counter()
        _last_oracle_gamma = oracle.gamma(case.ref, case.eval, case.dims, sp, f32(case.dd), f32(case.dta_mm), case.mode,
                                          f32(case.cutoff), voxels=voxels)
        best = min(best, time.perf_counter() - t0)
    return best, oracle.num_threads()


def parity_record(case, keep, timed_map):
    """The map the LAST TIMED step wrote (headline launch configuration) against the oracle, element by element, on the
    voxels the cpu_baseline leg has just computed (all evaluated voxels).  Bar: |dgamma| <= 1e-4 (BASELINE.json north_star),
    identical NaN masks, pass/fail equal outside 1e-4 of gamma = 1."""
    og = _last_oracle_gamma
    g = timed_map.astype(np.float64)
    excluded = np.ones(g.size, dtype=bool)
    excluded[keep] = False
    d = np.abs(g[keep] - og)
    near_one = np.abs(og - 1.0) <= 1e-4
    return {"compared_voxels": int(keep.size), "max_abs_dgamma": float(np.nanmax(d)) if keep.size else 0.0,
            "tolerance": 1e-4, "nan_mask_equal": bool(np.isnan(g[excluded]).all() and not np.isnan(g[keep]).any()
                                                      and not np.isnan(og).any()),
            "pass_equal": bool(np.array_equal((g[keep] <= 1.0)[~near_one], (og <= 1.0)[~near_one])),
            "what": "gamma map written by the last timed step (opts.back_to_back as timed) vs oracle/ fp64, all evaluated voxels"}


def evaluated_voxels(case):
    ref = case.ref.ravel().astype(np.float64)
    return np.flatnonzero(ref >= f32(case.cutoff) * ref.max())


def cpu_baseline(case):
    """The oracle on the whole workload (all evaluated voxels), best of 3: a few seconds of all host cores."""
    keep = evaluated_voxels(case)
    t, cores = oracle_time(case, keep, 3)
    return keep, {"value": keep.size / t, "unit": "evaluated reference voxels/s", "cores": cores, "kind": "oracle",
            "sample": f"all {keep.size} evaluated voxels of {case.name}, shell-form double-precision search, "
                      f"best of 3 runs ({t:.2f} s each)", "seconds_per_case": t}


def run_reference(args, case, rank):
    if rank != 0:
        return
    keep = evaluated_voxels(case)
    rng = np.random.default_rng([0, 99])
    # bounded sample per step: calibrate on 4 % of the voxels, then size a step to ~0.25 s
    probe = np.sort(rng.choice(keep, size=max(1, keep.size // 25), replace=False))
    t_probe, cores = oracle_time(case, probe, 1)
    per_voxel = t_probe / probe.size
    n_step = int(min(keep.size, max(256, 0.25 / per_voxel)))
    sample = np.sort(rng.choice(keep, size=n_step, replace=False))
    for _ in range(args.warmup):
        oracle_time(case, sample, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_time(case, sample, 1)
    dt = (time.perf_counter() - t0) / args.steps
    val = n_step / dt
    unit = "evaluated reference voxels/s"
    print(json.dumps({
        "impl": "reference", "metric": "gamma evaluations per second", "value": val, "unit": unit,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": case_desc(case), "sample_voxels_per_step": n_step},
        "cpu_baseline": {"value": val, "unit": unit, "cores": cores, "kind": "oracle",
                         "sample": f"{n_step} seeded random evaluated voxels of {case.name} per step "
                                   f"(of {keep.size}); rate is per voxel, so it extrapolates to the case"},
        "e2e": {"value": val, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def case_desc(case):
    nx, ny, nz = case.dims
    return (f"{case.name}: {nx}x{ny}x{nz} fp32 beam phantom, {case.spacing_mm[0]} mm voxels, "
            f"{case.dd * 100:g}%/{case.dta_mm:g} mm {'global' if case.mode == 0 else 'local'}, "
            f"{case.cutoff * 100:g}% cutoff (BASELINE.json configs[2])" if case.name == "cfg3" else
            f"{case.name}: {nx}x{ny}x{nz}, {case.dd * 100:g}%/{case.dta_mm:g} mm")


# ------------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--case", default="cfg3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config records (cfg1 .. cfg5, cfg5 without pre-sort)")
    ap.add_argument("--presort", type=int, default=0)
    ap.add_argument("--star-phase", type=int, default=0)
    ap.add_argument("--lanes", type=int, default=0)
    ap.add_argument("--serial-calls", action="store_true", help="do not overlap consecutive calls (opts.back_to_back = 0)")
    ap.add_argument("--star-load", type=int, default=0, help="opts.star_load: 1 compacted list (default), 2 TMA tiles, 3 tiles by loads")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from paper_1012_1900_b200 import phantoms
    case = phantoms.make_case(args.case)

    if args.impl == "reference":
        run_reference(args, case, rank)
        return

    import torch
    from paper_1012_1900_b200 import binding
    from paper_1012_1900_b200.binding import GammaOpts
    from paper_1012_1900_b200.replicas import Replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libgamma_b200 has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    rep = Replicas(device=dev)              # nccl group when WORLD_SIZE > 1; replicas only, no data-path collective
    barrier, max_over_ranks = rep.barrier, rep.max_over_ranks

    N = case.ref.size
    # back_to_back: the timed loop enqueues nothing but gamma_eval_ex calls on the stream, which is what the flag asserts
    okw = dict(presort=args.presort, star_phase=args.star_phase, lanes_per_voxel=args.lanes, star_load=args.star_load)
    opts = GammaOpts(back_to_back=0 if args.serial_calls else 1, **okw)
    popts = GammaOpts(profile_stages=1, **okw)
    # Rotating input sets larger than L2 (126 MB): every timed step reads buffers that the previous steps have
    # pushed out of L2.  Each set = ref + eval + out = 12 B/voxel.
    nsets = int(np.ceil(2.0 * L2_BYTES / (12.0 * N))) + 1
    t_pinned = time.perf_counter()
    ref_h = torch.from_numpy(case.ref.ravel().copy()).pin_memory()
    ev_h = torch.from_numpy(case.eval.ravel().copy()).pin_memory()
    out_h = torch.empty(N, dtype=torch.float32).pin_memory()
    refs = [ref_h.to(dev, non_blocking=True) for _ in range(nsets)]
    evs = [ev_h.to(dev, non_blocking=True) for _ in range(nsets)]
    outs = [torch.empty(N, dtype=torch.float32, device=dev) for _ in range(nsets)]
    stream = torch.cuda.current_stream()
    args_c = (case.dims, case.spacing_mm, case.dd, case.dta_mm, case.mode, case.cutoff)

    def step(i, o=opts):
        k = i % nsets
        binding.gamma_eval_ex(refs[k], evs[k], *args_c, o, outs[k], stream)

    clocks = ClockSampler(local_rank)

    # ---- device-resident timing --------------------------------------------------------------------
    # one-time set-up of the library, not part of the W warm-up steps: the first call on each of the six lane streams
    # allocates that lane's workspace (cudaMalloc synchronises) and builds its graph; two rounds over the lanes
    INIT_CALLS = 12
    for i in range(INIT_CALLS):
        step(i)
    torch.cuda.synchronize()
    for i in range(args.warmup):
        step(i)
    barrier()
    l0 = binding.gamma_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with clocks:
        e0.record(stream)
        t_sub = time.perf_counter()
        for i in range(args.steps):
            step(args.warmup + i)
        t_sub = (time.perf_counter() - t_sub) / args.steps
        e1.record(stream)
        barrier()
    launches = binding.gamma_launch_count() - l0
    ms_step = max_over_ranks(e0.elapsed_time(e1) / args.steps)
    cnt = binding.gamma_get_counters()
    M = cnt["n_evaluated"]
    torch.cuda.synchronize()
    timed_map = outs[(args.warmup + args.steps - 1) % nsets].cpu().numpy()      # what the last timed step wrote

    # ---- the same loop, one call after the other on the caller's stream (the library default, back_to_back = 0): with
    # default options this is the plain north_star signature gamma_eval(...); then isolated calls (a synchronise between)
    sopts = GammaOpts(**okw)
    plain = not any(okw.values())

    def serial_step(i):
        k = i % nsets
        if plain:
            binding.gamma_eval(refs[k], evs[k], *args_c, outs[k], stream)
        else:
            binding.gamma_eval_ex(refs[k], evs[k], *args_c, sopts, outs[k], stream)

    for i in range(max(args.warmup, 4)):
        serial_step(i)
    barrier()
    ls0 = binding.gamma_launch_count()
    ts0, ts1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with clocks:
        ts0.record(stream)
        for i in range(args.steps):
            serial_step(args.warmup + i)
        ts1.record(stream)
        barrier()
    serial_launches = binding.gamma_launch_count() - ls0
    serial_ms_step = max_over_ranks(ts0.elapsed_time(ts1) / args.steps)
    iso = []
    for i in range(min(args.steps, 50)):
        ti0, ti1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ti0.record(stream)
        serial_step(i)
        ti1.record(stream)
        ti1.synchronize()
        iso.append(ti0.elapsed_time(ti1))
    isolated_ms = max_over_ranks(float(np.median(iso)))

    # ---- per-stage CUDA events (library records them on the launching stream).  NOT the timed launch configuration:
    # opts.profile_stages switches back_to_back off, so these are the kernels of a SERIAL call on full-size grids
    stage_acc = {}
    nprof = min(args.steps, 50)
    barrier()
    with clocks:
        for i in range(nprof):
            step(i, popts)
            for k, v in binding.gamma_get_stage_times().items():
                stage_acc.setdefault(k, []).append(v)
    stages = {k: float(np.mean(v)) for k, v in stage_acc.items()}

    # ---- end to end through the host-buffer entry point ---------------------------------------------
    # warm-up: on this pool host<->device copies from pinned buffers run at a third of the link's rate for the first
    # second or two after the buffers were pinned (plain cudaMemcpyAsync calls show the same; it settles by itself,
    # busy or idle), so the untimed calls go on until that time has passed and two consecutive groups of calls agree
    def settle(fn, t_pinned, min_s=2.5, max_s=8.0):
        last = None
        while True:
            t0 = time.perf_counter()
            fn()
            dt = time.perf_counter() - t0
            age = time.perf_counter() - t_pinned
            if (age > min_s and last is not None and abs(dt - last) <= 0.03 * last) or age > max_s:
                return
            last = dt

    def host_calls(n=20):
        for _ in range(n):
            binding.gamma_eval_host(ref_h, ev_h, *args_c, opts, out_h, stream)

    settle(host_calls, t_pinned)
    barrier()
    ne2e = max(5, min(args.steps, 50))
    with clocks:
        t0 = time.perf_counter()
        for _ in range(ne2e):
            binding.gamma_eval_host(ref_h, ev_h, *args_c, opts, out_h, stream)   # synchronises before returning
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / ne2e
    e2e_s = max_over_ranks(e2e_s)

    # ---- end to end, a stream of cases: gamma_eval_host_batch overlaps the copies of consecutive cases with compute
    nhb = 32
    hb_refs = [ref_h] + [ref_h.clone().pin_memory() for _ in range(nhb - 1)]
    hb_evs = [ev_h] + [ev_h.clone().pin_memory() for _ in range(nhb - 1)]
    hb_outs = [torch.empty(N, dtype=torch.float32).pin_memory() for _ in range(nhb)]
    hb_dims, hb_sp = [case.dims] * nhb, [case.spacing_mm] * nhb
    hb_args = (case.dd, case.dta_mm, case.mode, case.cutoff)
    t_pinned_hb = time.perf_counter()
    settle(lambda: binding.gamma_eval_host_batch(hb_refs, hb_evs, hb_dims, hb_sp, *hb_args, None, hb_outs, stream), t_pinned_hb)
    barrier()
    nrep_hb = 3
    with clocks:
        t0 = time.perf_counter()
        for _ in range(nrep_hb):
            binding.gamma_eval_host_batch(hb_refs, hb_evs, hb_dims, hb_sp, *hb_args, None, hb_outs, stream)   # synchronises
        e2e_pipe_s = (time.perf_counter() - t0) / (nrep_hb * nhb)
    e2e_pipe_s = max_over_ranks(e2e_pipe_s)
    e2e_pipe_ok = bool(torch.equal(torch.nan_to_num(hb_outs[nhb - 1], nan=-1.0), torch.nan_to_num(out_h, nan=-1.0)))
    del hb_refs, hb_evs, hb_outs
    # what the PCIe link of this box gives for the same buffers (plain pinned copies, nothing else running): the bound
    # of any host-buffer path is 8N bytes / this host-to-device rate
    tc0, tc1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dst = torch.empty(2 * N, dtype=torch.float32, device=dev)
    dst[:N].copy_(ref_h, non_blocking=True)
    tc0.record(stream)
    for _ in range(10):
        dst[:N].copy_(ref_h, non_blocking=True)
        dst[N:].copy_(ev_h, non_blocking=True)
    tc1.record(stream)
    torch.cuda.synchronize()
    h2d_gbs = 10 * 8 * N / (tc0.elapsed_time(tc1) * 1e-3) / 1e9
    # ... and with the device-to-host copy of a result running at the same time on another stream, as in the pipeline
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s_out):
        for _ in range(24):
            out_h.copy_(outs[0], non_blocking=True)
    with torch.cuda.stream(s_in):
        tc0.record(s_in)
        for _ in range(10):
            dst[:N].copy_(ref_h, non_blocking=True)
            dst[N:].copy_(ev_h, non_blocking=True)
        tc1.record(s_in)
    torch.cuda.synchronize()
    h2d_gbs_duplex = 10 * 8 * N / (tc0.elapsed_time(tc1) * 1e-3) / 1e9
    del dst

    # ---- stats on the result (not timed: a6 is reported separately) ---------------------------------
    hist, summ = binding.gamma_stats(outs[0], 64, 4.0)
    torch.cuda.synchronize()
    tstat0, tstat1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    hbuf, sbuf = binding.gamma_stats_async(outs[0], 64, 4.0)
    tstat0.record(stream)
    for i in range(20):
        binding.gamma_stats_async(outs[i % nsets], 64, 4.0, hbuf, sbuf)
    tstat1.record(stream)
    torch.cuda.synchronize()
    stats_ms = tstat0.elapsed_time(tstat1) / 20
    # a6 fused into the call (gamma_opts::stats_*): the same loop as the headline with the statistics accumulated where
    # gamma is written; one pair of result buffers per input set so that consecutive calls stay pipelined
    sh = [torch.empty(64, dtype=torch.int64, device=dev) for _ in range(nsets)]
    ss = [torch.empty(48, dtype=torch.uint8, device=dev) for _ in range(nsets)]
    fopts = [GammaOpts(back_to_back=opts.back_to_back, stats_hist=sh[k], stats_summary=ss[k], stats_hist_max=4.0, **okw)
             for k in range(nsets)]
    for i in range(args.warmup):
        step(i, fopts[i % nsets])
    barrier()
    tf0, tf1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tf0.record(stream)
    for i in range(args.steps):
        step(args.warmup + i, fopts[(args.warmup + i) % nsets])
    tf1.record(stream)
    torch.cuda.synchronize()
    fused_ms_step = max_over_ranks(tf0.elapsed_time(tf1) / args.steps)
    fused_summ = binding.decode_summary(ss[(args.warmup + args.steps - 1) % nsets])

    # ---- the same loop with D_norm GIVEN (opts.norm_dose = the phantom's maximum): a0 is not computed, the call is three
    # kernels.  Reported beside the headline, never as it: the headline computes D_norm = max(ref) on the device.
    nopts = GammaOpts(back_to_back=opts.back_to_back, norm_dose=float(cnt["norm_dose"]), **okw)
    for i in range(max(args.warmup, 12)):
        step(i, nopts)
    barrier()
    tn0, tn1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tn0.record(stream)
    for i in range(args.steps):
        step(args.warmup + i, nopts)
    tn1.record(stream)
    torch.cuda.synchronize()
    given_ms_step = max_over_ranks(tn0.elapsed_time(tn1) / args.steps)

    # ---- the same cases, 16 per gamma_eval_batch call (reported beside the headline, not as it) --
    nbatch = min(16, nsets)
    bdims, bsp = [case.dims] * nbatch, [case.spacing_mm] * nbatch
    bargs = (case.dd, case.dta_mm, case.mode, case.cutoff)
    for _ in range(3):
        binding.gamma_eval_batch(refs[:nbatch], evs[:nbatch], bdims, bsp, *bargs, opts, outs[:nbatch], stream)
    barrier()
    tb0, tb1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    nrep = max(3, min(args.steps // nbatch, 20))
    tb0.record(stream)
    for _ in range(nrep):
        binding.gamma_eval_batch(refs[:nbatch], evs[:nbatch], bdims, bsp, *bargs, opts, outs[:nbatch], stream)
    tb1.record(stream)
    torch.cuda.synchronize()
    batch_ms_case = max_over_ranks(tb0.elapsed_time(tb1) / (nrep * nbatch))

    # ---- the other BASELINE.json configs and Table 2's pair (cfg5 with / without the voxel pre-sort), so
    # that the driver's run carries them: ms per case back to back (same loop as the headline), >= 50 timed steps each
    def warp_inst(n_vox, c):
        return (n_vox * (WINST["norm_per_voxel"] + WINST["classify_per_voxel"]) + WINST["norm_fixed"] + WINST["classify_fixed"]
                + c["n_evaluated"] * WINST["star_per_voxel"] + WINST["star_fixed"]
                + c["vertex_visits"] * WINST["visit"] + c["n_ring_search"] * WINST["ring_item"] + WINST["search_fixed"])

    def time_config(name, extra, steps=60):
        c = phantoms.make_case(name)
        n = c.ref.size
        ns = max(2, int(np.ceil(2.0 * L2_BYTES / (12.0 * n))) + 1)
        r_h, e_h = torch.from_numpy(c.ref.ravel().copy()), torch.from_numpy(c.eval.ravel().copy())
        rs, es = [r_h.to(dev) for _ in range(ns)], [e_h.to(dev) for _ in range(ns)]
        os_ = [torch.empty(n, dtype=torch.float32, device=dev) for _ in range(ns)]
        a = (c.dims, c.spacing_mm, c.dd, c.dta_mm, c.mode, c.cutoff)
        res = {"case": name, "dims": list(c.dims), "criteria": f"{c.dd * 100:g}%/{c.dta_mm:g}mm", "grid_voxels": n,
               "options": dict(extra), "steps": steps, "rotating_sets": ns}
        for label, b2b in (("ms_per_case", 1), ("ms_per_case_serial", 0)):
            o = GammaOpts(back_to_back=b2b, **extra)
            for i in range(12):
                binding.gamma_eval_ex(rs[i % ns], es[i % ns], *a, o, os_[i % ns], stream)
            torch.cuda.synchronize()
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with clocks:
                t0.record(stream)
                for i in range(steps):
                    binding.gamma_eval_ex(rs[i % ns], es[i % ns], *a, o, os_[i % ns], stream)
                t1.record(stream)
                torch.cuda.synchronize()
            res[label] = max_over_ranks(t0.elapsed_time(t1) / steps)
        cc = binding.gamma_get_counters()
        _, sm = binding.gamma_stats(os_[0], 64, 4.0)
        res.update({"evaluated_voxels": int(cc["n_evaluated"]), "n_table_search": int(cc["n_table_search"]),
                    "vertex_visits": int(cc["vertex_visits"]),
                    "value": world * cc["n_evaluated"] / (res["ms_per_case"] * 1e-3), "unit": "evaluated reference voxels/s",
                    "pass_rate": sm["n_pass"] / max(1, sm["n_eval"]), "sum_gamma3": float(sm["sum_gamma3"]),
                    "max_gamma": float(sm["max_gamma"])})
        if sum(d > 1 for d in c.dims) == 3:
            res["warp_inst"] = warp_inst(n, cc)
        del rs, es, os_
        torch.cuda.empty_cache()
        return res

    config_records = []
    if not args.no_configs:
        for name, extra in (("cfg1", {}), ("cfg2", {}), ("cfg4_coarse", {}), ("cfg4_fine", {}), ("cfg5", {}),
                            ("cfg5", {"presort": 2})):
            config_records.append(time_config(name, extra))

    probe_tflops = binding.gamma_fp32_probe(5)
    clk = clocks.report()

    if rank != 0:
        rep.close()
        return

    # ---- roofline of the dominant kernel ------------------------------------------------------------
    # bound "alu": executed FP32 flops (FADD + FMUL + 2 FFMA thread instructions; per-unit constants measured
    # with ncu) x the units the library counted for this launch / the kernel's CUDA-event
    # duration.  "canonical" is the useful rate by the normal-equations flop count of SURVEY.md section 8(d).
    wm = work_model(case.name) or {}
    ndim = sum(d > 1 for d in case.dims)
    fcell = F_CELL_3D if ndim == 3 else F_CELL_2D
    kernel_ms = {"k_star": stages["star_ms"], "k_table_search": stages["search_ms"]}
    search_flops = cnt["vertex_visits"] * FLOP_PER_VISIT + cnt["n_ring_search"] * FLOP_PER_RING_ITEM
    units = {"k_star": M, "k_table_search": max(1, cnt["n_table_search"])}       # voxels the launch works on
    flop_per_unit = {"k_star": FLOP_PER_STAR_VOXEL if ndim == 3 else 0.0,
                     "k_table_search": search_flops / max(1, cnt["n_table_search"])}
    peak = SM_COUNT * FP32_LANES * 2 * SM_MAX_MHZ_NOMINAL * 1e6 / 1e12
    per_kernel = {k: {"units_per_launch": units[k], "flop_per_unit": flop_per_unit[k],
                      "algorithmic_flops_per_launch": units[k] * flop_per_unit[k], "kernel_ms": kernel_ms[k],
                      "achieved": units[k] * flop_per_unit[k] / (kernel_ms[k] * 1e-3) / 1e12,
                      "frac": units[k] * flop_per_unit[k] / (kernel_ms[k] * 1e-3) / 1e12 / peak,
                      "traffic": TRAFFIC_BYTES.get(k)} for k in kernel_ms}
    # the dominant kernel is the one that executes more FP32 work (a count, the same on every box), not the longer of two
    # event times that differ by nanoseconds
    dom = max(per_kernel, key=lambda k: per_kernel[k]["algorithmic_flops_per_launch"])
    alg = units[dom] * flop_per_unit[dom]
    roof = {"bound": "alu", "kernel": dom, "kernels": per_kernel, "peak": peak, "unit": "TFLOP/s", "traffic": TRAFFIC_BYTES.get(dom),
            "kernel_time_source": "serial call, opts.profile_stages (CUDA events between the stages of a call on the caller's "
                                  "stream, full-size grids); the headline ms_per_step is the pipelined rate: whole_path.frac "
                                  "is the fraction of the timed configuration",
            "peak_source": "148 SM x 128 FP32 lanes x 2 flop x 1.965 GHz (guide unit counts and clocks.max.sm); "
                           "MEASURED_PEAKS.json has no FP32 figure",
            "ffma_chain_measured_tflops": probe_tflops, "stage_ms": stages,
            "units_per_launch": units[dom], "flop_per_unit": flop_per_unit[dom],
            "algorithmic_flops_per_launch": alg,
            "achieved": alg / (kernel_ms[dom] * 1e-3) / 1e12}
    roof["frac"] = roof["achieved"] / peak
    roof["frac_of_ffma_chain_probe"] = roof["achieved"] / probe_tflops if probe_tflops > 0 else None
    # the bound that actually limits this path: issue slots.  Warp instructions of one step (per-unit constants above x
    # the units the library counted) / (592 schedulers x 1 instruction per cycle x the SM clock)
    winst = warp_inst(N, cnt)
    clk_hz = (clk.get("sm_mhz") or SM_MAX_MHZ_NOMINAL) * 1e6
    issue_us = winst / SCHEDULERS / clk_hz * 1e6
    for r in config_records:
        if "warp_inst" in r:
            r["issue_frac"] = r["warp_inst"] / SCHEDULERS / clk_hz * 1e6 / (r["ms_per_case"] * 1e3)
    roof["issue"] = {"warp_inst": winst, "bound_us": issue_us, "frac": issue_us / (ms_step * 1e3),
                     "note": "executed warp instructions / (592 schedulers x 1 per cycle x SM clock) over the step time; "
                             "3D grids (per-unit constants measured on cfg2 / cfg3 / cfg5 / cfg4_fine)"}
    exec_total = units["k_star"] * flop_per_unit["k_star"] + units["k_table_search"] * flop_per_unit["k_table_search"]
    roof["whole_path"] = {"executed_fp32_flops": exec_total, "achieved": exec_total / (ms_step * 1e-3) / 1e12,
                          "frac": exec_total / (ms_step * 1e-3) / 1e12 / peak}
    if wm:
        total_flops = wm["sum_Ns"] * fcell
        roof["canonical"] = {"flops_per_cell_visit": fcell, "cell_visits": wm["sum_Ns"], "flops": total_flops,
                             "useful_tflops": total_flops / (ms_step * 1e-3) / 1e12,
                             "note": "normal-equations count of SURVEY.md 8(d); the closed form executes ~13x fewer "
                                     "operations, so this is a useful-work rate, not a utilisation"}

    line = {
        "metric": "gamma evaluations per second", "value": world * M / (ms_step * 1e-3),
        "unit": "evaluated reference voxels/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": case_desc(case), "grid_voxels": N, "evaluated_voxels": M,
                   "l2_policy": f"{nsets} rotating input/output sets ({nsets * 12 * N / 1e6:.0f} MB) > 126 MB L2",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "options": {"presort": args.presort, "star_phase": args.star_phase, "lanes": args.lanes,
                               "star_load": args.star_load, "back_to_back": opts.back_to_back},
                   "call_mode": ("pipelined: consecutive gamma_eval_ex calls with opts.back_to_back = 1 overlap on 6 library "
                                 "streams, ms_per_step is a throughput with about six calls in flight"
                                 if opts.back_to_back else "serial: one call after the other on the caller's stream"),
                   "init_calls_before_warmup": INIT_CALLS},
        "headline_mode": "pipelined" if opts.back_to_back else "serial",
        "ms_per_step_serial": serial_ms_step, "ms_per_call_isolated": isolated_ms,
        "serial_calls": {"entry_point": "gamma_eval" if plain else "gamma_eval_ex", "back_to_back": 0,
                         "ms_per_step": serial_ms_step, "value": world * M / (serial_ms_step * 1e-3),
                         "unit": "evaluated reference voxels/s", "steps": args.steps, "gpu_launches": int(serial_launches),
                         "ms_per_call_isolated": isolated_ms,
                         "note": "the library default: calls one after the other on the caller's stream (round 1's headline "
                                 "definition); isolated = median of calls with a synchronise between them"},
        "configs": config_records,
        "e2e_pipelined_ms_per_case": e2e_pipe_s * 1e3,
        "grid_voxels_per_s": world * N / (ms_step * 1e-3), "ms_per_case": ms_step,
        "e2e": {"value": world * M / e2e_s, "unit": "evaluated reference voxels/s", "ms_per_case": e2e_s * 1e3,
                "h2d_bytes_per_step": 8 * N, "d2h_bytes_per_step": 4 * N,
                "pipelined": {"value": world * M / e2e_pipe_s, "unit": "evaluated reference voxels/s",
                              "ms_per_case": e2e_pipe_s * 1e3, "cases_per_call": nhb, "same_result_as_single_call": e2e_pipe_ok,
                              "h2d_bytes_per_case": 8 * N, "d2h_bytes_per_case": 4 * N,
                              "h2d_gbs_of_this_box": h2d_gbs, "h2d_bound_ms_per_case": 8 * N / (h2d_gbs * 1e9) * 1e3,
                              "h2d_gbs_while_d2h_runs": h2d_gbs_duplex,
                              "h2d_bound_ms_per_case_while_d2h_runs": 8 * N / (h2d_gbs_duplex * 1e9) * 1e3,
                              "note": "gamma_eval_host_batch: pinned HOST buffers in and out, H2D of case i+1 and D2H of "
                                      "case i-1 overlapped with the kernels of case i; wall time of the synchronising call"}},
        "gpu_launches": int(launches), "host_submit_us_per_step": t_sub * 1e6,
        "clocks": clk, "roofline": roof,
        "counters": cnt, "stats": summ, "stats_ms": stats_ms,
        "stats_fused": {"ms_per_step_with_stats": fused_ms_step, "extra_ms": fused_ms_step - ms_step,
                        "agrees_with_gamma_stats": bool(fused_summ["n_eval"] == summ["n_eval"]
                                                        and fused_summ["n_pass"] == summ["n_pass"]),
                        "note": "gamma_opts::stats_*: a6 accumulated inside the gamma kernels; stats_ms is the separate gamma_stats call"},
        "norm_dose_given": {"ms_per_step": given_ms_step, "norm_dose": float(cnt["norm_dose"]),
                            "note": "opts.norm_dose = D_norm: no k_norm, three kernels per call; not the headline"},
        "batched": {"cases_per_call": nbatch, "ms_per_case": batch_ms_case,
                    "value": world * M / (batch_ms_case * 1e-3), "unit": "evaluated reference voxels/s",
                    "note": "gamma_eval_batch: independent cases spread over 6 library-owned streams"},
    }
    if not args.no_cpu_baseline and world == 1:
        keep, line["cpu_baseline"] = cpu_baseline(case)
        line["parity"] = parity_record(case, keep, timed_map)
    elif world > 1:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    rep.close()
    binding.gamma_release()                 # a -DGAMMA_HOSTPROF build prints its host-side time profile here (stderr)


if __name__ == "__main__":
    main()
