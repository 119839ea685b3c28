#!/usr/bin/env python
"""bench.py -- the contract benchmark: visibilities gridded + degridded per second on BASELINE.json's
w-projection workload (configs[1], "config2": 36 antennas, 300 time steps x 64 channels = 12,096,000 visibilities,
2048^2 grid, 32 w-planes, support 15..63, oversampling 4) on one B200.

A "step" is one pass of the whole hot path over the batch: A1 index -> A2 bucket/sort -> A3 gridding -> A6 degridding
(imager_grid cold + imager_degrid with index reuse).  `value` = visibilities / step time with inputs resident in HBM;
`e2e` = the same through the C-ABI binding with HOST (pinned) buffers, H2D/D2H copies inside the timed region.
`roofline` is for the dominant kernel (gridding, FP32-FMA bound): achieved = 8 flop x nominal complex MACs / its
CUDA-event duration (warm call, index reused).  `cpu_baseline` = the oracle on a bounded sample of the same workload.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload configN] [--time-stride s]
`--workload config5` feeds its 181 M visibilities in chunks of `--chunk-steps` time steps (one call holds < 2^31 hits).
N > 1 runs N independent replicas (the path does not shard: BASELINE.json north_star "no sharding, no collectives").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FP32_FMA_PER_CLK_SM = 128          # B200_PROFILING.md / SURVEY 8(d): 128 FP32 lanes per SM
N_SM = 148


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return json.load(open(path)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.rows, self.stamps, self.stop_flag, self.index = [], [], False, index
        self.t_begin, self.t_end = 0.0, float("inf")
        self.query = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
                      "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
                      "clocks_event_reasons.sw_power_cap")

    def _nvml_loop(self):
        """NVML directly (a query takes microseconds; nvidia-smi takes ~0.4 s per call on these boxes)."""
        import pynvml
        pynvml.nvmlInit()
        h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
        get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
        bits = [0x8, 0x40, 0x20, 0x4]            # hw_slowdown, hw_thermal_slowdown, sw_thermal_slowdown, sw_power_cap
        sm_max = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
        while not self.stop_flag:
            r = int(get_reasons(h))
            self.rows.append([str(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)), str(sm_max),
                              str(pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0)] + ["Active" if r & b else "Not Active" for b in bits])
            self.stamps.append(time.perf_counter())
            time.sleep(0.01)

    def run(self):
        try:
            self._nvml_loop()
            return
        except Exception:
            pass                                  # no NVML binding: fall back to the nvidia-smi command line
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.query}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [p.strip() for p in out.strip().split(",")]
                if len(parts) >= 7:
                    self.rows.append(parts)
                    self.stamps.append(time.perf_counter())
            except Exception:
                pass
            time.sleep(0.05)

    def summary(self):
        rows_in = [r for r, t in zip(self.rows, self.stamps) if self.t_begin <= t <= self.t_end]
        self.rows = rows_in or self.rows            # samples taken while the timed loops ran (all of them if none fell inside)
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows), "power_w_max": max(float(r[2]) for r in self.rows)}


def reduce_times_max(times, device):
    """Element-wise MAX of per-rank times over all ranks (the replicas run side by side: the job takes as long as its
    slowest rank).  Identity when torch.distributed is not initialised or has one rank."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def job_throughput(units_per_rank, world, ms):
    """Whole-job units per second of `world` replicas that each processed `units_per_rank` in `ms` (weak scaling)."""
    return world * units_per_rank / (ms * 1e-3)


def oracle_tables(params):
    from oracle import kernels as okern
    tabs, _ = okern.make_tables(params)
    return okern.flatten_tables(tabs)


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on a bounded sample of the same workload."""
    from oracle import index as oidx, gridder as ogrid
    from synth import make_workload
    ogrid.build()
    stride = args.ref_time_stride
    wl = make_workload(args.workload, time_stride=stride)
    flat, offs = oracle_tables(wl.params)
    n = wl.params["grid_size"]
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        rec = oidx.index_visibilities(wl.uvw, wl.a_index, wl.params)
        keys = oidx.bucket_keys(rec, wl.params, tile=32)
        oidx.bucket_sort(keys, wl.params, tile=32)
        out = ogrid.grid(rec, wl.vis, wl.weights, flat, offs, wl.params)
        ogrid.degrid(rec, out["grid"].astype(np.complex64), flat, offs, wl.params)
        if it >= args.warmup:
            times.append(time.perf_counter() - t0)
    t = float(np.mean(times))
    value = wl.nvis / t
    cores = ogrid.max_threads()
    sample = f"{args.workload} every {stride}th time step ({wl.nvis} visibilities, full grid and tables)"
    line = {"metric": "visibilities gridded+degridded/sec", "value": value, "unit": "vis/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": args.workload, "nvis": wl.nvis, "grid": n, "sample": sample},
            "cpu_baseline": {"value": value, "unit": "vis/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "vis/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_chunks(name, time_stride, chunk_steps):
    """The workload as a list of chunks of whole time steps (one chunk unless the workload is fed in pieces: config 5's
    181 M visibilities exceed the 2^31 hits one call may hold, include/imager.h "Limits per call")."""
    from synth import make_workload
    if name != "config5" or chunk_steps <= 0:
        return [make_workload(name, time_stride=time_stride)]
    probe = make_workload(name, time_stride=time_stride, time_range=(0, 1))
    n_time = probe.notes["n_time_all"]
    return [make_workload(name, time_stride=time_stride, time_range=(t0, t0 + chunk_steps)) for t0 in range(0, n_time, chunk_steps)]


def counters_of_capture(workload, time_stride):
    """Per-launch counters of the two hot kernels from the committed `ncu --set full` captures (profiles/r3_traffic.txt:
    DRAM bytes read + written, wavefronts of the LSU data pipe) -- used only if the capture was taken on the kernel source that is being
    benchmarked (the file carries the SHA-256 of gridder_tiled.cu) and on this workload at its full size."""
    import hashlib
    prof = os.path.join(ROOT, "profiles", "r3_traffic.txt")
    src = os.path.join(ROOT, "paper_2206_15117_b200", "csrc", "gridder_tiled.cu")
    if not (os.path.exists(prof) and os.path.exists(src)) or time_stride != 1:
        return {}, "no capture for this workload"
    fields = dict(ln.split(None, 1) for ln in open(prof) if ln.strip() and not ln.startswith("#"))
    digest = hashlib.sha256(open(src, "rb").read()).hexdigest()
    if fields.get("gridder_tiled_cu_sha256", "").strip() != digest:
        return {}, "stale: the captures in profiles/r3_traffic.txt are of another version of gridder_tiled.cu"
    out = {k[len(workload) + 1:]: int(v) for k, v in fields.items() if k.startswith(workload + ".")}
    return out, ("profiles/r3_traffic.txt (ncu --set full, same kernel source)" if out else "no capture for this workload")


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libimager has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    from paper_2206_15117_b200 import Plan, REUSE_INDEX

    wls = workload_chunks(args.workload, args.time_stride, args.chunk_steps)
    params = wls[0].params
    nvis = sum(w.nvis for w in wls)
    multi = len(wls) > 1
    n, nc, npol = params["grid_size"], params["n_corr"], params["n_pol"]
    plan = Plan(params, max(w.nvis for w in wls))      # the library generates its own kernel tables (A0, untimed)
    path, why = plan.path()
    if path != "tiled" and not args.allow_reference:
        raise SystemExit(f"bench.py: this plan would run on the library's reference kernels, not the tiled ones ({why}); "
                         f"no line is printed for that path unless --allow-reference is given")

    # resident inputs, chunk by chunk
    def to_dev(w):
        return dict(uvw=torch.from_numpy(w.uvw).to(dev), vis=torch.from_numpy(w.vis).to(dev), wts=torch.from_numpy(w.weights).to(dev),
                    a=torch.from_numpy(w.a_index).to(dev) if w.a_index is not None else None,
                    out=torch.empty((w.nvis, nc), dtype=torch.complex64, device=dev))
    data = [to_dev(w) for w in wls]
    grid = torch.zeros((npol, n, n), dtype=torch.complex64, device=dev)
    stream = torch.cuda.current_stream()
    launches = 0
    reuse_degrid = 0 if multi else REUSE_INDEX          # one plan: with several chunks the degridding pass re-indexes too

    def step():
        nonlocal launches
        grid.zero_()
        for d in data:
            plan.grid(d["uvw"], d["vis"], d["wts"], grid, d["a"])                 # cold: A1 + A2 + A3
            launches += plan.last_launch_count()
        for d in data:
            plan.degrid(d["uvw"], grid, d["out"], d["a"], flags=reuse_degrid)      # A6 (+ A1 + A2 when chunked)
            launches += plan.last_launch_count()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(max(args.warmup, 3)):
        step()
    t_wait = time.perf_counter()
    while rank == 0 and not sampler.rows and time.perf_counter() - t_wait < 3.0:
        step()                                  # untimed: keep the GPU under load until nvidia-smi has answered once
    barrier()
    launches = 0
    sampler.t_begin = time.perf_counter()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    for a, b in ev:
        a.record(stream)
        step()
        b.record(stream)
    barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    # dominant kernels: warm gridding and warm degridding calls timed on their own (index reused), summed over the chunks;
    # the MAC counts come from the plan (imager_index_stats), not from the checker
    kern = {"grid": 0.0, "degrid": 0.0}
    stats = {"nominal_cmacs": 0, "executed_cmacs": 0, "n_merged": 0, "n_hits": 0, "n_kept": 0, "n_dropped": 0}
    reps = args.steps if not multi else min(args.steps, 3)
    for d in data:
        if multi:
            plan.index(d["uvw"], d["a"])
        st = plan.index_stats()
        for k in stats:
            stats[k] += st[k]
        for name, fn in (("grid", lambda: plan.grid(d["uvw"], d["vis"], d["wts"], grid, d["a"], flags=REUSE_INDEX)),
                         ("degrid", lambda: plan.degrid(d["uvw"], grid, d["out"], d["a"], flags=REUSE_INDEX))):
            for _ in range(3 if not multi else 1):
                fn()
            torch.cuda.synchronize()
            es = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
            for a, b in es:
                a.record(stream)
                fn()
                b.record(stream)
            torch.cuda.synchronize()
            kern[name] += float(np.mean([a.elapsed_time(b) for a, b in es]))
    barrier()
    sampler.t_end = time.perf_counter()
    sampler.stop_flag = True
    cmacs, cmacs_exec = stats["nominal_cmacs"], stats["executed_cmacs"]

    # end to end: pinned host buffers, H2D of the step's inputs and D2H of its results inside the timed region
    def pin(w):
        return dict(uvw=torch.from_numpy(w.uvw).pin_memory(), vis=torch.from_numpy(w.vis).pin_memory(),
                    wts=torch.from_numpy(w.weights).pin_memory(),
                    a=torch.from_numpy(w.a_index).pin_memory() if w.a_index is not None else None,
                    out=torch.empty((w.nvis, nc), dtype=torch.complex64).pin_memory())
    h_grid = torch.empty((npol, n, n), dtype=torch.complex64).pin_memory()
    h2d_stream, d2h_stream = torch.cuda.Stream(), torch.cuda.Stream()
    chunk_plans = []
    if multi:
        host = [pin(w) for w in wls]

        def e2e_step():
            # chunked workload: per chunk H2D -> imager_grid (cold); D2H grid; per chunk imager_degrid (cold) -> D2H
            grid.zero_()
            for d, h in zip(data, host):
                for k in ("uvw", "vis", "wts", "a"):
                    if h[k] is not None:
                        d[k].copy_(h[k], non_blocking=True)
                plan.grid(d["uvw"], d["vis"], d["wts"], grid, d["a"])
            h_grid.copy_(grid, non_blocking=True)
            for d, h in zip(data, host):
                plan.degrid(d["uvw"], grid, d["out"], d["a"])
                h["out"].copy_(d["out"], non_blocking=True)
        e2e_desc = f"{len(wls)} chunks in sequence: H2D chunk -> imager_grid; D2H grid; imager_degrid chunk -> D2H vis"
        h2d = sum(h[k].numel() * h[k].element_size() for h in host for k in ("uvw", "vis", "wts", "a") if h[k] is not None)
        d2h = sum(h["out"].numel() * 8 for h in host) + h_grid.numel() * 8
    else:
        # The call sequence a user with host buffers makes: the visibilities are cut into `e2e_chunks` chunks (gridding is
        # linear in them), each with its own plan; all H2D copies are queued on a copy stream, chunk k is indexed
        # (imager_index) as soon as its uvw have arrived and gridded (REUSE_INDEX) as soon as its visibilities and weights
        # have; the grid goes back to the host while the chunks are degridded, and every chunk's predictions follow it.
        # Steps are pipelined over TWO sets of device buffers: the H2D copies of step k + 1 run while step k is degridded and
        # its results go back (PCIe is full duplex); every step still copies all its inputs in and all its results out.
        w = wls[0]
        h = pin(w)
        h_uvw, h_vis, h_wts, h_a, h_out = h["uvw"], h["vis"], h["wts"], h["a"], h["out"]
        sets = [dict(data[0], grid=grid), dict(to_dev(w), grid=torch.zeros_like(grid))]
        for bs in sets:
            bs["in_free"] = None          # compute stream: the step that used these inputs has finished with them
            bs["out_free"] = None         # D2H stream: the results of the step that used these outputs are on the host
        nch = max(1, args.e2e_chunks)
        bounds = [(k * nvis) // nch for k in range(nch + 1)]
        chunk_plans = [Plan(params, bounds[k + 1] - bounds[k]) for k in range(nch)] if nch > 1 else [plan]
        step_no = [0]

        def e2e_step():
            bs = sets[step_no[0] % 2]
            step_no[0] += 1
            uvw, vis, wts, aidx, vout, g_dev = bs["uvw"], bs["vis"], bs["wts"], bs["a"], bs["out"], bs["grid"]
            if bs["in_free"] is not None:
                h2d_stream.wait_event(bs["in_free"])                     # this set's inputs are free again (two steps back)
            ev_u, ev_v = [], []
            with torch.cuda.stream(h2d_stream):
                for k in range(nch):
                    sl = slice(bounds[k], bounds[k + 1])
                    uvw[sl].copy_(h_uvw[sl], non_blocking=True)
                    if h_a is not None:
                        aidx[sl].copy_(h_a[sl], non_blocking=True)
                    ev_u.append(h2d_stream.record_event())
                    vis[sl].copy_(h_vis[sl], non_blocking=True)
                    wts[sl].copy_(h_wts[sl], non_blocking=True)
                    ev_v.append(h2d_stream.record_event())
            if bs["out_free"] is not None:
                stream.wait_event(bs["out_free"])                        # this set's grid and predictions have reached the host
            g_dev.zero_()
            for k in range(nch):
                sl = slice(bounds[k], bounds[k + 1])
                a_k = aidx[sl] if aidx is not None else None
                stream.wait_event(ev_u[k])
                chunk_plans[k].index(uvw[sl], a_k)                                               # A1 + A2
                stream.wait_event(ev_v[k])
                chunk_plans[k].grid(uvw[sl], vis[sl], wts[sl], g_dev, a_k, flags=REUSE_INDEX)    # A3
            d2h_stream.wait_event(stream.record_event())
            with torch.cuda.stream(d2h_stream):
                h_grid.copy_(g_dev, non_blocking=True)
            for k in range(nch):
                sl = slice(bounds[k], bounds[k + 1])
                a_k = aidx[sl] if aidx is not None else None
                chunk_plans[k].degrid(uvw[sl], g_dev, vout[sl], a_k, flags=REUSE_INDEX)          # A6
                d2h_stream.wait_event(stream.record_event())
                with torch.cuda.stream(d2h_stream):
                    h_out[sl].copy_(vout[sl], non_blocking=True)
            bs["in_free"] = stream.record_event()
            bs["out_free"] = d2h_stream.record_event()
        e2e_desc = (f"{nch} chunks: H2D uvw_k -> imager_index_k || H2D vis_k, weights_k -> imager_grid_k; "
                    f"D2H grid || imager_degrid_k -> D2H vis_k; consecutive steps alternate between two sets of device buffers, "
                    f"so that the copies of one step overlap the kernels of its neighbours")
        h2d = h_uvw.numel() * 4 + h_vis.numel() * 8 + h_wts.numel() * 4 + (h_a.numel() * 4 if h_a is not None else 0)
        d2h = h_out.numel() * 8 + h_grid.numel() * 8

    e2e_steps = max(1, min(args.steps, 50 if not multi else 2))       # the pipeline's fill and drain are inside the timed region
    e2e_step()
    e2e_step()
    barrier()
    t0 = torch.cuda.Event(enable_timing=True)
    t1 = torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    for _ in range(e2e_steps):
        e2e_step()
    stream.wait_event(d2h_stream.record_event())        # the last results are on the host before the clock stops
    t1.record(stream)
    barrier()
    e2e_ms = t0.elapsed_time(t1) / e2e_steps

    total_ms, e2e_ms = reduce_times_max([total_ms, e2e_ms], dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peaks, peaks_kind = load_peaks()
    ms_per_step = total_ms / args.steps
    value = job_throughput(nvis, world, ms_per_step)
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    peak_tflops = N_SM * FP32_FMA_PER_CLK_SM * sm_mhz * 1e6 * 2 / 1e12
    # flop rates on EXECUTED complex MACs (8 flop each); the nominal count also holds the MACs of duplicate visibilities
    # that the library pre-sums (same kernel set, cell and sub-cell: exact algebra, R16) and never executes
    achieved = 8.0 * cmacs_exec / (kern["grid"] * 1e-3) / 1e12
    achieved_nominal = 8.0 * cmacs / (kern["grid"] * 1e-3) / 1e12
    achieved_d = 8.0 * cmacs_exec / (kern["degrid"] * 1e-3) / 1e12
    achieved_d_nominal = 8.0 * cmacs / (kern["degrid"] * 1e-3) / 1e12
    cap, traffic_src = counters_of_capture(args.workload, args.time_stride)
    traffic, traffic_d = cap.get("grid.dram_bytes"), cap.get("degrid.dram_bytes")
    # the unit that binds both kernels: the LSU data pipe passes one 128-byte wavefront per clock per SM
    lsu_floor = lambda wavefronts: None if wavefronts is None else wavefronts / N_SM / (sm_mhz * 1e6) * 1e3
    in_bytes = nvis * (12 + 8 * nc + 4 * nc + (4 if wls[0].a_index is not None else 0))
    grid_bytes = npol * n * n * 8
    step_desc = ("imager_grid (index+sort+plan+grid) + imager_degrid (index reused)" if not multi else
                 f"{len(wls)} chunks of {args.chunk_steps} time steps through ONE plan: imager_grid per chunk (index+sort+plan+grid), "
                 f"then imager_degrid per chunk (index+sort+plan+degrid: the index of another chunk cannot be reused)")
    peak_kind = f"148 SM x 128 FP32 lanes x 2 flop x {sm_mhz:.0f} MHz ({peaks_kind} max SM clock)"
    dup_rate = stats["n_merged"] / max(1, stats["n_kept"])
    mac_note = ("achieved / frac count EXECUTED complex MACs (8 flop each); *_nominal_incl_presummed also count the MACs of the "
                "duplicate visibilities (same kernel set, cell and sub-cell) that the library sums before gridding and never "
                "executes -- duplicate_rate = merged / kept visibilities says how much of the synthetic workload that is")
    line = {
        "metric": "visibilities gridded+degridded/sec", "value": value, "unit": "vis/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "nvis": nvis, "grid": n, "n_wplanes": params["n_wplanes"],
                   "support": [params["support_min"], params["support_max"]], "oversample": params["oversample"],
                   "n_corr": nc, "time_stride": args.time_stride, "chunks": len(wls), "parallelism": f"replicas x{world}",
                   "kernel_path": path,
                   "l2": f"inputs ({in_bytes / 1e6:.0f} MB of visibilities + {grid_bytes / 1e6:.1f} MB grid) "
                         f"{'exceed' if in_bytes + grid_bytes > 126e6 else 'FIT IN'} the 126 MB L2; no explicit flush",
                   "step": step_desc, "e2e_step": e2e_desc},
        "clocks": sampler.summary(),
        "e2e": {"value": job_throughput(nvis, world, e2e_ms), "unit": "vis/s", "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms},
        "gpu_launches": launches,
        "roofline": {"bound": "alu", "kernel": "gridding (imager_grid, index reused)", "achieved": achieved,
                     "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops, "traffic": traffic,
                     "traffic_source": traffic_src, "peak_kind": peak_kind,
                     "lsu_wavefronts": cap.get("grid.lsu_wavefronts"), "lsu_floor_ms": lsu_floor(cap.get("grid.lsu_wavefronts")),
                     "kernel_ms": kern["grid"], "nominal_cmacs": cmacs, "executed_cmacs": cmacs_exec,
                     "achieved_nominal_incl_presummed": achieved_nominal,
                     "frac_nominal_incl_presummed": achieved_nominal / peak_tflops,
                     "merged_duplicates": stats["n_merged"], "duplicate_rate": dup_rate, "note": mac_note,
                     "hits": stats["n_hits"],
                     "grid_vis_per_s": nvis / (kern["grid"] * 1e-3), "grid_cmac_per_s": cmacs_exec / (kern["grid"] * 1e-3),
                     "cold_path_ms": ms_per_step - kern["grid"] - kern["degrid"],
                     "hbm_gbs_grid": (nvis * (16 + 4 + 8 * nc + 4 * nc) + 2 * grid_bytes) / (kern["grid"] * 1e-3) / 1e9},
        "roofline_degrid": {"bound": "alu", "kernel": "degridding (imager_degrid, index reused)", "achieved": achieved_d,
                            "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved_d / peak_tflops, "traffic": traffic_d,
                            "traffic_source": traffic_src, "peak_kind": peak_kind,
                            "lsu_wavefronts": cap.get("degrid.lsu_wavefronts"), "lsu_floor_ms": lsu_floor(cap.get("degrid.lsu_wavefronts")), "kernel_ms": kern["degrid"], "nominal_cmacs": cmacs,
                            "executed_cmacs": cmacs_exec, "achieved_nominal_incl_presummed": achieved_d_nominal,
                            "frac_nominal_incl_presummed": achieved_d_nominal / peak_tflops,
                            "degrid_vis_per_s": nvis / (kern["degrid"] * 1e-3),
                            "degrid_cmac_per_s": cmacs_exec / (kern["degrid"] * 1e-3)},
        "step_ms_all": step_ms,
    }
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args)
    print(json.dumps(line))
    for cp in chunk_plans:
        if cp is not plan:
            cp.close()
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def cpu_baseline(args):
    """The oracle as it stands on a bounded sample (about 10-30 s of CPU work) of the same workload."""
    from oracle import index as oidx, gridder as ogrid
    from synth import make_workload
    stride = args.ref_time_stride
    wl = make_workload(args.workload, time_stride=stride)
    flat, offs = oracle_tables(wl.params)
    t0 = time.perf_counter()
    rec = oidx.index_visibilities(wl.uvw, wl.a_index, wl.params)
    keys = oidx.bucket_keys(rec, wl.params, tile=32)
    oidx.bucket_sort(keys, wl.params, tile=32)
    out = ogrid.grid(rec, wl.vis, wl.weights, flat, offs, wl.params)
    ogrid.degrid(rec, out["grid"].astype(np.complex64), flat, offs, wl.params)
    t = time.perf_counter() - t0
    return {"value": wl.nvis / t, "unit": "vis/s", "cores": ogrid.max_threads(), "kind": "oracle",
            "sample": f"{args.workload} every {stride}th time step ({wl.nvis} visibilities, full grid and tables), "
                      f"index+sort+grid+degrid in {t:.1f} s"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default: 50, or 5 for --impl reference)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--time-stride", type=int, default=1, help="keep every n-th time step (1 = the full workload)")
    ap.add_argument("--ref-time-stride", type=int, default=20, help="time-step stride of the CPU oracle's sample")
    ap.add_argument("--e2e-chunks", type=int, default=1, help="chunks of the end-to-end pipeline within a step (1 = one call per stage; steps are pipelined over two buffer sets either way)")
    ap.add_argument("--chunk-steps", type=int, default=100, help="config5: time steps per chunk fed through the API")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--allow-reference", action="store_true", help="print a line even if the plan runs on the library's slow reference kernels")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 5 if args.impl == "reference" else 50
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            run_reference(args)
        return
    run_ours(args)


if __name__ == "__main__":
    main()
