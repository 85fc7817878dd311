"""bench.py -- TPC clusters/s and Pb-Pb collisions/s on B200 (BASELINE.json metric), one JSON line on stdout.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]

A step = one pass of the whole hot path (S0..S6: K1 grid, K2 neighbours, K3 clean/start, K5 tracklets, K6 selector) over one
synthetic time frame.  Default workload: config C3 (2 ms continuous frame at 50 kHz, ~12.5 M clusters, ~93 collisions).
`value`: clusters/s with the clusters already resident in HBM (tpc_find_tracks_device, results stay on the device).
`e2e`:   same metric through the C ABI with HOST buffers: pinned host -> device copy of (pad-y, time), all kernels, and the
         device -> host copy of the tracks, every step.
N > 1 (torchrun): every rank processes its own time frame (seed 3+rank) -- independent units, no data-path collective, weak
scaling; time = max over ranks.  --impl reference: the CPU oracle (oracle/), as it stands, on a bounded sample.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tpc_clusters_per_s"
UNIT = "clusters/s"
# algorithmic HBM bytes per cluster
BYTES_PER_CLUSTER = {"grid": 24.0, "neighbours": 20.0, "clean_start": 24.0}
# fp32 flops per S5 primitive, counted from csrc/kalman.cuh / k5_tracklets.cu: a fused multiply-add (reading A43)
# counts two flops, everything else one; INST_* are the fp32 instructions that carry them (an FMA is one instruction)
FLOP_PROPAGATE, FLOP_UPDATE, FLOP_PICKUP = 173.0, 133.0, 28.0
INST_PROPAGATE, INST_UPDATE, INST_PICKUP = 112.0, 79.0, 28.0


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe): one `nvidia-smi -lms 20`
    process streams samples while the steps run."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thr = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.strip().split(",")])
        self.thr = threading.Thread(target=pump, daemon=True)
        self.thr.start()
        t0 = time.time()
        while not self.rows and time.time() - t0 < 3.0:      # first sample before the timed region starts
            time.sleep(0.01)
        self.n_before = len(self.rows)

    def stop(self):
        if self.proc is not None:
            time.sleep(0.03)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=3)
            except Exception:
                self.proc.kill()
        rows = self.rows[max(0, getattr(self, "n_before", 1) - 1):]
        sm = [float(r[0]) for r in rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in rows if len(r) >= 6 for i in range(4) if r[2 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(rows)}


def oracle_run(w, sectors):
    """The oracle as it stands on a sector sample of the workload; returns (seconds, clusters, cores)."""
    from tests import parity as P
    ws = w.sector_slice(sectors)
    o = P.make_oracle(ws)
    t0 = time.perf_counter()
    o.run("s6")
    return time.perf_counter() - t0, ws.n_clusters, 1


def oracle_run_parallel(w, n_threads):
    """The same oracle over ALL sectors of the workload, one independent instance per sector, the instances shared out over
    n_threads host threads (sectors are independent; the paper's CPU tracking scales linearly with cores).
    Returns (seconds, clusters, threads)."""
    import queue
    from tests import parity as P
    n_threads = max(1, min(n_threads, w.n_sectors))
    orcs = [P.make_oracle(w.sector_slice([s])) for s in range(w.n_sectors)]      # ctypes calls release the GIL
    todo = queue.SimpleQueue()
    for o in orcs:
        todo.put(o)

    def work():
        while True:
            try:
                o = todo.get_nowait()
            except Exception:      # noqa: BLE001  (queue.Empty)
                return
            o.run("s6")
    th = [threading.Thread(target=work) for _ in range(n_threads)]
    t0 = time.perf_counter()
    [t.start() for t in th]
    [t.join() for t in th]
    return time.perf_counter() - t0, w.n_clusters, n_threads


def run_reference(args, rank, world):
    if rank != 0:
        return
    from gen import workloads as W
    w = W.config(args.config, seed=args.config)
    sectors = list(range(args.ref_sectors))
    times, n = [], 0
    for i in range(args.warmup + args.steps):
        dt, n, cores = oracle_run(w, sectors)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    v = n / (ms * 1e-3)
    sample = f"sectors 0..{args.ref_sectors - 1} of C{args.config} ({n} clusters) per step, full S0..S6, fp32 oracle instance"
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f32", "data": "synthetic", "config": {"workload": f"C{args.config}", "sample": sample},
                      "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


def run_gpu(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import paper_1905_05515_b200 as T
    from gen import workloads as W

    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    w = W.config(args.config, seed=args.config + rank)          # every rank its own time frame (weak scaling)
    N = w.n_clusters
    stream = torch.cuda.current_stream()
    trk = T.Tracker(**w.geometry(), **dict((kv.split("=")[0], float(kv.split("=")[1])) for kv in args.param))
    trk.set_stream(stream.cuda_stream)
    y_d, t_d = torch.from_numpy(w.y).cuda(), torch.from_numpy(w.t).cuda()
    y_h, t_h = torch.from_numpy(w.y).pin_memory(), torch.from_numpy(w.t).pin_memory()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    # ---- device-resident arm: `value`
    trk.load_batch(w.unit_off, y_d, t_d)
    for _ in range(args.warmup):
        res = trk.find_tracks_device()
    keys = ("ms_grid", "ms_neighbours", "ms_clean_start", "ms_tracklets", "ms_selector")
    acc = {k: 0.0 for k in keys}
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    launches = 0
    for _ in range(args.steps):
        res = trk.find_tracks_device()
        tm = trk.timings()
        launches += tm["launches"]
        for k in keys:
            acc[k] += tm[k]
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms = max_over_ranks(e0.elapsed_time(e1) / args.steps)
    total_clusters = sum_over_ranks(float(N))
    total_colls = sum_over_ranks(float(w.n_collisions))
    value = total_clusters / (ms * 1e-3)
    kern = {k: acc[k] / args.steps for k in keys}
    n_tracks, n_refs = res.n_tracks, res.n_cluster_refs
    # fp32 FMA-loop peak of this box at the clocks of this run (untimed part): the roofline denominator of S5
    fma_peak = trk.measure_fp32_peak() if rank == 0 else None
    # S8 (NEXT-4, not part of the timed step): attachment status of every cluster (Fig. 7's attached / adjacent)
    mk = [trk.mark_clusters(1.5, device_result=True) for _ in range(3)]
    mark_ms = float(np.mean([m["ms_mark"] for m in mk[1:]]))
    mst = mk[-1]["status"]
    marks = {"ms": mark_ms, "clusters_per_s": N / (mark_ms * 1e-3), "tube_cm": 1.5, "attached_frac": float((mst == 1).sum().item()) / N,
             "adjacent_frac": float((mst == 2).sum().item()) / N, "note": "S8 cluster attachment status (SURVEY 8(f).4), outside the timed step"}
    # S9 (NEXT-3, not part of the timed step): cross-sector segment matching
    mg = [trk.merge_tracks(device_result=True) for _ in range(3)]
    merges = {"ms": float(np.mean([m["ms_merge"] for m in mg[1:]])), "matched_pairs": int((mg[-1]["next"] >= 0).sum().item()),
              "note": "S9 cross-sector segment matching (SURVEY 8(f).3), outside the timed step"}
    # S10 (NEXT-3, second half, not part of the timed step): turns of one looping particle
    lo = [trk.find_loopers(device_result=True) for _ in range(3)]
    loopers = {"ms": float(np.mean([m["ms_loopers"] for m in lo[1:]])), "linked_tracks": int((lo[-1]["prev"] >= 0).sum().item()),
               "note": "S10 looper turns (SURVEY 8(f).3), outside the timed step"}
    # NEXT-2 variant (seed bridging, reading A39), measured beside the default path, never mixed into `value`
    variant = None
    if args.variant and rank == 0:
        variant = {}
        for vname, vp in (("skip_links", dict(link_skip=1.0)),
                          ("skip_links_strict", dict(link_skip=1.0, skip_cut2=0.4375)),
                          ("drop_bridged", dict(bridge_rows=4.0, bridge_min=8.0)),
                          ("rescue_wave", dict(bridge_rows=4.0, bridge_min=3.0, bridge_rescue=1.0))):
            with T.Tracker(**w.geometry(), **vp) as tv:
                tv.set_stream(stream.cuda_stream)
                tv.load_batch(w.unit_off, y_d, t_d)
                for _ in range(args.warmup):
                    rv = tv.find_tracks_device()
                torch.cuda.synchronize()
                e0.record(stream)
                for _ in range(args.steps):
                    rv = tv.find_tracks_device()
                e1.record(stream)
                torch.cuda.synchronize()
                vms = e0.elapsed_time(e1) / args.steps
                vt = tv.timings()
                variant[vname] = {"params": vp, "ms_per_step": vms, "value": N / (vms * 1e-3), "unit": UNIT,
                                  "n_start_hits": int(vt["n_start_hits"]), "n_tracklets_fitted": int(vt["n_tracklets_kept"]),
                                  "tracks_per_step": int(rv.n_tracks), "cluster_refs_per_step": int(rv.n_cluster_refs),
                                  "kernel_ms": {k: vt[k] for k in keys}}
        variant["note"] = ("NEXT-2 variants (SURVEY 8(f).2), all off by default because they change the result: skip_links = S2', links "
                           "that may skip one pad row (reading A45), skip_links_strict = the same with a quarter of cut2 for the pairs that skip a row "
                           "(the setting that keeps the efficiency of the default path); seed bridging (readings A39 / A39c): drop_bridged drops the start hits "
                           "that continue a lower chain, rescue_wave fits them in a second K5 wave when the first left their chain unused; "
                           "efficiency versus generator truth in DESIGN.md section 11")
    # S7 (NEXT-1, not part of the timed S0..S6 step): refit over the owned clusters + collision time, device-resident result
    refit_ms = float(np.mean([trk.refit_tracks(device_result=True)["ms_refit"] for _ in range(4)][1:]))

    # ---- end-to-end arm: host buffers in, host tracks out, every step.  Serial (one frame at a time: latency) and pipelined
    #      (two contexts on two streams, one host thread each: the copies of one frame overlap the kernels of the other).
    for _ in range(min(args.warmup, 3)):
        trk.load_batch(w.unit_off, y_h, t_h); trk.find_tracks()
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        trk.load_batch(w.unit_off, y_h, t_h)
        hres = trk.find_tracks()
    e1.record(stream)
    barrier()
    ms_e2e_serial = max_over_ranks(e0.elapsed_time(e1) / args.steps)

    NF = max(1, args.frames_in_flight)
    streams = [torch.cuda.Stream() for _ in range(NF)]
    trks = [T.Tracker(**w.geometry(), pinned_async=1, **dict((kv.split("=")[0], float(kv.split("=")[1])) for kv in args.param)) for _ in streams]
    for t_, s_ in zip(trks, streams):
        t_.set_stream(s_.cuda_stream)
        t_.load_batch(w.unit_off, y_h, t_h); t_.find_tracks()            # warm-up: buffers allocated
    steps_of = [list(range(j, args.steps, NF)) for j in range(NF)]
    errs = []

    def worker(j):
        try:
            torch.cuda.set_device(local_rank)
            for _ in steps_of[j]:
                trks[j].load_batch(w.unit_off, y_h, t_h)
                trks[j].find_tracks()
        except Exception as ex:      # noqa: BLE001
            errs.append(ex)

    barrier()
    e0.record(stream)
    for s_ in streams:
        s_.wait_event(e0)
    th = [threading.Thread(target=worker, args=(j,)) for j in range(NF)]
    [t_.start() for t_ in th]
    [t_.join() for t_ in th]
    for s_ in streams:
        stream.wait_stream(s_)
    e1.record(stream)
    barrier()
    if errs:
        raise errs[0]
    ms_e2e = max_over_ranks(e0.elapsed_time(e1) / args.steps)
    # the same NF contexts / streams on the frame they hold (device-resident: no load, results stay in HBM): what a stream of frames
    # gains when the kernel chains of two frames run side by side and fill each other's tails (extra key, not `value`)

    def worker_dev(j):
        try:
            torch.cuda.set_device(local_rank)
            for _ in steps_of[j]:
                trks[j].find_tracks_device()
        except Exception as ex:      # noqa: BLE001
            errs.append(ex)

    for t_ in trks:
        t_.find_tracks_device()
    barrier()
    e0.record(stream)
    for s_ in streams:
        s_.wait_event(e0)
    th = [threading.Thread(target=worker_dev, args=(j,)) for j in range(NF)]
    [t_.start() for t_ in th]
    [t_.join() for t_ in th]
    for s_ in streams:
        stream.wait_stream(s_)
    e1.record(stream)
    barrier()
    if errs:
        raise errs[0]
    ms_dev_pipe = max_over_ranks(e0.elapsed_time(e1) / args.steps)
    for t_ in trks:
        t_.close()
    h2d = 2 * 4 * N
    d2h = hres.n_tracks * (4 + 4 + 20 + 60 + 4 + 4 + 4) + (hres.n_tracks + 1) * 8 + hres.n_cluster_refs * 8
    trk.close()
    # ---- linearity check (PAPER.md:41 / Fig. 1 "almost linear" run time versus event size): ns per cluster of the same
    #      device-resident step on C2 (one event), the benched workload and C5 (10 ms frame), outside the timed region of `value`
    linearity = None
    if rank == 0 and world == 1 and not args.no_linearity:
        linearity = {f"C{args.config}": {"clusters": N, "ms_per_step": ms, "ns_per_cluster": ms * 1e6 / N}}
        for k in (2, 5):
            if k == args.config:
                continue
            wk = W.config(k, seed=k)
            with T.Tracker(**wk.geometry()) as tk:
                tk.set_stream(stream.cuda_stream)
                yk, tk_d = torch.from_numpy(wk.y).cuda(), torch.from_numpy(wk.t).cuda()
                tk.load_batch(wk.unit_off, yk, tk_d)
                for _ in range(3):
                    rk = tk.find_tracks_device()
                torch.cuda.synchronize()
                e0.record(stream)
                nst = 5
                for _ in range(nst):
                    rk = tk.find_tracks_device()
                e1.record(stream)
                torch.cuda.synchronize()
                msk = e0.elapsed_time(e1) / nst
                linearity[f"C{k}"] = {"clusters": wk.n_clusters, "ms_per_step": msk, "ns_per_cluster": msk * 1e6 / wk.n_clusters,
                                      "tracks_per_step": int(rk.n_tracks), "collisions": wk.n_collisions,
                                      "kernel_ms": {kk: tk.timings()[kk] for kk in keys}}
                del yk, tk_d
            if k == 2 and not args.no_cpu_baseline:      # the oracle on all 36 sectors of C2 as well (one core, and all cores)
                dt1, n1, _ = oracle_run(wk, list(range(wk.n_sectors)))
                dtp, np_, nth = oracle_run_parallel(wk, min(36, len(os.sched_getaffinity(0))))
                linearity["C2"]["cpu_baseline"] = {"value": n1 / dt1, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt1,
                                                   "sample": f"all 36 sectors of C2 ({n1} clusters)"}
                linearity["C2"]["cpu_baseline_parallel"] = {"value": np_ / dtp, "unit": UNIT, "cores": nth, "seconds": dtp,
                                                            "sample": f"all 36 sectors of C2 ({np_} clusters), one oracle instance per sector"}
            del wk
        torch.cuda.empty_cache()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of every kernel; the dominant one goes into "roofline"
    hbm_peak, peak_src, sm_max = _peaks()
    nominal_issue = 148 * 128 * sm_max * 1e6 / 1e12  # T fp32 instructions/s: one per lane per clock (B200_PROFILING.md unit counts)
    alu_peak = fma_peak if fma_peak else 2.0 * nominal_issue   # TFLOP/s: the FMA-loop throughput measured above (two flops per FMA)
    issue_peak = 0.5 * alu_peak                      # T fp32 instructions/s
    traffic, traffic_source = {}, None
    tp = os.path.join(ROOT, "profiles", f"traffic_c{args.config}.csv")   # DRAM bytes per launch from the committed ncu --set full capture
    if os.path.exists(tp):
        for line in open(tp):
            f = line.strip().split(",")
            if line.startswith("#"):
                traffic_source = f"profiles/traffic_c{args.config}.csv: " + line[1:].strip()
            elif len(f) == 2 and f[1].isdigit():
                traffic[f[0]] = int(f[1])
    roofs = {}
    for name, key in (("grid", "ms_grid"), ("neighbours", "ms_neighbours"), ("clean_start", "ms_clean_start")):
        a = BYTES_PER_CLUSTER[name] * N / (kern[key] * 1e-3) / 1e9
        roofs[name] = {"bound": "hbm", "achieved": a, "peak": hbm_peak, "unit": "GB/s", "frac": a / hbm_peak, "peak_source": peak_src,
                       "ms": kern[key], "traffic": traffic.get(name)}
    flops = FLOP_PROPAGATE * tm["n_propagations"] + FLOP_UPDATE * tm["n_updates"] + FLOP_PICKUP * tm["n_pickups"]
    a = flops / (kern["ms_tracklets"] * 1e-3) / 1e12
    insts = INST_PROPAGATE * tm["n_propagations"] + INST_UPDATE * tm["n_updates"] + INST_PICKUP * tm["n_pickups"]
    roofs["tracklets"] = {"bound": "alu", "achieved": a, "peak": alu_peak, "unit": "TFLOP/s", "frac": a / alu_peak,
                          "peak_source": "measured: FMA loop of tpc_measure_fp32_peak in this run" if fma_peak else "nominal",
                          "peak_nominal": 2.0 * nominal_issue, "ms": kern["ms_tracklets"],
                          "fp32_inst_frac": insts / (kern["ms_tracklets"] * 1e-3) / 1e12 / issue_peak,
                          "traffic": traffic.get("tracklets")}
    roofs["selector"] = {"bound": "hbm", "achieved": None, "peak": hbm_peak, "unit": "GB/s", "frac": None, "ms": kern["ms_selector"],
                         "traffic": traffic.get("selector")}
    dominant = max(("grid", "neighbours", "clean_start", "tracklets"), key=lambda k: roofs[k]["ms"])
    roofline = dict(roofs[dominant]); roofline["kernel"] = dominant
    roofline["traffic_source"] = traffic_source

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        dt, n, cores = oracle_run(w, list(range(args.ref_sectors)))
        cpu = {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": f"sectors 0..{args.ref_sectors - 1} of C{args.config} ({n} clusters), full S0..S6, fp32 oracle instance, 1 thread"}
    cpu_par = None
    if cpu is not None:
        try:
            cores = len(os.sched_getaffinity(0))
        except AttributeError:
            cores = os.cpu_count() or 1
        dt, n, nth = oracle_run_parallel(w, min(36, cores))
        cpu_par = {"value": n / dt, "unit": UNIT, "cores": nth, "kind": "oracle, one instance per sector", "seconds": dt,
                   "sample": f"all {w.n_sectors} sectors of C{args.config} ({n} clusters), one oracle instance per sector over {nth} threads, full S0..S6",
                   "host_cores": cores}
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": f"C{args.config}: {w.params.t_frame:g} us frame, {N} clusters, {w.n_collisions} collisions per GPU",
                      "l2": "inputs+tables larger than L2 (no flush needed)" if N * 40 > 126e6 else "working set fits L2",
                      "parallelism": f"{world} independent time frames"},
           "collisions_per_s": total_colls / (ms * 1e-3), "tracks_per_step": n_tracks, "cluster_refs_per_step": n_refs,
           "realtime_factor": (w.params.t_frame * 1e-3 * world) / ms if w.params.t_frame > 0 else None,
           "e2e": {"value": total_clusters / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e, "h2d_bytes_per_step": h2d,
                   "d2h_bytes_per_step": d2h, "mode": f"{NF} frames in flight ({NF} contexts, {NF} streams, one host thread each, pinned_async=1: the pinned input is read by DMA after the load call returns): copies overlap kernels",
                   "serial_ms_per_step": ms_e2e_serial, "serial_value": total_clusters / (ms_e2e_serial * 1e-3)},
           "device_resident_in_flight": {"value": total_clusters / (ms_dev_pipe * 1e-3), "unit": UNIT, "ms_per_step": ms_dev_pipe, "frames_in_flight": NF,
                                         "note": "the same step with the kernel chains of several frames side by side (one context and stream per frame in flight, "
                                                 "inputs and results in HBM): they fill each other's tails; `value` is one frame at a time"},
           "gpu_launches": int(launches), "kernel_ms": kern,
           "s5_work": {k: int(tm[k]) for k in ("n_start_hits", "n_propagations", "n_updates", "n_pickups")}, "roofline": roofline, "roofline_all": roofs, "cpu_baseline": cpu, "cpu_baseline_parallel": cpu_par,
           "linearity": linearity, "variant_seed_bridging": variant, "cluster_marks": marks, "sector_merges": merges, "looper_turns": loopers,
           "refit": {"ms": refit_ms, "tracks_per_s": n_tracks / (refit_ms * 1e-3), "note": "S7 refit + collision time (SURVEY 8(f).1), outside the timed step"},
           "clocks": clocks}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="workload preset C1..C5 (default C3, the 50 kHz time frame)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-sectors", type=int, default=8, help="sectors of the workload the CPU oracle is timed on")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-linearity", action="store_true", help="skip the C2 / C5 runs of the linearity check")
    ap.add_argument("--frames-in-flight", type=int, default=2, help="contexts / streams of the pipelined end-to-end arm")
    ap.add_argument("--variant", action="store_true", help="also time the NEXT-2 seed-bridging variant (extra field, not `value`)")
    ap.add_argument("--param", action="append", default=[], help="library tunable name=value (tpc_set_param), e.g. chunk=1024")
    args = ap.parse_args()
    rank, world, local = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))
    if args.impl == "reference":
        return run_reference(args, rank, world)
    run_gpu(args, rank, world, local)


if __name__ == "__main__":
    main()
