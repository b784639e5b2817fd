"""bench.py -- clusters tracked per second on B200 for BASELINE.json configs[1] (central Pb-Pb).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--batch-events B] [--impl ours|reference]

One "step" = one tpc_track call = one pass of the whole hot path (a1 grid, a2 neighbours, a3 cleaner/seeds,
a4 follower, a5 ownership/selection) over a batch of B distinct synthetic central Pb-Pb events, concatenated as
B*36 independent sectors.  Prints ONE JSON line (rank 0).

  value        clusters/s over all ranks, inputs resident in HBM, CUDA events on the launching stream
  e2e          the same metric through tpc_track_host: pinned HOST buffers in, host buffers out, copies timed
  roofline     the dominant kernel (a4 follower): algorithmic work / its mean launch duration, measured with
               CUDA events recorded between the stages inside the timed region; plus roofline_path (whole step
               against the HBM roofline, the figure BASELINE.json's metric names) and per-stage times
  cpu_baseline the oracle (oracle/, fp64, OpenMP) timed on this box's host cores on a bounded sample

--impl reference times the oracle itself (there is no reference implementation to install; the paper has no
code), one bounded sample per step, rank 0 only.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "TPC clusters tracked/sec on 1 B200 (central Pb-Pb); % of HBM roofline"
UNIT = "clusters/s"
CFG_ID = 1
DEFAULT_BATCH_EVENTS = 32   # events per tpc_track call
# algorithmic work per unit: N clusters, N_b grid bins, T tracklet-hits, S seeds
# a4: fp32 flop EXECUTED per tracklet-hit (two filter passes + searches), counted from the SASS of the five a4 kernels
# with ncu's per-instruction thread counts: FFMA = 2, FMUL / FADD / FMNMX / FSETP / FSEL / MUFU = 1; no fp64 left.
FLOP_PER_TRACKLET_HIT = 566.0
FLOP_MODEL_SOURCE = "profiles/r02_a4_flop_model.md (SASS thread-instruction counts, ncu source page)"


def stage_bytes(n, n_bins, t_hits, seeds):
    """Algorithmic bytes per stage."""
    return {
        "a1": 20.0 * n + 4.0 * n_bins,
        "a2": 20.0 * n + 4.0 * n_bins,
        "a3": 24.0 * n + 8.0 * seeds,
        "a4": 16.0 * t_hits + 100.0 * seeds,
        "a5": 20.0 * t_hits,
    }


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback", 1965.0


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self._period = period_s
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _loop(self):
        nv = self._nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "applications_clocks_setting": 0x2, "sync_boost": 0x10}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self._period)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def shard_seeds(rank: int, world: int, batch_events: int) -> list[int]:
    """Weak scaling: every rank tracks its own `batch_events` distinct events; seeds never repeat across ranks."""
    return [1000 * CFG_ID + rank * batch_events + k for k in range(batch_events)]


def aggregate(local_ms: float, local_units: float, dist=None, device=None):
    """(max elapsed ms over ranks, total units over ranks).  Works on gloo (CPU tensors) and nccl."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_units
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def make_batch(seeds, n_tracks=None):
    from gen.events import make_event, concat_events
    evs = [make_event(CFG_ID, s, n_tracks=n_tracks) for s in seeds]
    return concat_events(evs), evs


def timed_round_robin(handles, steps, main):
    """`steps` tpc_track calls dealt round-robin over the (handle, stream, inputs, out) tuples in `handles`, timed with
    CUDA events on `main`: every stream waits for the start event, `main` waits for every stream's last call."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(main)
    for h in handles:
        if h["stream"] is not main:
            h["stream"].wait_event(e0)
    for k in range(steps):
        h = handles[k % len(handles)]
        h["trk"].track(h["y"], h["z"], h["ro"], h["out"], h["stream"])
    for h in handles:
        if h["stream"] is not main:
            done = torch.cuda.Event()
            done.record(h["stream"])
            main.wait_event(done)
    e1.record(main)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2502_09138_b200 import Tracker, load_library
    from paper_2502_09138_b200.events import geometry_from_event, upload

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU path")
    load_library()   # fails loudly if libtpctrack.so is missing
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)   # only for the barriers and the final max / sum

    B = args.batch_events
    ev, evs = make_batch(shard_seeds(rank, world, B))
    n = ev.n
    y, z, ro = upload(ev, dev)
    main = torch.cuda.current_stream()
    sweep = [args.streams] if args.streams > 0 else [1, 2, 3, 4]   # K handles/streams, best reported
    if args.profile:
        sweep = [1]
    handles = []
    for k in range(max(sweep)):
        t = Tracker(geometry_from_event(ev))
        t.set_a2_variant(args.a2_variant)
        handles.append({"trk": t, "stream": main if k == 0 else torch.cuda.Stream(dev), "y": y, "z": z, "ro": ro,
                        "out": t.alloc_out(n, track_capacity=n // 40 + 1024, hit_capacity=n + 1024)})
    trk, out = handles[0]["trk"], handles[0]["out"]

    if args.profile:   # for ncu: W warm-up calls + K calls on one stream, nothing else (see profiles/*.md)
        for _ in range(args.warmup + args.steps):
            trk.track(y, z, ro, out, main)
        torch.cuda.synchronize()
        print(json.dumps({"profile_run": True, "calls": args.warmup + args.steps, "launches_per_call": trk.launches_per_call(),
                          "clusters_per_call": n, "batch_events": B}))
        for h in handles:
            h["trk"].close()
        return

    # ---- device-resident arm: no stage events, no host work inside the timed region ------------------------
    for h in handles:
        for _ in range(args.warmup):
            h["trk"].track(h["y"], h["z"], h["ro"], h["out"], h["stream"])
    torch.cuda.synchronize()
    results = {}
    with ClockSampler(local_rank) as clk:
        for K in sweep:
            if world > 1:
                dist.barrier()
            for h in handles[:K]:   # the caller says how many calls it keeps in flight (sizes a4's persistent grids)
                h["trk"].set_concurrency(K)
            ms_k = timed_round_robin(handles[:K], args.steps, main)
            ms_k, units_k = aggregate(ms_k, float(n) * args.steps, dist if world > 1 else None, dev)
            results[K] = (ms_k, units_k)
    if world > 1:
        dist.barrier()
    best_k = min(results, key=lambda k: results[k][0])
    ms_max, units = results[best_k]
    value = units / (ms_max * 1e-3)

    for h in handles:
        h["trk"].set_concurrency(1)
    # ---- stage times: a separate pass on one stream with CUDA events between the stages ---------------------
    trk.set_stage_timing(True)
    for _ in range(min(args.steps, 16)):
        trk.track(y, z, ro, out, main)
    torch.cuda.synchronize()
    stage_ms, n_avg = trk.stage_ms_mean()
    trk.set_stage_timing(False)
    ms_total = results[1][0] if 1 in results else sum(stage_ms) * args.steps

    tracks, hit_ids, n_seeds = out.to_host()
    _, _, _, tl_nh, _ = trk.debug_tracklets(n_seeds)
    t_hits = float(tl_nh.sum())
    grid = trk.debug_grid(n)
    n_bins = float(grid["stride"]) * trk.n_sectors * trk.n_rows
    stream = main

    # ---- NEXT-1: tpc_refit on the tracks of the last call (not part of the step; reported beside it) --------
    for _ in range(2):
        trk.refit(y, z, ro, out, stream)
    torch.cuda.synchronize()
    r0e, r1e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    r0e.record(stream)
    for _ in range(5):
        trk.refit(y, z, ro, out, stream)
    r1e.record(stream)
    torch.cuda.synchronize()
    refit_ms = r0e.elapsed_time(r1e) / 5
    refit_recs = trk.refit(y, z, ro, out, stream)
    for _ in range(2):
        mres = trk.merge(refit_recs, out.counts, None, stream)
    torch.cuda.synchronize()
    r0e.record(stream)
    for _ in range(5):
        mres = trk.merge(refit_recs, out.counts, None, stream)
    r1e.record(stream)
    torch.cuda.synchronize()
    merge_ms = r0e.elapsed_time(r1e) / 5
    merge_counts = mres[3].cpu().numpy()
    for _ in range(2):
        trk.refit_merged(y, z, ro, out, mres[0], mres[1], None, stream)
    torch.cuda.synchronize()
    r0e.record(stream)
    for _ in range(5):
        trk.refit_merged(y, z, ro, out, mres[0], mres[1], None, stream)
    r1e.record(stream)
    torch.cuda.synchronize()
    refit_merged_ms = r0e.elapsed_time(r1e) / 5
    # NEXT-3: residual transform of the owned clusters + the entropy an ideal coder would reach on its histograms
    for _ in range(2):
        comp = trk.compress(y, z, ro, out, stream)
    torch.cuda.synchronize()
    r0e.record(stream)
    for _ in range(5):
        comp = trk.compress(y, z, ro, out, stream)
    r1e.record(stream)
    torch.cuda.synchronize()
    compress_ms = r0e.elapsed_time(r1e) / 5

    def _entropy(h):
        h = h.cpu().numpy().astype(np.float64)
        p = h[h > 0] / max(h.sum(), 1.0)
        return float(-(p * np.log2(p)).sum())

    comp_bits = {"ry": _entropy(comp["hist_ry"]), "rz": _entropy(comp["hist_rz"]), "drow": _entropy(comp["hist_drow"])}
    # NEXT-3, entropy stage: the three residual streams through tpc_rans_encode / tpc_rans_decode (chunks of 512)
    nh_owned = int(out.counts.cpu().numpy()[1])
    streams3 = [(comp["ry"][:nh_owned].contiguous(), 12), (comp["rz"][:nh_owned].contiguous(), 12),
                (comp["drow"][:nh_owned].contiguous(), 8)]
    encs = [trk.rans_encode(v, alphabet_bits=b, chunk=512, stream=stream) for v, b in streams3]
    torch.cuda.synchronize()
    r0e.record(stream)
    for _ in range(5):
        for (v, b), enc in zip(streams3, encs):
            trk.rans_encode(v, alphabet_bits=b, chunk=512, stream=stream, into=enc)
    r1e.record(stream)
    torch.cuda.synchronize()
    rans_encode_ms = r0e.elapsed_time(r1e) / 5
    decs = [trk.rans_decode(enc, stream=stream) for enc in encs]
    torch.cuda.synchronize()
    r0e.record(stream)
    for _ in range(5):
        for enc in encs:
            trk.rans_decode(enc, stream=stream)
    r1e.record(stream)
    torch.cuda.synchronize()
    rans_decode_ms = r0e.elapsed_time(r1e) / 5
    rans_lossless = all(bool(torch.equal(d, v)) for d, (v, _) in zip(decs, streams3))
    rans_bytes = 0
    for enc in encs:   # payload + raw escapes + two 32-bit offsets per chunk + the frequency table
        c = enc["counts"].cpu().numpy()
        rans_bytes += int(c[0]) + 4 * int(c[1]) + 8 * int(c[2]) + 4 * int(enc["freq"].shape[0])
    # NEXT-2: clusterizer on the synthetic digits of ONE configs[1] event (gen/digits.py)
    from gen.digits import make_digits
    dg = make_digits(evs[0])
    trk_c = Tracker(geometry_from_event(evs[0]))
    u16 = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(dev).view(torch.uint16)   # noqa: E731
    d_pad, d_time, d_adc = u16(dg.pad), u16(dg.time), u16(dg.adc)
    d_off = torch.from_numpy(dg.offsets.view(np.int32).copy()).to(dev)
    for _ in range(2):
        cl_out = trk_c.clusterize(d_pad, d_time, d_adc, d_off, dg.n_pads, stream=stream)
    torch.cuda.synchronize()
    r0e.record(stream)
    for _ in range(5):
        cl_out = trk_c.clusterize(d_pad, d_time, d_adc, d_off, dg.n_pads, stream=stream)
    r1e.record(stream)
    torch.cuda.synchronize()
    clusterize_ms = r0e.elapsed_time(r1e) / 5
    n_found = int(cl_out["counts"][0])
    trk_c.close()

    # ---- single-event latency (B = 1), for context -------------------------------------------------------
    ev1 = evs[0]
    trk1 = Tracker(geometry_from_event(ev1))
    y1, z1, ro1 = upload(ev1, dev)
    out1 = trk1.alloc_out(ev1.n)
    for _ in range(3):
        trk1.track(y1, z1, ro1, out1, stream)
    torch.cuda.synchronize()
    l0, l1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0.record(stream)
    for _ in range(10):
        trk1.track(y1, z1, ro1, out1, stream)
    l1.record(stream)
    torch.cuda.synchronize()
    latency_ms = l0.elapsed_time(l1) / 10
    # the same call captured once into a CUDA graph and replayed (14 launches become one)
    cg = torch.cuda.CUDAGraph()
    gs = torch.cuda.Stream(device=dev)
    with torch.cuda.graph(cg, stream=gs):
        trk1.track(y1, z1, ro1, out1, torch.cuda.current_stream())
    for _ in range(3):
        cg.replay()
    torch.cuda.synchronize()
    l0.record()
    for _ in range(10):
        cg.replay()
    l1.record()
    torch.cuda.synchronize()
    latency_graph_ms = l0.elapsed_time(l1) / 10
    trk1.close()

    # ---- end to end through the host-buffer entry point --------------------------------------------------
    # tpc_track_host returns when the results are in host memory.  A caller keeps the GPU busy the usual way: T host
    # threads, each with its own handle, stream and pinned buffers, so that one call's copies overlap another
    # call's kernels (ctypes releases the GIL during the call).  Every step still pays its own H2D and D2H.
    T = max(1, args.e2e_threads)
    hy = torch.from_numpy(ev.y.copy()).pin_memory()
    hz = torch.from_numpy(ev.z.copy()).pin_memory()
    hro = torch.from_numpy(ev.row_offsets.view(np.int32).copy()).pin_memory()
    e2e_steps = max(3 * T, min(args.steps, 20) // T * T)
    workers = []
    for k in range(T):
        w = {"trk": handles[k]["trk"] if k < len(handles) else Tracker(geometry_from_event(ev)),
             "stream": torch.cuda.Stream(dev),
             "tr": torch.empty(out.tracks.shape[0], dtype=torch.uint8).pin_memory(),
             "hi": torch.empty(out.hit_ids.shape[0], dtype=torch.int32).pin_memory(),
             "cn": torch.zeros(4, dtype=torch.int32).pin_memory()}
        w["trk"].set_concurrency(T)
        workers.append(w)

    def run_host(w, n_calls):
        torch.cuda.set_device(local_rank)
        for _ in range(n_calls):
            w["trk"].track_host(hy, hz, hro, w["tr"], w["hi"], w["cn"], w["stream"])

    for w in workers:   # warm-up (also sizes each handle's staging)
        run_host(w, 2)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    threads = [threading.Thread(target=run_host, args=(w, e2e_steps // T)) for w in workers]
    t0 = time.perf_counter()
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_max, e2e_units = aggregate(e2e_ms, float(n) * e2e_steps, dist if world > 1 else None, dev)
    hcn = workers[0]["cn"]
    h2d = int(hy.numel() * 4 + hz.numel() * 4 + hro.numel() * 4)
    d2h = int(16 + int(hcn[0]) * 112 + int(hcn[1]) * 4)
    for w in workers:
        assert int(w["cn"][0]) == len(tracks) and int(w["cn"][1]) == len(hit_ids), "host-buffer path disagrees with device path"
    for w in workers[len(handles):]:
        w["trk"].close()

    # ---- roofline ----------------------------------------------------------------------------------------
    hbm_peak, peak_kind, sm_max = read_peaks()
    sb = stage_bytes(float(n), n_bins, t_hits, float(n_seeds))
    names = ["a1", "a2", "a3", "a4", "a5"]
    stages = {k: {"ms": stage_ms[i], "alg_bytes": sb[k], "hbm_gbs": sb[k] / (stage_ms[i] * 1e-3) / 1e9}
              for i, k in enumerate(names)}
    dom = max(names, key=lambda k: stages[k]["ms"])
    step_ms = ms_max / args.steps        # the timed region's (best K)
    path_bytes = sum(sb.values())
    # a4 is plain-ALU bound (no dense contraction): fp32 FMA peak = SMs x 128 lanes x 2 flop x max SM clock
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    alu_peak_tf = n_sm * 128 * 2 * sm_max * 1e6 / 1e12
    a4_tf = FLOP_PER_TRACKLET_HIT * t_hits / (stages["a4"]["ms"] * 1e-3) / 1e12
    if dom == "a4":
        # large calls run a4 as four phase kernels + a vote kernel (api.cu); the stage events bracket all of them
        a4_name = ("a4_phase_kernel<0..3> + a4_votes_kernel" if trk.launches_per_call() == 12 else "a4_follow_kernel")
        roofline = {"kernel": a4_name, "bound": "alu", "achieved": a4_tf, "peak": alu_peak_tf,
                    "unit": "TFLOP/s", "frac": a4_tf / alu_peak_tf, "traffic": None,
                    "peak_kind": "derived: %d SM x 128 fp32 lanes x 2 x %.0f MHz (DESIGN.md)" % (n_sm, sm_max),
                    "flop_model": {"fp32_flop_per_tracklet_hit": FLOP_PER_TRACKLET_HIT, "fp64_flop_per_tracklet_hit": 0.0,
                                   "source": FLOP_MODEL_SOURCE},
                    "hbm_achieved_gbs": stages["a4"]["hbm_gbs"], "hbm_frac": stages["a4"]["hbm_gbs"] / hbm_peak,
                    "share_of_step": stages["a4"]["ms"] / sum(s["ms"] for s in stages.values())}
    else:
        roofline = {"kernel": dom, "bound": "hbm", "achieved": stages[dom]["hbm_gbs"], "peak": hbm_peak,
                    "unit": "GB/s", "frac": stages[dom]["hbm_gbs"] / hbm_peak, "traffic": None,
                    "peak_kind": peak_kind,
                    "share_of_step": stages[dom]["ms"] / sum(s["ms"] for s in stages.values())}
    try:   # measured DRAM bytes of the dominant kernel (one ncu --set full capture, see profiles/)
        tr = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(roofline["kernel"])
        if tr and int(tr["batch_events"]) == B:
            roofline["traffic"] = float(tr["dram_bytes_per_launch"])
            roofline["traffic_source"] = tr["source"]
    except (OSError, ValueError, KeyError):
        pass
    path_gbs = path_bytes / (step_ms * 1e-3) / 1e9
    roofline_path = {"bound": "hbm", "achieved": path_gbs, "peak": hbm_peak, "unit": "GB/s",
                     "frac": path_gbs / hbm_peak, "peak_kind": peak_kind, "frac_of_8TBs_nominal": path_gbs / 8000.0,
                     "alg_bytes_per_cluster": path_bytes / n}

    # ---- oracle on the host cores (rank 0, N = 1 only) ----------------------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle
        oracle.build()
        oracle.track(evs[0])   # warm the page cache / OpenMP pool
        t0 = time.perf_counter()
        done, k = 0, 0
        while time.perf_counter() - t0 < 12.0 and k < 64 * len(evs):
            oracle.track(evs[k % len(evs)])
            done += evs[k % len(evs)].n
            k += 1
        dt = time.perf_counter() - t0
        cpu = {"value": done / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{k} single configs[1] events ({done} clusters) in {dt:.1f} s, g++ -O2 -fopenmp fp64"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32 (a1-a3, a5) / f32 (a4: U-D factorised filter)", "data": "synthetic",
            "config": {"workload": f"configs[1] central Pb-Pb (4000 tracks, 36 sectors, 5% noise), {B} distinct "
                                   f"events per call as {B * 36} sectors", "batch_events": B,
                       "clusters_per_step_per_gpu": n, "seeds_per_step": int(n_seeds), "tracks_per_step": len(tracks),
                       "tracklet_hits_per_step": int(t_hits), "parallelism": "none (sectors independent; "
                       "ranks = replicas on their own events)", "streams": best_k,
                       "streams_sweep_clusters_per_s": {str(k): v[1] / (v[0] * 1e-3) for k, v in results.items()},
                       "l2": f"working set {trk.scratch_bytes() / 1e6:.0f} MB scratch + {8 * n / 1e6:.0f} MB input "
                             f"> 126 MB L2; no explicit flush"},
            "tracks_per_s": len(tracks) * world * args.steps / (ms_max * 1e-3),
            "single_event_latency_ms": latency_ms, "single_event_latency_cuda_graph_ms": latency_graph_ms,
            "next": {"a6_refit_ms": refit_ms, "tracks_refitted": len(tracks), "a7_merge_ms": merge_ms, "a6_refit_merged_ms": refit_merged_ms, "a8_compress_ms": compress_ms, "a9_clusterize_ms_one_event": clusterize_ms,
                     "clusterize_digits": int(dg.n), "clusterize_clusters": n_found,
                     "clusterize_digits_per_s": dg.n / (clusterize_ms * 1e-3),
                     "compress_entropy_bits_per_symbol": comp_bits, "owned_clusters": int(len(hit_ids)),
                     "compress_bits_per_owned_cluster": comp_bits["ry"] + comp_bits["rz"] + comp_bits["drow"],
                     "a10_rans_encode_ms": rans_encode_ms, "a10_rans_decode_ms": rans_decode_ms,
                     "rans_bytes": rans_bytes, "rans_bits_per_owned_cluster": 8.0 * rans_bytes / max(nh_owned, 1),
                     "rans_raw_bits_per_owned_cluster": 72, "rans_lossless": rans_lossless,
                     "merge_links": int(merge_counts[0]), "merged_tracks": int(merge_counts[1]),
                     "note": "tpc_refit, tpc_merge, tpc_refit_merged, tpc_compress, tpc_rans_encode / _decode over the step's output and tpc_clusterize on one event's digits; outside the timed step"},
            "e2e": {"value": e2e_units / (e2e_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "steps": e2e_steps, "ms_per_step": e2e_max / e2e_steps,
                    "host_threads": T},
            "gpu_launches": trk.launches_per_call() * args.steps,
            "clocks": clk.summary(),
            "roofline": roofline, "roofline_path": roofline_path, "stages": stages, "stage_calls_averaged": n_avg,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line))
    for h in handles:
        h["trk"].close()
    if world > 1:
        dist.destroy_process_group()


def run_reference(args):
    """The oracle as it stands, timed on the host cores: there is no reference implementation for this path (the
    paper publishes no code), so the base contract's reference arm is the oracle.  Rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from gen.events import make_event
    from oracle import oracle
    oracle.build()
    cores = oracle.num_threads()
    # bounded sample: one configs[1] event per step; shrink it if the whole run would exceed ~3 minutes
    total = args.steps + args.warmup
    ev = make_event(CFG_ID)
    t0 = time.perf_counter()
    oracle.track(ev)
    t_ev = time.perf_counter() - t0
    n_tracks = None
    if t_ev * total > 180.0:
        n_tracks = max(50, int(4000 * 180.0 / (t_ev * total)))
        ev = make_event(CFG_ID, n_tracks=n_tracks)
    for _ in range(args.warmup):
        oracle.track(ev)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.track(ev)
    dt = time.perf_counter() - t0
    value = ev.n * args.steps / dt
    sample = (f"one configs[1] event per step ({ev.n} clusters"
              + (f", reduced to {n_tracks} tracks to bound the run" if n_tracks else "") + ")")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int64 / f64", "data": "synthetic",
        "config": {"workload": "configs[1] central Pb-Pb (4000 tracks, 36 sectors, 5% noise)", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_config(args):
    """`--config C`: one event of BASELINE.json configs[C] (30 = the 2 M-cluster reading 3b) per tpc_track call, on one
    stream: the per-config rows of BASELINE.md section 5.  Not the headline (that is configs[1] x 32 events)."""
    import torch
    from gen.events import make_event
    from paper_2502_09138_b200 import Tracker
    from paper_2502_09138_b200.events import geometry_from_event, upload
    ev = make_event(args.config)
    trk = Tracker(geometry_from_event(ev))
    y, z, ro = upload(ev)
    out = trk.alloc_out(ev.n)
    st = torch.cuda.current_stream()
    for _ in range(args.warmup):
        trk.track(y, z, ro, out, st)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for _ in range(args.steps):
        trk.track(y, z, ro, out, st)
    e1.record(st)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    trk.set_stage_timing(True)
    for _ in range(min(args.steps, 8)):
        trk.track(y, z, ro, out, st)
    torch.cuda.synchronize()
    stage_ms, _ = trk.stage_ms_mean()
    tracks, hit_ids, n_seeds = out.to_host()
    _, _, _, nh, _ = trk.debug_tracklets(n_seeds)
    grid = trk.debug_grid(ev.n)
    sb = stage_bytes(float(ev.n), float(grid["stride"]) * trk.n_sectors * trk.n_rows, float(nh.sum()), float(n_seeds))
    hbm_peak, peak_kind, _ = read_peaks()
    gbs = sum(sb.values()) / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": METRIC, "config": {"workload": f"one event of configs[{args.config}] ({ev.cfg.name}) per call"},
                      "value": ev.n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": args.steps,
                      "clusters": ev.n, "seeds": int(n_seeds), "tracks": len(tracks), "tracks_per_s": len(tracks) / (ms * 1e-3),
                      "alg_bytes_per_cluster": sum(sb.values()) / ev.n, "hbm_gbs": gbs, "hbm_frac_measured": gbs / hbm_peak,
                      "hbm_frac_8TBs": gbs / 8000.0, "stage_ms": dict(zip(["a1", "a2", "a3", "a4", "a5"], stage_ms)),
                      "a4_variant": "phases" if trk.launches_per_call() == 12 else "uniform",
                      "scratch_gb": trk.scratch_bytes() / 1e9}))
    trk.close()


def launch_replicas(args):
    """`python bench.py --gpus N` outside torchrun: start N replica ranks of this script (one per GPU, torchrun's
    environment variables, rendezvous on 127.0.0.1) and pass rank 0's JSON line through."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for r in range(args.gpus):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__)] + sys.argv[1:], env=env,
                                      stdout=subprocess.PIPE if r == 0 else subprocess.DEVNULL, text=True))
    out0, _ = procs[0].communicate()
    rcs = [p.wait() for p in procs]
    sys.stdout.write(out0)
    sys.stdout.flush()
    return max(abs(rc) for rc in rcs)


def run_selftest_ranks(args):
    """CPU-only check of the N > 1 plumbing (tests/test_abi_and_host.py): the launcher's environment, the seed
    sharding and the max / sum aggregation, over gloo.  No tracking is done."""
    import torch.distributed as dist
    dist.init_process_group("gloo")
    r, w = dist.get_rank(), dist.get_world_size()
    seeds = shard_seeds(r, w, args.batch_events)
    ms, units = aggregate(10.0 + 5.0 * r, 100.0 * (r + 1), dist, None)
    gathered = [None] * w
    dist.all_gather_object(gathered, seeds)
    if r == 0:
        flat = [x for g in gathered for x in g]
        print(json.dumps({"selftest": "ranks", "n_gpus": w, "ms_max": ms, "units_sum": units,
                          "seeds_distinct": len(set(flat)) == len(flat) == args.batch_events * w}))
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--batch-events", type=int, default=DEFAULT_BATCH_EVENTS)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--streams", type=int, default=0, help="handles/streams of the device arm; 0 = sweep 1..4")
    ap.add_argument("--e2e-threads", type=int, default=8, help="host threads (handles, streams) of the e2e arm")
    ap.add_argument("--selftest-ranks", action="store_true", help="CPU check of the multi-rank plumbing (gloo)")
    ap.add_argument("--a2-variant", type=int, default=0, help="0 = direct a2 (default), 1 = TMA-staged rows (evidence run)")
    ap.add_argument("--config", type=int, default=None, choices=[0, 1, 2, 3, 30, 4],
                    help="time one event of that config per call instead of the headline batch (BASELINE.md section 5)")
    ap.add_argument("--profile", action="store_true", help="only W + K tpc_track calls on one stream (for ncu)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:   # not under torchrun: start the replica ranks here
        sys.exit(launch_replicas(args))
    if args.selftest_ranks:
        run_selftest_ranks(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.config is not None:
        run_config(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
