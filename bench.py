"""bench.py -- events/s and digis/s of the Clusters chain on B200, with its HBM roofline fraction.

    python bench.py --gpus 1 --steps 10 --warmup 3            # this repo's CUDA path
    python bench.py --impl reference --steps 3 --warmup 1     # the oracle on the host cores (the reference arm)
A step = one pass of the whole hot path (init; runs = module boundaries + work items; the tile kernel = unpack +
calibrate + cluster + cut + renumber; the block-per-run kernel for the runs it leaves; finalize = offsets + scatter)
over one batch of synthetic events: BASELINE.json configs[2], 1000 PU50-like events (config[1]'s
generator, seeds 0..999), through pix_process_batch.  `value` is timed with the inputs resident in HBM; `e2e`
goes through pix_process_batch_host with pinned HOST buffers, host<->device copies inside the timed region.
Under torchrun (N > 1) every rank runs its own 1000 events (seeds rank*1000 ..): weak scaling, no collective
on the data path; the time is the max over ranks.
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

import pixgen  # noqa: E402

PARAMS = dict(pixgen.DEFAULT_PARAMS)
WORKLOAD = "cfg2: 1000 PU50-like events (1856 modules, ~60.6k words/event), pix_process_batch"


def peak_hbm():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.first = [], None, 0
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def mark(self, timeout=2.0):
        """Waits until nvidia-smi delivers rows, then marks the start of the region of interest."""
        t0 = time.perf_counter()
        while self.proc and not self.rows and time.perf_counter() - t0 < timeout:
            time.sleep(0.005)
        self.first = len(self.rows)

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        if len(self.rows) > self.first:
            self.rows = self.rows[self.first:]  # samples taken after mark(): under load
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def shard_seeds(n_events: int, rank: int):
    """Event seeds of one rank: events are independent, so the path shards by events with no
    data-path collective; rank r takes seeds r*1000 .. r*1000 + n_events - 1 (weak scaling)."""
    return rank * 1000 + np.arange(n_events)


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """The step time of the job is the slowest rank's (one scalar all_reduce(MAX), outside the timed region)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def generate(n_events: int, rank: int):
    det = pixgen.detector("full")
    batch = pixgen.events(det, "pu50", shard_seeds(n_events, rank), cap_words_per_event=1 << 17)
    return det, batch


def algorithmic_bytes(W, K, M, E):
    """bytes(event) = 19 W + 22 K + 12 M + 68, summed over the batch."""
    return 19 * W + 22 * K + (12 * M + 68) * E


# ---------------------------------------------------------------------------------------------- reference arm
def run_reference(args):
    """The oracle, as it stands, single-threaded on the host cores, on the same workload (bounded sample per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    n_sample = min(args.ref_events, args.events)
    det, batch = generate(n_sample, 0)
    sizes = np.diff(batch.event_offsets.astype(np.int64))

    def step():
        for e in range(n_sample):
            oracle.process(det, *batch.event(e), PARAMS, max_clusters_per_event=int(sizes[e]))

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    v = n_sample / dt
    line = {"impl": "reference", "metric": "events/s", "value": v, "unit": "events/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32+f32", "data": "synthetic",
            "digis_per_s": float(sizes.sum()) / dt,
            "config": {"workload": WORKLOAD, "sample": f"first {n_sample} events of the batch per step"},
            "cpu_baseline": {"value": v, "unit": "events/s", "cores": 1, "kind": "oracle",
                             "sample": f"first {n_sample} events of cfg2 per step, {args.steps} steps"},
            "e2e": {"value": v, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------- graph-per-event mode
def run_graph_per_event(pix, torch, det, batch, dev, kmax, n_streams=8):
    """BASELINE.json configs[2] as written: every event is one CUDA-graph launch (pix_process captured once per
    event), round-robin over 8 streams with one cloned handle each.  Secondary number: the launch rate binds it.
    Returns (events/s, dict of outputs) with events laid out at 16-word-aligned offsets."""
    E, M, F = batch.n_events, det.n_modules, det.n_feds
    sizes = np.diff(batch.event_offsets.astype(np.int64))
    poff = np.concatenate([[0], np.cumsum((sizes + 15) // 16 * 16)]).astype(np.int64)
    wp = np.zeros(int(poff[-1]) + 16, np.uint32)
    for e in range(E):
        a = int(batch.event_offsets[e])
        wp[poff[e]:poff[e] + sizes[e]] = batch.words[a:a + sizes[e]]
    words = torch.from_numpy(wp.view(np.int32)).to(dev)
    fed_off = torch.from_numpy(batch.fed_offsets.view(np.int32).reshape(-1).copy()).to(dev)
    digis, clusters = pix.alloc_outputs(int(poff[-1]), E, M, kmax, dev)
    wmax = (int(sizes.max()) + 1023) // 1024 * 1024
    h0 = pix.pix_create(det.cabling, F, M, det.gain, det.pedestal, pix.make_params(PARAMS, wmax, kmax, 1, 1))
    handles = [h0] + [pix.pix_clone(h0) for _ in range(n_streams - 1)]
    streams = [torch.cuda.Stream(dev) for _ in range(n_streams)]
    strides = dict(module=kmax, first_digi=kmax, n_pix=kmax, charge=kmax, x_col=kmax, y_row=kmax, module_first=M,
                   module_end=M, clus_module_start=M + 1, summary=16)

    def call(e, s):
        d = {k: v[int(poff[e]):] for k, v in digis.items()}
        c = {k: v[e * strides[k]:] for k, v in clusters.items()}
        pix.pix_process(handles[e % n_streams], s, words[int(poff[e]):], fed_off[e * (F + 1):], int(sizes[e]), d, c)

    for e in range(min(E, n_streams)):  # warm-up outside capture
        call(e, streams[e % n_streams])
    torch.cuda.synchronize()
    graphs = []
    for e in range(E):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=streams[e % n_streams]):
            call(e, streams[e % n_streams])
        graphs.append(g)
    torch.cuda.synchronize()

    def replay_all():
        for e, g in enumerate(graphs):
            with torch.cuda.stream(streams[e % n_streams]):
                g.replay()

    replay_all()
    torch.cuda.synchronize()
    start = torch.cuda.Event(enable_timing=True)
    ends = [torch.cuda.Event(enable_timing=True) for _ in streams]
    start.record(streams[0])
    for s in streams[1:]:
        s.wait_event(start)
    replay_all()
    for s, ev in zip(streams, ends):
        ev.record(s)
    torch.cuda.synchronize()
    ms = max(start.elapsed_time(ev) for ev in ends)
    out = {"clus": digis["clus"], "status": digis["status"], "summary": clusters["summary"], "poff": poff}
    for hh in handles:
        pix.pix_destroy(hh)
    return E / (ms * 1e-3), ms, out


# ---------------------------------------------------------------------------------------------- this repo's arm
def kernel_source_hash():
    """Hash of the CUDA sources: profiles/traffic.json is stamped with it, so a capture taken from other kernel code
    is reported as stale instead of being divided by a live duration."""
    import hashlib
    d = os.path.join(ROOT, "paper_2104_06573_b200", "csrc")
    hsh = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            hsh.update(f.encode()); hsh.update(open(os.path.join(d, f), "rb").read())
    return hsh.hexdigest()[:16]


def timed_passes(torch, stream, fn, n_pass):
    """n_pass single passes, each between its own pair of CUDA events on the launch stream -> list of ms."""
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_pass)]
    for a, b in evs:
        a.record(stream); fn(); b.record(stream)
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


def oracle_baseline(det, batch, sizes, n_events, budget_s=10.0):
    """The oracle as it stands on the host cores, same events: (1) one thread, (2) one event per thread on all cores
    (the paper's own CPU strategy).  ctypes releases the GIL during the call, so plain threads do."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    ns = min(n_events, batch.n_events)

    def one(e):
        oracle.process(det, *batch.event(e), PARAMS, max_clusters_per_event=int(sizes[e]))

    t0 = time.perf_counter(); passes = 0
    while passes == 0 or (time.perf_counter() - t0 < budget_s and passes < 50):
        for e in range(ns):
            one(e)
        passes += 1
    dt1 = time.perf_counter() - t0
    cores = os.cpu_count() or 1
    with ThreadPoolExecutor(max_workers=cores) as ex:
        list(ex.map(one, range(min(ns, cores))))  # start the threads
        t0 = time.perf_counter(); passes_n = 0
        while passes_n == 0 or (time.perf_counter() - t0 < budget_s and passes_n < 200):
            list(ex.map(one, range(ns), chunksize=max(1, ns // (cores * 8))))
            passes_n += 1
        dtn = time.perf_counter() - t0
    wsum = float(sizes[:ns].sum())
    return {"value": ns * passes / dt1, "unit": "events/s", "cores": 1, "kind": "oracle",
            "sample": f"first {ns} events of the same batch x {passes} passes, single thread, {dt1:.1f} s",
            "digis_per_s": wsum * passes / dt1,
            "all_cores": {"value": ns * passes_n / dtn, "unit": "events/s", "cores": cores, "digis_per_s": wsum * passes_n / dtn,
                          "sample": f"same {ns} events x {passes_n} passes, one event per thread, {dtn:.1f} s"}}


def run_ours(args):
    import torch
    import paper_2104_06573_b200 as pix

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    E = args.events
    det, batch = generate(E, rank)
    M, F = det.n_modules, det.n_feds
    sizes = np.diff(batch.event_offsets.astype(np.int64))
    W = int(sizes.sum())
    wmax = (int(sizes.max()) + 1023) // 1024 * 1024
    kmax = args.max_clusters
    params = pix.make_params(PARAMS, wmax, kmax, E, args.chunk_events)
    h = pix.pix_create(det.cabling, F, M, det.gain, det.pedestal, params)

    dev = torch.device("cuda", local)
    pad = np.zeros(16, np.uint32)
    words_h = torch.from_numpy(np.concatenate([batch.words, pad]).view(np.int32)).pin_memory()
    evoff_h = torch.from_numpy(batch.event_offsets.view(np.int32).copy()).pin_memory()
    fedoff_h = torch.from_numpy(batch.fed_offsets.view(np.int32).reshape(-1).copy()).pin_memory()
    words, ev_off, fed_off = words_h.to(dev), evoff_h.to(dev), fedoff_h.to(dev)
    digis, clusters = pix.alloc_outputs(W, E, M, kmax, dev)
    stream = torch.cuda.Stream(dev)

    def step():
        pix.pix_process_batch(h, stream, E, words, W, ev_off, fed_off, digis, clusters)

    # ---- device-resident timing: W warm-up steps, then exactly K steps between CUDA events on the launch stream.
    # Inputs (242 MB) + outputs (~1.3 GB) per step exceed the 126 MB L2, so no explicit flush is needed.
    sampler = ClockSampler(local) if rank == 0 else None  # started early: nvidia-smi needs ~0.1 s to deliver rows
    for _ in range(args.warmup):
        step()
    if sampler:
        sampler.mark()  # rows from here on are taken under load (timed steps + their per-kernel repeat)
    barrier()
    n0 = pix.pix_kernel_launches(h)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1) / args.steps
    launches = pix.pix_kernel_launches(h) - n0
    ms = max_over_ranks(ms, dist, dev)
    # ---- the same step again as single passes (at least 5 timed passes, median and best)
    passes = timed_passes(torch, stream, step, max(5, args.steps))

    # ---- per-kernel device time (CUDA events between the kernels, on the launch stream), same steps again
    pix.pix_set_profiling(h, True)
    for _ in range(args.steps):
        step()
    prof, n_chunks = pix.pix_read_profile(h)
    pix.pix_set_profiling(h, False)
    prof = {k: v / args.steps for k, v in prof.items()}  # ms per step, summed over the step's chunks
    clocks = sampler.stop() if sampler else None  # sampled over the timed steps and their per-kernel repeat
    chunks_per_step = n_chunks // args.steps

    # ---- SURVEY 8f NEXT-1, outside the step: RecHits-lite over the step's outputs (CUDA events on the launch stream)
    hits = pix.alloc_hits(E, kmax, dev)
    pix.pix_rechits(h, stream, E, ev_off, digis, clusters, hits)
    rechits_ms = float(np.median(timed_passes(torch, stream, lambda: pix.pix_rechits(h, stream, E, ev_off, digis, clusters, hits), 5)))
    del hits

    # ---- what the step produced (for the byte counts) + a parity spot check against the oracle (rank 0)
    torch.cuda.synchronize()
    summ = clusters["summary"].cpu().numpy().reshape(E, 16).astype(np.int64)
    K = int(summ[:, 14].sum())
    # algorithmic bytes per kernel: the runs pre-pass reads the raw word and writes one bit; the
    # tile kernel reads the raw word and writes the six digi arrays (19 B per word) and the 20 B temp records;
    # finalize moves the records (20 B in, 22 B out) and writes the per-event arrays
    kernel_bytes = {"init": 12 * M * E, "runs": 4 * W + W // 8, "tile": 19 * W + 20 * K, "overflow": 0,
                    "finalize": 42 * K + (4 * (M + 1) + 64 + 4 * M) * E}
    top = max(prof, key=prof.get)
    peak, peak_src = peak_hbm()
    top_launches = chunks_per_step
    top_gbs = kernel_bytes[top] / (prof[top] * 1e-3) / 1e9 if prof[top] > 0 else 0.0
    traffic = winst = None
    traffic_note = "no capture"
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        tj = json.load(open(tp))
        fresh = tj.get("kernel_source_hash") == kernel_source_hash()
        traffic_note = ("fresh" if fresh else "stale") + f": ncu capture at commit {tj.get('commit', '?')}, sources {tj.get('kernel_source_hash', '?')}"
        if fresh and E == 1000:  # captured on the 1000-event launch; a capture of other kernel code is not reported as this run's
            traffic = tj.get("dram_bytes_per_launch", {}).get(top)
            winst = tj.get("warp_instructions_per_launch", {}).get(top)
            chain_traffic = sum(tj.get("dram_bytes_per_launch", {}).values()) or None
        else:
            chain_traffic = None
    else:
        chain_traffic = None
    chain_bytes = algorithmic_bytes(W, K, M, E)
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    sm_max_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
    chain_gbs = chain_bytes / (ms * 1e-3) / 1e9

    parity = None
    if rank == 0 and not args.no_check:
        import oracle
        bad = 0
        for e in (0, E // 2, E - 1):
            o = oracle.process(det, *batch.event(e), PARAMS, max_clusters_per_event=kmax)
            a, b = int(batch.event_offsets[e]), int(batch.event_offsets[e + 1])
            bad += int(not np.array_equal(o["summary"].astype(np.int64), summ[e]))
            for name in ("module", "row", "col", "charge", "clus", "status"):
                bad += int(not np.array_equal(o[name], digis[name][a:b].cpu().numpy()))
            k = len(o["c_charge"])
            for name, key in (("module", "c_module"), ("first_digi", "c_first_digi"), ("n_pix", "c_n_pix"), ("charge", "c_charge")):
                bad += int(not np.array_equal(o[key], clusters[name][e * kmax:e * kmax + k].cpu().numpy()))
            for name, key in (("x_col", "c_x_col"), ("y_row", "c_y_row")):
                bad += int(not np.allclose(o[key], clusters[name][e * kmax:e * kmax + k].cpu().numpy(), rtol=1e-5, atol=0))
        parity = ("ok (3 events, every digi and record array bit-exact, centroids 1e-5; the full comparison is tests/)"
                  if bad == 0 else f"MISMATCH x{bad}")

    # ---- batch-size sweep: the first E' events of the same batch per call
    sweep = None
    if rank == 0 and not args.no_sweep:
        sweep = {}
        for Es in (1, 8, 32, 125, 1000):
            if Es > E:
                continue
            Ws = int(batch.event_offsets[Es])
            fn = lambda: pix.pix_process_batch(h, stream, Es, words, Ws, ev_off, fed_off, digis, clusters)  # noqa: E731
            for _ in range(3):
                fn()
            t = timed_passes(torch, stream, fn, 7)
            sweep[str(Es)] = {"events_per_s_median": Es / (float(np.median(t)) * 1e-3), "events_per_s_best": Es / (min(t) * 1e-3),
                              "ms_median": float(np.median(t))}

    # ---- secondary mode (rank 0): one CUDA-graph launch per event over 8 streams (BASELINE.json configs[2] as written)
    graph_mode = None
    if rank == 0 and not args.no_graph_mode:
        step(); torch.cuda.synchronize()  # the sweep's last call may have been a shorter batch
        gps, gms, gout = run_graph_per_event(pix, torch, det, batch, dev, kmax)
        same = True
        for e in (0, E // 2, E - 1):  # graph replay == batch launch
            a, b = int(batch.event_offsets[e]), int(batch.event_offsets[e + 1])
            pa = int(gout["poff"][e])
            same &= bool(torch.equal(gout["clus"][pa:pa + (b - a)], digis["clus"][a:b]))
            same &= bool(torch.equal(gout["status"][pa:pa + (b - a)], digis["status"][a:b]))
            same &= bool(torch.equal(gout["summary"][e * 16:(e + 1) * 16], clusters["summary"][e * 16:(e + 1) * 16]))
        graph_mode = {"value": gps, "unit": "events/s", "ms_per_1000_events": gms * 1000.0 / E, "streams": 8,
                      "launches": "one CUDA graph (8 kernels) per event", "equals_batch_launch": same}
        del gout

    # ---- end to end: same metric through pix_process_batch_host, pinned host buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hd, hc = pix.alloc_outputs(W, E, M, kmax, "cpu", pinned=True)
        h2d = W * 4 + (E + 1) * 4 + E * (F + 1) * 4

        def host_timing(hdig):
            fn = lambda: pix.pix_process_batch_host(h, stream, E, words_h, W, evoff_h, fedoff_h, hdig, hc)  # noqa: E731
            fn()
            barrier()
            n_e2e = max(1, min(args.steps, 5))
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                fn()  # synchronous: returns after the device->host copies have landed
            torch.cuda.synchronize()
            dt = max_over_ranks((time.perf_counter() - t0) / n_e2e, dist, dev)
            return dt, n_e2e, pix.pix_host_bytes_out(h)

        dt, n_e2e, d2h = host_timing(hd)
        e2e = {"value": E * world / dt, "unit": "events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "ms_per_step": dt * 1e3, "steps": n_e2e, "api": "pix_process_batch_host, every output array requested"}
        dtc, _, d2hc = host_timing({k: None for k in hd})  # clusters only: no digi array travels back
        e2e["clusters_only"] = {"value": E * world / dtc, "unit": "events/s", "h2d_bytes_per_step": h2d,
                                "d2h_bytes_per_step": d2hc, "ms_per_step": dtc * 1e3,
                                "api": "pix_process_batch_host, digi arrays NULL"}
        del hd, hc

    # ---- BASELINE.json configs[3]: 200 PU200-like events through the same call (rank 0)
    pu200 = None
    if rank == 0 and not args.no_pu200:
        pu200 = run_pu200(pix, torch, det, dev, stream, peak)

    # ---- the oracle on this box's host cores (rank 0, N = 1 only), bounded sample
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_baseline(det, batch, sizes, args.ref_events)

    pix.pix_destroy(h)
    if rank == 0:
        line = {
            "metric": "events/s", "value": E * world / (ms * 1e-3), "unit": "events/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32+f32", "data": "synthetic",
            "digis_per_s": W * world / (ms * 1e-3),
            "passes": {"n": len(passes), "ms_median": float(np.median(passes)), "ms_best": min(passes),
                       "events_per_s_median": E / (float(np.median(passes)) * 1e-3), "events_per_s_best": E / (min(passes) * 1e-3)},
            "config": {"workload": WORKLOAD, "events_per_gpu": E, "words_per_step_per_gpu": W, "clusters_per_step_per_gpu": K,
                       "chunk_events": h.params["chunk_events"] or "auto", "chunks_per_step": chunks_per_step,
                       "l2": "inputs+outputs per step (~1.5 GB) exceed the 126 MB L2; no flush"},
            "clocks": clocks, "gpu_launches": int(launches), "e2e": e2e,
            # the chain's algorithmic bytes per step over the step time, against the measured copy bandwidth
            "roofline": {"bound": "hbm", "kernel": "chain (init, segfill, runs, pack, tile, overflow, offsets, scatter)", "achieved": chain_gbs,
                         "peak": peak, "unit": "GB/s", "frac": chain_gbs / peak, "traffic": chain_traffic, "traffic_note": traffic_note,
                         "peak_source": peak_src, "algorithmic_bytes_per_step": chain_bytes, "formula": "19 W + 22 K + (12 M + 68) E"},
            # the dominant kernel by device time: its own algorithmic bytes over its own launch duration
            "roofline_kernel": {"bound": "hbm", "kernel": top, "achieved": top_gbs, "peak": peak, "unit": "GB/s",
                                "frac": top_gbs / peak, "traffic": traffic,
                                "algorithmic_bytes_per_launch": kernel_bytes[top] / max(top_launches, 1),
                                "avg_launch_ms": prof[top] / max(top_launches, 1), "launches_per_step": top_launches},
            # that kernel is bound by instruction issue: warp instructions per launch (ncu, profiles/) over the live launch
            # time, against SMs x 4 schedulers x 1 instruction/clk at the maximum SM clock
            "roofline_issue": (None if not winst or not prof[top] else {
                "bound": "alu", "kernel": top, "achieved": winst / (prof[top] / max(top_launches, 1) * 1e-3) / 1e9,
                "peak": n_sm * 4 * sm_max_mhz * 1e6 / 1e9, "unit": "G warp-instructions/s",
                "frac": winst / (prof[top] / max(top_launches, 1) * 1e-3) / (n_sm * 4 * sm_max_mhz * 1e6),
                "warp_instructions_per_word": winst / W}),
            "kernel_ms_per_step": prof, "kernel_algorithmic_bytes_per_step": kernel_bytes,
            "cpu_baseline": cpu, "parity_spot_check": parity, "sweep": sweep, "pu200": pu200,
            "graph_per_event": graph_mode,
            "next": {"rechits_lite_ms_per_1000_events": rechits_ms * 1000.0 / E, "note": "pix_rechits, not part of the step"},
        }
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def run_pu200(pix, torch, det, dev, stream, peak, n_events=200):
    """BASELINE.json configs[3] (200 PU200-like events, about 250k words each, 2% long clusters) through
    pix_process_batch: events/s, digis/s, chain roofline fraction, per-kernel ms."""
    b = pixgen.events(det, "pu200", np.arange(n_events), cap_words_per_event=1 << 19)
    sizes = np.diff(b.event_offsets.astype(np.int64))
    E, M, F, W = b.n_events, det.n_modules, det.n_feds, int(sizes.sum())
    wmax = (int(sizes.max()) + 1023) // 1024 * 1024
    kmax = 65536
    h = pix.pix_create(det.cabling, F, M, det.gain, det.pedestal, pix.make_params(PARAMS, wmax, kmax, E, 0))
    words = torch.from_numpy(np.concatenate([b.words, np.zeros(16, np.uint32)]).view(np.int32)).to(dev)
    ev_off = torch.from_numpy(b.event_offsets.view(np.int32).copy()).to(dev)
    fed_off = torch.from_numpy(b.fed_offsets.view(np.int32).reshape(-1).copy()).to(dev)
    digis, cl = pix.alloc_outputs(W, E, M, kmax, dev)
    fn = lambda: pix.pix_process_batch(h, stream, E, words, W, ev_off, fed_off, digis, cl)  # noqa: E731
    for _ in range(3):
        fn()
    t = timed_passes(torch, stream, fn, 7)
    pix.pix_set_profiling(h, True)
    for _ in range(3):
        fn()
    prof, _ = pix.pix_read_profile(h)
    pix.pix_set_profiling(h, False)
    torch.cuda.synchronize()
    K = int(cl["summary"].cpu().numpy().reshape(E, 16)[:, 14].astype(np.int64).sum())
    pix.pix_destroy(h)
    msm = float(np.median(t))
    bytes_ = algorithmic_bytes(W, K, M, E)
    return {"workload": "cfg3: 200 PU200-like events, one pix_process_batch call", "events_per_s": E / (msm * 1e-3),
            "events_per_s_best": E / (min(t) * 1e-3), "digis_per_s": W / (msm * 1e-3), "ms_median": msm, "words": W, "clusters": K,
            "roofline_frac": bytes_ / (msm * 1e-3) / 1e9 / peak, "algorithmic_bytes": bytes_,
            "kernel_ms": {k: v / 3 for k, v in prof.items()}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=1000, help="events per step per GPU (cfg2: 1000)")
    ap.add_argument("--chunk-events", type=int, default=0, help="events per internal launch group (0 = library default)")
    ap.add_argument("--max-clusters", type=int, default=20480, help="cluster record capacity per event")
    ap.add_argument("--ref-events", type=int, default=1000, help="events of the oracle sample (cpu_baseline / reference arm)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-check", action="store_true")
    ap.add_argument("--no-graph-mode", action="store_true", help="skip the one-graph-per-event secondary measurement")
    ap.add_argument("--no-sweep", action="store_true", help="skip the batch-size sweep")
    ap.add_argument("--no-pu200", action="store_true", help="skip the PU200 (configs[3]) measurement")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
