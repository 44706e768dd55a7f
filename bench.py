#!/usr/bin/env python
"""bench.py — VELO events/s on B200 for the nu=6, 10k-event batch (BASELINE.json metric), with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--events 10000] [--impl ours|reference]
    python bench.py --sweep            # BASELINE.json configs[4] (500 / 2 000 / 10 000 / 50 000 events at nu = 6) and
                                       # configs[3] (nu = 12, 10 000 events): one JSON line per point, the headline last
    python bench.py --paper-protocol   # e2e as the paper measures: 12 streams x 1000-event chunks, 100
                                       # repetitions, mean +- sigma over 10 different event sets

A "step" is one pass of the whole hot path (allen_velo_reconstruct: decode -> cluster -> phi sort -> search by triplet
-> fit -> compaction) over one batch of synthetic events.  `value` is events/s with inputs resident in
HBM; `e2e` is the same metric through the C ABI with HOST buffers (pinned), H2D of the raw banks and D2H of the tracks
inside the timed region.  N > 1 (torchrun): one process per GPU, each reconstructs its own batch (events are
independent: replicas, no collective on the data path); time = max over ranks, value = all events / time.
`--impl reference` times the CPU oracle (test infrastructure) on the host cores on a bounded sample per step.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "velo_events_per_s"
UNIT = "events/s"


def env_int(name, default):
    return int(os.environ.get(name, default))


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def source_hash():
    """Hash of the CUDA sources the library is built from: the committed ncu counters name the sources they were taken
    with, and are not used for any other (the GPU box has the sources, not the git history)."""
    import glob
    import hashlib

    h = hashlib.sha256()
    for path in sorted(glob.glob(os.path.join(ROOT, "paper_1912_09161_b200", "csrc", "*"))):
        h.update(os.path.basename(path).encode())
        with open(path, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_counters(workload_key):
    """Per-kernel counters of one launch from the newest profiles/*_counters.csv (written from an `ncu --set full`
    capture of this very command; the file names the command).  Only rows whose `source_hash` equals the hash of the
    sources in the tree are used: counters of other sources would divide a stale count by a fresh time."""
    import csv
    import glob

    out = {}
    want = source_hash()
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_counters.csv"))):
        with open(path) as f:
            for row in csv.DictReader(f):
                if row.get("workload") == workload_key and row.get("source_hash") == want:
                    out[row["kernel"]] = dict(dram_bytes=int(row["dram_read_bytes"]) + int(row["dram_write_bytes"]),
                                              warp_instructions=int(row["warp_instructions"]),
                                              lanes=float(row["active_lanes_per_instruction"]))
                    out["_source"] = os.path.relpath(path, ROOT)
    return out


class ClockSampler:
    """nvidia-smi clocks/throttle-reason sampler running beside the timed region (B200_PROFILING.md recipe)."""

    FIELDS = ("timestamp,index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index: int):
        self.path = tempfile.mktemp(prefix="clocks_", suffix=".csv")
        self.proc = None
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                                          "-lms", "50", "-i", str(device_index)], stdout=self.f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self, windows):
        """windows: list of (t0, t1) wall-clock intervals (time.time()) to keep samples from."""
        import datetime

        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.proc is None:
            return out
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        rows = []
        try:
            with open(self.path) as f:
                for line in f:
                    p = [x.strip() for x in line.split(",")]
                    if len(p) < 10:
                        continue
                    try:
                        ts = datetime.datetime.strptime(p[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                        rows.append((ts, float(p[2]), float(p[3]), p[5:10]))
                    except Exception:
                        continue
            os.unlink(self.path)
        except Exception:
            return out
        sel = [r for r in rows if any(t0 - 0.05 <= r[0] <= t1 + 0.05 for t0, t1 in windows)] or rows
        if not sel:
            return out
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = set()
        for r in sel:
            for name, v in zip(names, r[3][1:]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        out.update(sm_mhz=statistics.median(r[1] for r in sel), sm_max_mhz=max(r[2] for r in sel),
                   reasons=sorted(reasons), samples=len(sel))
        return out


def algorithmic_bytes(n_events, n_layers, raw_bytes, n_clusters, n_tracks, n_track_hits):
    """Compulsory traffic of one step, exact from the array lengths."""
    raw = raw_bytes + 4 * (n_events + 1)
    clusters = 30 * n_clusters + 4 * (n_events * n_layers + 1) + 4 * (n_events + 1) + 4 * n_events
    tracks = 4 * (n_events + 1) + 4 * (n_tracks + 1) + 2 * n_track_hits + 16 * n_tracks
    return dict(raw=raw, clusters=clusters, tracks=tracks, total=raw + clusters + tracks,
                # per-kernel shares: each compulsory byte is charged to the kernel that moves it.  The
                # cluster kernel reads the raw banks; the seed kernel writes the compacted clusters (it carries that
                # compaction); follow + compact_tracks write the tracks.  The slab, the candidate lists and the
                # forwarding windows between them are overhead, not algorithmic traffic.
                velo_cluster=raw, velo_seed=clusters, velo_follow=tracks, compact_tracks=tracks)


def run_reference(args):
    """The oracle as it stands on the host cores; each step = a bounded sample of the workload."""
    rank = env_int("RANK", 0)
    if rank != 0:
        return 0
    import oracle
    from paper_1912_09161_b200 import workload

    cores = os.cpu_count() or 1
    sample = min(args.events, args.reference_events)
    batch = workload.generate(args.config, n_events=sample)
    for _ in range(args.warmup):
        oracle.reconstruct(batch.geometry, batch.raw, batch.event_offsets, n_threads=cores, export=False)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.reconstruct(batch.geometry, batch.raw, batch.event_offsets, n_threads=cores, export=False)
    dt = time.perf_counter() - t0
    value = sample * args.steps / dt
    line = dict(metric=METRIC, value=value, unit=UNIT, impl="reference", n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * dt / args.steps, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f32", data="synthetic",
                config=dict(workload=f"config{args.config}: first {sample} events of the nu={'12' if args.config == 3 else '6'} batch",
                            events_per_step=sample, input_sha=batch.sha()),
                cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle",
                                  sample=f"{sample} events per step, {cores} threads over contiguous event ranges"),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line, default=float))
    return 0


def measure_ours(args, headline=True):
    """One measurement of the hot path on args.config / args.events.  headline=False (points of --sweep): no single-call
    e2e, no CPU baseline, no near-cut comparison.  Returns the JSON line as a dict (None on ranks other than 0)."""
    import torch

    from paper_1912_09161_b200 import binding, workload

    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=device)

    from paper_1912_09161_b200 import replicas

    red = replicas.Reducer(device)
    barrier, max_over_ranks, sum_over_ranks = red.barrier, red.max, red.sum

    # ---- workload: every rank reconstructs its own batch (batch_index = rank)
    t_gen = time.time()
    batch = workload.generate(args.config, n_events=args.events, batch_index=replicas.batch_index_of(rank))
    t_gen = time.time() - t_gen
    geo = batch.geometry
    n_events, L = batch.n_events, geo.n_layers
    raw_bytes = int(batch.raw.size)
    n_sp = batch.n_sp_words()

    velo = binding.AllenVelo(geo)
    ccap = int(1.15 * n_sp) + 4096
    oc, ot = binding.alloc_outputs(n_events, L, ccap, ccap // 3, ccap // 2, device, with_checksum=False,
                                   with_kalman=args.with_kalman or args.with_vertices)
    if args.with_vertices:
        d_nv = torch.zeros(n_events, dtype=torch.int32, device=device)
        d_pv = torch.zeros((n_events, 32, 8), dtype=torch.float32, device=device)
        velo.set_vertex_output(d_nv, d_pv)
    ws = torch.empty(velo.workspace_bytes(n_events, raw_bytes), dtype=torch.uint8, device=device)
    velo.set_workspace(ws)
    velo.set_occupancy_hint(n_events, raw_bytes)
    h_raw = torch.from_numpy(batch.raw).pin_memory()
    h_off = torch.from_numpy(batch.event_offsets.view(np.int32)).pin_memory()
    d_raw = h_raw.to(device)
    d_off = h_off.to(device)
    stream = torch.cuda.current_stream()

    def step():
        rc = velo.reconstruct(d_raw, d_off, n_events, stream, oc, ot)
        if rc != 0:
            raise RuntimeError(f"allen_velo_reconstruct -> {rc}: {velo.last_error()}")

    sampler = ClockSampler(local) if rank == 0 else None
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    status = oc.status.cpu().numpy().view(np.uint32)
    n_clusters = int(oc.event_offsets.cpu().numpy().view(np.uint32)[n_events])
    te = ot.event_offsets.cpu().numpy().view(np.uint32)
    n_tracks = int(te[n_events])
    n_track_hits = int(ot.hit_offsets.cpu().numpy().view(np.uint32)[n_tracks])
    if status.any():
        raise RuntimeError(f"status bits set on {int((status != 0).sum())} events: {np.unique(status)} (capacity?)")

    # ---- device-resident timing: exactly K steps between barriers + synchronize, CUDA events on the launch stream
    velo.enable_timing(args.steps)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    w0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    w1 = time.time()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = velo.last_launch_count() * args.steps
    kt = np.stack([velo.kernel_times(i) for i in range(args.steps)])  # [steps, kernels]
    velo.enable_timing(0)
    ms_step = max_over_ranks(ms_total / args.steps)
    total_events = sum_over_ranks(float(n_events))
    value = total_events / (ms_step * 1e-3)

    # ---- end to end through the public API with host buffers: H2D raw + offsets, reconstruct, D2H tracks
    h_te = torch.empty(n_events + 1, dtype=torch.int32).pin_memory()
    h_ce = torch.empty(n_events + 1, dtype=torch.int32).pin_memory()
    h_st = torch.empty(n_events, dtype=torch.int32).pin_memory()
    h_ho = torch.empty(ot.capacity_tracks + 1, dtype=torch.int32).pin_memory()
    h_hits = torch.empty(ot.capacity_hits, dtype=torch.int16).pin_memory()
    h_fit = [torch.empty(ot.capacity_tracks, dtype=torch.float32).pin_memory() for _ in range(4)]
    d_raw2, d_off2 = torch.empty_like(d_raw), torch.empty_like(d_off)
    h2d = raw_bytes + 4 * (n_events + 1)
    d2h_holder = [0]

    def e2e_step():
        d_raw2.copy_(h_raw, non_blocking=True)
        d_off2.copy_(h_off, non_blocking=True)
        rc = velo.reconstruct(d_raw2, d_off2, n_events, stream, oc, ot)
        if rc != 0:
            raise RuntimeError(f"allen_velo_reconstruct -> {rc}: {velo.last_error()}")
        h_te.copy_(ot.event_offsets, non_blocking=True)
        h_ce.copy_(oc.event_offsets, non_blocking=True)
        h_st.copy_(oc.status, non_blocking=True)
        stream.synchronize()  # the sizes of the result are needed on the host to fetch exactly the tracks
        nt = int(h_te[n_events])
        h_ho[:nt + 1].copy_(ot.hit_offsets[:nt + 1], non_blocking=True)
        for hbuf, dbuf in zip(h_fit, (ot.x0, ot.y0, ot.tx, ot.ty)):
            hbuf[:nt].copy_(dbuf[:nt], non_blocking=True)
        nh = n_track_hits  # identical input every step; avoids a third round trip
        h_hits[:nh].copy_(ot.hits[:nh], non_blocking=True)
        stream.synchronize()
        d2h_holder[0] = 4 * (n_events + 1) * 2 + 4 * n_events + 4 * (nt + 1) + 16 * nt + 2 * nh

    e0 = e1 = time.time()
    single_ms = single_value = None
    if headline:
        for _ in range(2):
            e2e_step()
        barrier()
        torch.cuda.synchronize()
        e0 = time.time()
        for _ in range(args.steps):
            e2e_step()
        torch.cuda.synchronize()
        e1 = time.time()
        barrier()
        single_ms = max_over_ranks((e1 - e0) * 1e3 / args.steps)
        single_value = total_events / (single_ms * 1e-3)

    # ---- the same, streamed: chunks of the batch on several streams so that copies and kernels overlap
    paper = None
    if headline and args.paper_protocol and world == 1:
        paper = paper_protocol(args, geo, device)
    chunk = min(args.e2e_chunk, n_events)
    chunk_raw = int(1.25 * raw_bytes * chunk / n_events) + (1 << 20)
    sv = binding.StreamedVelo(geo, chunk, chunk_raw, n_streams=args.e2e_streams, device=device)
    off64 = batch.event_offsets.astype(np.int64)
    first_chunk = [min(args.e2e_first_chunk, chunk)] if args.e2e_first_chunk > 0 and n_events > chunk else None
    for _ in range(2):
        infos = sv.reconstruct(h_raw, off64, chunk_sizes=first_chunk)
    if sum(i["n_tracks"] for i in infos) != n_tracks:
        raise RuntimeError("streamed reconstruction found a different number of tracks")
    barrier()
    torch.cuda.synchronize()
    e2 = time.time()
    for _ in range(args.steps):
        sv.reconstruct(h_raw, off64, chunk_sizes=first_chunk)
    torch.cuda.synchronize()
    e3 = time.time()
    barrier()
    e2e_ms = max_over_ranks((e3 - e2) * 1e3 / args.steps)
    e2e_value = total_events / (e2e_ms * 1e-3)
    h2d, d2h_holder[0] = sv.h2d_bytes, sv.d2h_bytes
    sv.destroy()

    clocks = sampler.stop([(w0, w1), (e0, e1), (e2, e3)]) if sampler else None

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return None

    # ---- roofline of the dominant kernel (own algorithmic bytes / own mean duration) and of the whole path
    names = velo.kernel_names()
    mean_ms = kt.mean(axis=0)
    dom = int(np.argmax(mean_ms))
    ab = algorithmic_bytes(n_events, L, raw_bytes, n_clusters, n_tracks, n_track_hits)
    peak, peak_src = peaks()
    dom_bytes = ab.get(names[dom], 0)
    achieved = dom_bytes / (mean_ms[dom] * 1e-3) / 1e9
    # DRAM traffic and instruction counts of the same launch configuration, from the committed ncu capture
    counters = ncu_counters(f"config{args.config}_{n_events}")
    traffic = counters.get(names[dom], {}).get("dram_bytes")
    roofline = dict(bound="hbm", kernel=names[dom], achieved=achieved, peak=peak, unit="GB/s", frac=achieved / peak,
                    traffic=traffic, peak_source=peak_src, algorithmic_bytes_per_launch=dom_bytes,
                    kernel_ms=float(mean_ms[dom]), kernel_share_of_step=float(mean_ms[dom] / mean_ms.sum()),
                    traffic_source=counters.get("_source"))
    # why the HBM fraction is low: the path is bound by instruction issue, not by memory
    issue_peak = 148 * 4 * (clocks or {}).get("sm_mhz", 1965.0) * 1e6 if clocks and clocks.get("sm_mhz") else 148 * 4 * 1.965e9
    roofline_issue = None
    if names[dom] in counters and counters[names[dom]].get("warp_instructions"):
        wi = counters[names[dom]]["warp_instructions"]
        roofline_issue = dict(bound="alu", kernel=names[dom], achieved=wi / (mean_ms[dom] * 1e-3) / 1e9,
                              peak=issue_peak / 1e9, unit="G warp-instr/s", frac=wi / (mean_ms[dom] * 1e-3) / issue_peak,
                              warp_instructions_per_launch=wi, active_lanes_per_instruction=counters[names[dom]].get("lanes"),
                              source=counters.get("_source"))
    path_gbs = ab["total"] / (ms_step * 1e-3) / 1e9
    roofline_path = dict(bound="hbm", achieved=path_gbs, peak=peak, unit="GB/s", frac=path_gbs / peak,
                         frac_of_8TBs_nominal=path_gbs / 8000.0, algorithmic_bytes_per_step=ab["total"],
                         bytes_per_event=ab["total"] / n_events)

    cpu_baseline = near_cut = None
    if headline and world == 1 and not args.no_cpu_baseline:
        import oracle

        cores = os.cpu_count() or 1
        n1 = min(n_events, args.cpu_events_single)
        sub = batch.select(np.arange(n1))
        t0 = time.perf_counter()
        oracle.reconstruct(geo, sub.raw, sub.event_offsets, n_threads=1, export=False)
        single = n1 / (time.perf_counter() - t0)
        nm = min(n_events, args.cpu_events_multi)
        subm = batch.select(np.arange(nm))
        t0 = time.perf_counter()
        oracle.reconstruct(geo, subm.raw, subm.event_offsets, n_threads=cores, export=False)
        multi = nm / (time.perf_counter() - t0)
        cpu_baseline = dict(value=multi, unit=UNIT, cores=cores, kind="oracle (a plain, unoptimised restatement of the "
                            "paper's definitions: linear window scans, no phi look-up; a reported baseline, not a target)",
                            sample=f"first {nm} events of the same batch on {cores} threads (contiguous ranges); "
                                   f"single thread over the first {n1} events: {single:.1f} events/s",
                            single_thread_value=single)
        # near-cut accounting (BASELINE.json: "counted and reported"): the oracle's log over the same sample, and the
        # tracks of the timed batch that differ from the oracle's on it (outside the timed regions)
        ref = oracle.reconstruct(geo, subm.raw, subm.event_offsets, n_threads=cores)
        rt = ref.tracks
        g_ho = ot.hit_offsets.cpu().numpy().view(np.uint32)
        g_hits = ot.hits.cpu().numpy().view(np.uint16)
        t1 = int(te[nm])
        same = (np.array_equal(te[:nm + 1], rt.event_offsets) and np.array_equal(g_ho[:t1 + 1], rt.hit_offsets)
                and np.array_equal(g_hits[:int(g_ho[t1])], rt.hits))
        mismatched = 0
        if not same:
            for e in range(nm):
                got = {tuple(sorted(g_hits[g_ho[t]:g_ho[t + 1]].tolist())) for t in range(int(te[e]), int(te[e + 1]))}
                want = set(rt.hit_sets(e))
                mismatched += len(got ^ want)
        near_cut = dict(events=nm, tracks=int(rt.event_offsets[-1]), near_cut_decisions=int(ref.near_cut_per_event.sum()),
                        events_with_near_cut_decisions=int((ref.near_cut_per_event > 0).sum()),
                        near_cut_mismatches=mismatched, identical_hit_lists_and_order=bool(same))

    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
        ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
        config=dict(workload=f"config{args.config}: {n_events} events/GPU at nu={'12' if args.config == 3 else '6'} "
                             f"(BASELINE.json configs[{args.config}])",
                    events_per_gpu=n_events, parallelism=f"replicas x{world} (events independent, no collective)", kalman_fit=bool(args.with_kalman or args.with_vertices), vertices=bool(args.with_vertices),
                    l2_policy="inputs+outputs per step (%.0f MB) larger than the 126 MB L2" % (ab["total"] / 1e6),
                    input_sha=batch.sha(), sp_words_per_event=n_sp / n_events, clusters_per_event=n_clusters / n_events,
                    tracks_per_event=n_tracks / n_events, hits_per_track=n_track_hits / max(1, n_tracks),
                    raw_bytes_per_event=raw_bytes / n_events, generator_s=round(t_gen, 2)),
        e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h_holder[0],
                 ms_per_step=e2e_ms, how=f"binding.StreamedVelo: chunks of {chunk} events "
                                         f"{'(the first one ' + str(first_chunk[0]) + ') ' if first_chunk else ''}on {args.e2e_streams} streams, "
                                         "pinned host buffers, H2D raw + offsets and D2H tracks inside the timed region; "
                                         "the clusters stay on the device (P:132: only tracks and vertices are copied back)",
                 single_call=dict(value=single_value, ms_per_step=single_ms) if single_ms else None,
                 paper_protocol=paper),
        gpu_launches=launches,
        kernels={n: float(m) for n, m in zip(names, mean_ms)},
        roofline=roofline, roofline_path=roofline_path, roofline_issue=roofline_issue, cpu_baseline=cpu_baseline,
        near_cut=near_cut, clocks=clocks, source_hash=source_hash(),
    )
    if dist is not None:
        dist.destroy_process_group()
    return line


def paper_protocol(args, geo, device):
    """The paper's own throughput protocol: 12 host-thread/stream pairs with 1000 events each, processed 100
    times, for 10 different sets of events; mean and standard deviation over the sets.  Here: binding.StreamedVelo with
    12 streams and 1000-event chunks over a 12 000-event batch (every stream one chunk per repetition), H2D of the raw
    banks and D2H of the tracks inside the timed region, wall clock from the first launch to the last stream's return."""
    import torch

    from paper_1912_09161_b200 import binding, workload

    n_streams, chunk, reps, n_sets = 12, 1000, args.paper_reps, args.paper_sets
    values = []
    sv = None
    for k in range(n_sets):
        batch = workload.generate(args.config, n_events=n_streams * chunk, batch_index=100 + k)
        if sv is None:
            sv = binding.StreamedVelo(geo, chunk, int(1.3 * batch.raw.size / n_streams) + (1 << 20), n_streams=n_streams,
                                      device=device)
        h_raw = torch.from_numpy(batch.raw).pin_memory()
        off64 = batch.event_offsets.astype(np.int64)
        sv.reconstruct(h_raw, off64)
        torch.cuda.synchronize()
        t0 = time.time()
        for _ in range(reps):
            sv.reconstruct(h_raw, off64)
        torch.cuda.synchronize()
        values.append(batch.n_events * reps / (time.time() - t0))
    sv.destroy()
    return dict(value=float(np.mean(values)), sigma=float(np.std(values)), unit=UNIT, streams=n_streams, events_per_stream=chunk,
                repetitions=reps, event_sets=n_sets, per_set=[float(v) for v in values],
                how="P:277-279 with binding.StreamedVelo; copies inside the timed region, clusters stay on the device")


def run_ours(args):
    import copy

    if args.sweep:
        if env_int("WORLD_SIZE", 1) != 1:
            raise RuntimeError("--sweep is a single-GPU measurement")
        for config, events in ((2, 500), (2, 2000), (2, 50000), (3, 10000)):
            a = copy.copy(args)
            a.config, a.events = config, events
            line = measure_ours(a, headline=False)
            line["sweep_point"] = True
            print(json.dumps(line, default=float), flush=True)
            import gc

            import torch

            del line
            gc.collect()
            torch.cuda.empty_cache()
    line = measure_ours(args, headline=True)
    if line is not None:
        print(json.dumps(line, default=float))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[0, 1, 2, 3])
    ap.add_argument("--events", type=int, default=10000)
    ap.add_argument("--reference-events", type=int, default=2000, help="events per step of the reference arm")
    ap.add_argument("--cpu-events-single", type=int, default=1000)
    ap.add_argument("--cpu-events-multi", type=int, default=4000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--with-kalman", action="store_true",
                    help="also produce the simple Kalman fit (SURVEY 8(f1), beyond the headline path; +48 B per track)")
    ap.add_argument("--with-vertices", action="store_true",
                    help="also find primary vertices (SURVEY 8(f2), beyond the headline path; implies --with-kalman)")
    ap.add_argument("--e2e-chunk", type=int, default=3000, help="events per chunk of the streamed end-to-end run")
    ap.add_argument("--e2e-first-chunk", type=int, default=1000,
                    help="events of the first chunk when the batch needs several (gets the GPU started early); 0 = e2e-chunk")
    ap.add_argument("--e2e-streams", type=int, default=4)
    ap.add_argument("--sweep", action="store_true",
                    help="also measure BASELINE.json configs[4] (500 / 2k / 50k events) and configs[3] (nu = 12): one line each, "
                         "the headline line last")
    ap.add_argument("--paper-protocol", action="store_true",
                    help="add e2e.paper_protocol: 12 streams x 1000-event chunks, repeated, mean +- sigma over event sets (P:277-279)")
    ap.add_argument("--paper-reps", type=int, default=100)
    ap.add_argument("--paper-sets", type=int, default=10)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
