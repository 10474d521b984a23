#!/usr/bin/env python
"""bench.py -- throughput of the TPC sector tracker (a1..a5 in one tpcRun) on synthetic time frames.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (grid, neighbour finder, cleaner + start hits, tracklet
constructor, selector) over one synthetic event.  At N=1 the workload is BASELINE.json configs[4] (the
200-collision time frame the north_star quotes its target on); with N>1 every rank tracks its own
time frame (different seed), no data-path collective ("replicas only") -> weak scaling.
Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for the roofline accounting.
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

METRIC = "tpc_clusters_per_s_tracked"
UNIT = "clusters/s"
WORKLOADS = {0: "config0 single sector, 200 primaries", 1: "config1 central Pb-Pb-like event, 8000 primaries",
             2: "config2 loopers + primaries", 3: "config3 time slice, 50 collisions",
             4: "config4 time frame, 200 collisions"}


ALU_SMS = 148
# ncu figures of ONE launch of the hot kernels on the bench workload, keyed by (config, generator seed): DRAM bytes
# (dram__bytes_read.sum + dram__bytes_write.sum) and warp instructions (smsp__inst_executed.sum) of the committed
# `ncu --set full` capture named in "file".  They are cited constants (a number taken under a profiler is never a bench
# value); every other configuration or seed reports "traffic": null.
NCU_CAPTURE = {
    (4, 5): {"file": "profiles/r2h_full_capture.md",
             "a4_constructor": {"kernel": "constructUp + constructDown<0,0> + constructDown<0,1> + constructDown<1,0>",
                                "warp_inst": 1.8536e10, "dram_bytes": 22244717000},
             "a2_neighbours": {"kernel": "neighbourFinder", "warp_inst": 8.491e9, "dram_bytes": 1624126000}},
}
STAGE_KERNEL = {"a1_grid": "gridBuild", "a2_neighbours": "neighbourFinder", "a3_cleaner_start": "cleanLinks",
                "a4_constructor": "constructUp + constructDown<0,0> + constructDown<0,1> + constructDown<1,0> (the passes of the "
                                  "tracklet constructor: one step body, launched back to back)",
                "a5_selector": "selectClaim+selectCount+selectEmit"}

# fp32 operations of one Propagate, Update, Search and of one cluster inside a road, and of one window candidate and one
# (u, d) pair of the neighbour finder, as DESIGN.md section 3 writes them (adds, multiplies, divisions, square roots each
# counted once; R0: nothing is fused): DESIGN.md section 8.  HOW OFTEN each runs per unit comes from the oracle's own
# counters on this run's cpu_baseline sample (orcGetO4Counts / orcGetO2Counts), not from a stored table.
O4_FLOPS = (176, 100, 6, 5)
O2_FLOPS = (4, 5)            # slopes of a window candidate (2 subtractions, 2 products); Dev of a pair (2, 2, 1)
SURVEY_BYTES_PER_CLUSTER = 140   # the fixed accounting with H = N
TUBE_CHI2_MAX = 25.0             # the chi2 tube of the second flags run (R49)


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms",
                                          "100", "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL,
                                         text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[2:6]):
                if v == "Active":
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _sector_sample(ev, n_keep_sectors=1, z_frac=1.0):
    """Bounded sample of the workload for the CPU oracle: the first sector(s), optionally a z slab of it."""
    from paper_1910_12214_b200 import datagen
    R = ev.n_rows
    hi = int(ev.row_offset[n_keep_sectors * R])
    off = ev.row_offset[:n_keep_sectors * R + 1].astype(np.int64)
    y, z = ev.y[:hi], ev.z[:hi]
    if z_frac < 1.0:
        zc = 0.5 * (ev.z_min + ev.z_max) + 0.25 * (ev.z_max - ev.z_min)     # slab inside the z > 0 drift volume
        hw = 0.25 * (ev.z_max - ev.z_min) * z_frac
        keep = np.abs(z - zc) <= hw
        bucket = np.repeat(np.arange(n_keep_sectors * R), np.diff(off))
        counts = np.bincount(bucket[keep], minlength=n_keep_sectors * R)
        off = np.concatenate([[0], np.cumsum(counts)])
        y, z = y[keep], z[keep]
    return datagen.event_from_arrays(off, y, z, n_keep_sectors, R, row_x=ev.row_x, z_min=ev.z_min, z_max=ev.z_max,
                                     bz_tesla=ev.bz_tesla)


def _time_oracle(sample, repeats=1):
    from oracle import tpc_oracle as orc
    best = None
    for _ in range(repeats):
        t = time.perf_counter()
        res = orc.run(sample)
        dt = time.perf_counter() - t
        best = dt if best is None else min(best, dt)
    return best, res


def run_reference(args, rank):
    """--impl reference: the CPU oracle as it stands, single thread, on a bounded sample of the same workload."""
    if rank != 0:
        return
    from paper_1910_12214_b200 import datagen
    ev = datagen.make_event(args.config)
    total = args.steps + args.warmup
    # one sector of config 4 costs ~15 s on one core; keep the whole run within ~150 s
    z_frac = 1.0
    if ev.n_sectors > 1 and ev.n_clusters > 5e6:
        z_frac = min(1.0, max(0.02, 150.0 / (15.0 * max(total, 1))))
    sample = _sector_sample(ev, 1, z_frac) if ev.n_sectors > 1 and ev.n_clusters > 2e6 else ev
    times = []
    for i in range(total):
        dt, _ = _time_oracle(sample)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times)) if times else 0.0
    value = sample.n_clusters / (ms * 1e-3) if ms > 0 else 0.0
    desc = (f"sector 0 of {WORKLOADS[args.config]}" + (f", z slab of {z_frac:.2f} of the drift length" if z_frac < 1 else "")
            + f" ({sample.n_clusters} clusters per step)") if sample is not ev else f"whole event ({ev.n_clusters} clusters)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "n_clusters_per_step": int(sample.n_clusters), "sample": desc},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def aggregate(units: float, ms: float, device, world: int):
    """Whole-job figures of a replicated (weak-scaling) run: units summed over ranks, time = max over ranks."""
    import torch
    import torch.distributed as dist
    u = torch.tensor([units], dtype=torch.float64, device=device)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item())


def _oracle_counts(ores):
    """Per-unit operation counts of the oracle's own counters on the cpu_baseline sample: O4 per hit of the accepted
    tracklets (Propagate, Update, Search, clusters inside the roads), O2 per cluster (window candidates, pairs)."""
    H0 = int(ores.tl_nhits[ores.tl_status == 2].sum())
    n0 = int(ores.n_clusters)
    o4 = [float(v) / max(H0, 1) for v in ores.o4_ops]
    o2 = [float(ores.o2_ops[1] + ores.o2_ops[2]) / max(n0, 1), float(ores.o2_ops[3]) / max(n0, 1)]
    return o4, o2


def run_dry(args, rank, world):
    """--dry-run: the N > 1 plumbing without a GPU (gloo): every rank contributes made-up figures through the same
    aggregate(); rank 0 prints one line.  Used by tests/test_multirank_gloo.py to cover the spawner."""
    import torch
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("gloo")
    units, ms = aggregate(1000.0 * (rank + 1), 10.0 * (rank + 1), torch.device("cpu"), world)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"metric": METRIC, "dry_run": True, "n_gpus": world, "units": units, "ms": ms}), flush=True)


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_1910_12214_b200 import datagen, tpc

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the tracker has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    # every rank tracks its own time frame (replicas: independent data per GPU)
    seed = args.config + 1 + 100 * rank
    ev = datagen.generate(datagen.config(args.config, seed=seed), name=f"config{args.config}")
    N = ev.n_clusters
    trk = tpc.TpcTracker.from_event(ev, device=local_rank)
    off, y, z = trk.upload(ev)
    first = trk.run(off, y, z)                     # discovers the capacities (grows once if needed)
    st0 = first.status
    assert st0.status == 0, st0.status
    capT = int(st0.n_start_hits * 1.05) + 1024
    capK = int(st0.n_tracks * 1.05) + 1024
    capC = int(st0.n_track_clusters * 1.05) + 1024
    stream = torch.cuda.current_stream()
    dev = torch.device("cuda", local_rank)

    def step():
        trk.run(off, y, z, cap_tracklets=capT, cap_tracks=capK, cap_track_clusters=capC, sync=False)

    trk.set_profiling(False)
    W = max(args.warmup, 3)
    for _ in range(W):
        step()
    st = trk.status()
    assert st.status == 0
    # ---- the timed region: exactly K steps back to back on one stream, no host synchronisation inside; one CUDA event
    #      between consecutive steps gives the per-step times (median and min) -------------------------
    K = args.steps
    sampler = ClockSampler(local_rank) if rank == 0 else None
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.time()
    evs[0].record(stream)
    for i in range(K):
        step()
        evs[i + 1].record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t1 = time.time()
    st = trk.status()
    assert st.status == 0
    per = np.array([evs[i].elapsed_time(evs[i + 1]) for i in range(K)])
    ms_total = evs[0].elapsed_time(evs[K])
    total_clusters, ms_total_max = aggregate(float(N), ms_total, dev, world)
    _, ms_median = aggregate(float(N), float(np.median(per)), dev, world)
    _, ms_min = aggregate(float(N), float(per.min()), dev, world)
    ms_mean = ms_total_max / K
    ms_step = ms_median                              # `value` stands on the median step (max over ranks)
    value = total_clusters / (ms_step * 1e-3)
    clocks = sampler.stop(t0, t1) if sampler else None

    # ---- per-stage CUDA-event times: a separate instrumented run (the library records an event between the stages) ---
    trk.set_profiling(True)
    stage = np.zeros(8)
    n_inst = 3
    for _ in range(n_inst):
        step()
        s = trk.status()
        stage += np.array(list(s.stage_ms))
    stage /= n_inst

    # ---- the NEXT rows (a6 refit, a7 merger, a10 legs, a8 flags, a9 codes), timed apart: not part of the a1..a5 step ----
    refit_ms = merge_ms = flags_ms = pack_ms = legs_ms = merged_ms = None
    n_links = n_legs = n_two_leg = 0
    flag_frac = {}
    flag_names = (("attached", 1), ("adjacent", 2), ("protected", 4), ("removed_A", 8), ("removed_B", 16))
    if not args.no_refit:
        acc = accm = accf = accp = accl = accd = 0.0
        dq = torch.from_numpy(ev.q).to(y.device)
        for i in range(4):
            trk.run(off, y, z, cap_tracklets=capT, cap_tracks=capK, cap_track_clusters=capC, sync=False, merge=True, flags=True, q=dq,
                    legs=True, pos=True, merged=True)
            s = trk.status()
            if i > 0:
                acc += float(s.stage_ms[7])
                accm += float(s.merge_ms)
                accf += float(s.flags_ms)
                accp += float(s.pack_ms)
                accl += float(s.legs_ms)
                accd += float(s.merged_ms)
        refit_ms, merge_ms, flags_ms, pack_ms, legs_ms, merged_ms = acc / 3, accm / 3, accf / 3, accp / 3, accl / 3, accd / 3
        fl = trk._out["cl_flags"][:N]
        flag_frac = {name: round(float(((fl & bit) != 0).float().mean().item()), 4) for name, bit in flag_names}
        n_two_leg = int((trk._out["trk_mt_rank"][:int(s.n_tracks)] == 1).sum().item())
        n_links = int((trk._out["trk_mg_next"][:int(s.n_tracks)] >= 0).sum().item())
        n_legs = int((trk._out["trk_leg_partner"][:int(s.n_tracks)] >= 0).sum().item()) // 2
    trk.set_profiling(False)

    # ---- end to end through the host-buffer ABI call (pinned host memory; copies inside the timed region) ----
    hy = torch.from_numpy(ev.y).pin_memory()
    hz = torch.from_numpy(ev.z).pin_memory()
    hoff = torch.from_numpy(ev.row_offset.view(np.int32)).pin_memory()
    ny, nz, noff = hy.numpy(), hz.numpy(), hoff.numpy().view(np.uint32)
    e2e_steps = max(2, min(args.steps, 10))
    sth, outh = trk.run_host(noff, ny, nz, cap_tracks=capK, cap_track_clusters=capC)     # warm-up: pools and hints grow here
    assert sth.status == 0
    # Double-buffered: the copies of one event overlap the kernels of the other (tpcSubmitHost / tpcCollectHost).  Every
    # step still copies its inputs from pinned host memory and its tracks back to the host inside the timed region.
    for w in range(2):
        trk.submit_host(w, noff, ny, nz, capK, capC)
    for w in range(2):
        sth, outh = trk.collect_host(w)                # warm-up of both slots (their pools are allocated here)
        assert sth.status == 0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t_e2e = time.perf_counter()
    e0.record(stream)
    trk.submit_host(0, noff, ny, nz, capK, capC)
    for i in range(e2e_steps):
        if i + 1 < e2e_steps:
            trk.submit_host((i + 1) % 2, noff, ny, nz, capK, capC)
        sth, outh = trk.collect_host(i % 2)
        assert sth.status == 0
    e1.record(stream)
    torch.cuda.synchronize()
    wall_e2e = (time.perf_counter() - t_e2e) * 1e3 / e2e_steps
    # the slots run on the library's own streams: the host clock around submit ... collect is the measure (the events on
    # torch's stream only bracket it); max over ranks as for `value`
    _, ms_e2e = aggregate(float(N), max(wall_e2e, e0.elapsed_time(e1) / e2e_steps), dev, world)
    e2e_value = total_clusters / (ms_e2e * 1e-3)
    h2d = 4 * (len(ev.row_offset)) + 8 * N
    # tpcSubmitHost copies back up to the capacities (the counts are not known on the host at submit time)
    d2h = capK * (5 * 4 + 4 + 20 + 60 + 4) + 4 * (capK + 1) + 4 * capC + 8 * 11

    # ---- the flags once more with the chi2 criterion of PAPER.md L108 / L114 on top of the fixed tube (R49): a second
    #      tracker, because the criterion is a creation-time parameter ------------------------------------------------
    flag_frac_chi2, flags_chi2_ms = {}, None
    if not args.no_refit and rank == 0:
        trk.close()
        p2 = tpc.tpcDefaultParams()
        p2.tube_chi2_max = TUBE_CHI2_MAX
        trk2 = tpc.TpcTracker.from_event(ev, params=p2, device=local_rank)
        trk2.set_profiling(True)
        for i in range(2):
            trk2.run(off, y, z, cap_tracklets=capT, cap_tracks=capK, cap_track_clusters=capC, sync=False, flags=True, merged=True)
            s2 = trk2.status()
        flags_chi2_ms = float(s2.flags_ms)
        fl = trk2._out["cl_flags"][:N]
        flag_frac_chi2 = {name: round(float(((fl & bit) != 0).float().mean().item()), 4) for name, bit in flag_names}
        trk2.close()
    if rank != 0:
        return
    # ---- CPU baseline: the oracle on one sector of this event (rank 0, N = 1 only); its operation counters give the
    #      per-unit algorithmic operation counts of the roofline below ------------------------------------------------
    cpu = None
    o4_per_hit = o2_per_cluster = None
    if world == 1 and not args.no_cpu_baseline:
        sample = _sector_sample(ev, 1) if ev.n_sectors > 1 and N > 2e6 else ev
        dt, ores = _time_oracle(sample)
        o4_per_hit, o2_per_cluster = _oracle_counts(ores)
        cpu = {"value": sample.n_clusters / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": (f"sector 0 of the event ({sample.n_clusters} clusters, 1/{ev.n_sectors} of the step), {dt:.1f} s"
                          if sample is not ev else f"whole event ({N} clusters), {dt:.2f} s"),
               "host_cores_available": os.cpu_count(),
               "o4_ops_per_tracklet_hit": [round(v, 4) for v in o4_per_hit],
               "o2_candidates_and_pairs_per_cluster": [round(v, 3) for v in o2_per_cluster]}
        # the same oracle on several sectors at once, one thread per sector (ctypes releases the GIL): what the host's
        # cores do together; `cpu_baseline` above stays the single-core figure of the contract
        if ev.n_sectors > 1 and N > 2e6 and (os.cpu_count() or 1) > 1:
            from concurrent.futures import ThreadPoolExecutor
            from oracle import tpc_oracle as orc
            ncore = min(os.cpu_count() or 1, ev.n_sectors, 16)
            R = ev.n_rows
            samples = []
            for sct in range(ncore):
                lo, hi = int(ev.row_offset[sct * R]), int(ev.row_offset[(sct + 1) * R])
                o = (ev.row_offset[sct * R:(sct + 1) * R + 1].astype(np.int64) - lo).astype(np.uint32)
                samples.append(datagen.event_from_arrays(o, ev.y[lo:hi], ev.z[lo:hi], 1, R, row_x=ev.row_x, z_min=ev.z_min,
                                                         z_max=ev.z_max, bz_tesla=ev.bz_tesla))
            t0m = time.perf_counter()
            with ThreadPoolExecutor(ncore) as pool:
                list(pool.map(orc.run, samples))
            dtm = time.perf_counter() - t0m
            cpu["multicore"] = {"value": sum(s.n_clusters for s in samples) / dtm, "unit": UNIT, "cores": ncore,
                                "sample": f"sectors 0..{ncore - 1} of the event, one oracle thread each, {dtm:.1f} s"}

    # ---- roofline of the dominant kernel ---------------------------------------------------
    peak, peak_src = _peaks()
    H = int(st.n_tracklet_hits)
    nT = int(st.n_tracklets)
    alg = {"a1_grid": 24 * N, "a2_neighbours": 20 * N, "a3_cleaner_start": 24 * N, "a4_constructor": 40 * H + 100 * nT,
           "a5_selector": 32 * H}
    names = list(alg)
    stages = {}
    for i, k in enumerate(names):
        ms = float(stage[i])
        stages[k] = {"ms": round(ms, 4), "alg_bytes": int(alg[k]),
                     "gbs": round(alg[k] / (ms * 1e-3) / 1e9, 1) if ms > 0 else None,
                     "frac_of_hbm_peak": round(alg[k] / (ms * 1e-3) / 1e9 / peak, 4) if ms > 0 else None}
    dom = max(names, key=lambda k: stages[k]["ms"])
    dom_ms = stages[dom]["ms"]
    total_alg = sum(alg.values())
    survey_alg = SURVEY_BYTES_PER_CLUSTER * N
    whole = {"alg_bytes": int(total_alg), "gbs": round(total_alg / (ms_step * 1e-3) / 1e9, 1),
             "frac_of_hbm_peak": round(total_alg / (ms_step * 1e-3) / 1e9 / peak, 5),
             "survey_fixed_accounting": {"bytes_per_cluster": SURVEY_BYTES_PER_CLUSTER, "alg_bytes": int(survey_alg),
                                         "frac_of_hbm_peak": round(survey_alg / (ms_step * 1e-3) / 1e9 / peak, 5)},
             "target_frac": 0.40, "hbm_peak_gbs": peak, "peak_source": peak_src}
    share = round(dom_ms / max(float(stage[6]), 1e-9), 4)
    cap = NCU_CAPTURE.get((args.config, seed))
    ncu = cap.get(dom) if cap else None
    sm_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
    alu_peak = ALU_SMS * 128 * sm_mhz * 1e6 / 1e12
    hbm = {"alg_bytes": int(alg[dom]), "alg_gbs": round(alg[dom] / (dom_ms * 1e-3) / 1e9, 1),
           "alg_frac_of_hbm_peak": round(alg[dom] / (dom_ms * 1e-3) / 1e9 / peak, 5), "hbm_peak_gbs": peak}
    # algorithmic fp32 operations of one launch of the dominant kernel, when it is one of the two arithmetic stages and
    # the oracle leg of this run counted the operations per unit
    flops = per_unit = None
    if dom == "a4_constructor" and o4_per_hit is not None:
        per_unit = sum(a * b for a, b in zip(o4_per_hit, O4_FLOPS))
        flops = H * per_unit
        unit_name = "flops_per_tracklet_hit"
    elif dom == "a2_neighbours" and o2_per_cluster is not None:
        per_unit = sum(a * b for a, b in zip(o2_per_cluster, O2_FLOPS))
        flops = N * per_unit
        unit_name = "flops_per_cluster"
    if dom in ("a4_constructor", "a2_neighbours"):
        # These two stages are bound by instruction issue, not by HBM (DRAM at 1-6 % of peak in the
        # committed captures): "bound": "alu", achieved = algorithmic fp32 operations / live CUDA-event time of the stage,
        # peak = SMs x 128 fp32 lanes x 1 operation / clock (R0 forbids the FMA that would double it).
        roofline = {"bound": "alu", "kernel": STAGE_KERNEL[dom], "unit": "TFLOP/s", "peak": round(alu_peak, 2),
                    "peak_source": f"{ALU_SMS} SMs x 128 fp32 lanes x {sm_mhz:.0f} MHz, no FMA (B200_PROFILING.md unit counts "
                                   "and clocks; DESIGN.md section 8)"}
        if flops is not None:
            achieved = flops / (dom_ms * 1e-3) / 1e12
            roofline.update({"achieved": round(achieved, 3), "frac": round(achieved / alu_peak, 5), "alg_flops": int(flops),
                             unit_name: round(per_unit, 1), "counts_from": "this run's cpu_baseline oracle leg"})
        else:
            roofline.update({"achieved": None, "frac": None, "alg_flops": None,
                             "counts_from": "unavailable: the cpu_baseline oracle leg did not run (N > 1 or --no-cpu-baseline)"})
    else:
        achieved = alg[dom] / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0
        roofline = {"bound": "hbm", "kernel": STAGE_KERNEL[dom], "achieved": round(achieved, 2), "peak": peak, "unit": "GB/s",
                    "frac": round(achieved / peak, 5), "peak_source": peak_src}
    roofline.update({"traffic": ncu["dram_bytes"] if ncu else None, "traffic_from": cap["file"] if ncu else None,
                     "hbm_view": hbm, "whole_path": whole, "share_of_step": share, "launch_ms": round(dom_ms, 4)})
    if ncu:
        issue_peak = ALU_SMS * 4 * sm_mhz * 1e6 / 1e9
        issued = ncu["warp_inst"] / (dom_ms * 1e-3) / 1e9
        roofline["issue"] = {"achieved": round(issued, 2), "peak": round(issue_peak, 1), "unit": "Gwarp-inst/s",
                             "frac": round(issued / issue_peak, 5), "counts_from": cap["file"],
                             "peak_source": f"{ALU_SMS} SMs x 4 schedulers x {sm_mhz:.0f} MHz"}
    # the other arithmetic stage, in the same terms (a2 when the constructor dominates, and the other way round)
    other = "a2_neighbours" if dom == "a4_constructor" else "a4_constructor" if dom == "a2_neighbours" else None
    roofline_second = None
    if other is not None:
        o_ms = stages[other]["ms"]
        o_ncu = cap.get(other) if cap else None
        if other == "a2_neighbours" and o2_per_cluster is not None:
            o_unit = sum(a * b for a, b in zip(o2_per_cluster, O2_FLOPS))
            o_flops, o_name = N * o_unit, "flops_per_cluster"
        elif other == "a4_constructor" and o4_per_hit is not None:
            o_unit = sum(a * b for a, b in zip(o4_per_hit, O4_FLOPS))
            o_flops, o_name = H * o_unit, "flops_per_tracklet_hit"
        else:
            o_flops = None
        roofline_second = {"bound": "alu", "kernel": STAGE_KERNEL[other], "unit": "TFLOP/s", "peak": round(alu_peak, 2),
                           "launch_ms": round(o_ms, 4), "share_of_step": round(o_ms / max(float(stage[6]), 1e-9), 4),
                           "traffic": o_ncu["dram_bytes"] if o_ncu else None, "traffic_from": cap["file"] if o_ncu else None,
                           "alg_bytes": int(alg[other]),
                           "alg_frac_of_hbm_peak": round(alg[other] / (o_ms * 1e-3) / 1e9 / peak, 5) if o_ms > 0 else None}
        if o_flops is not None and o_ms > 0:
            o_ach = o_flops / (o_ms * 1e-3) / 1e12
            roofline_second.update({"achieved": round(o_ach, 3), "frac": round(o_ach / alu_peak, 5), "alg_flops": int(o_flops),
                                    o_name: round(o_unit, 1), "counts_from": "this run's cpu_baseline oracle leg"})
        else:
            roofline_second.update({"achieved": None, "frac": None, "alg_flops": None})
        if o_ncu and o_ms > 0:
            o_iss = o_ncu["warp_inst"] / (o_ms * 1e-3) / 1e9
            roofline_second["issue"] = {"achieved": round(o_iss, 2), "peak": round(ALU_SMS * 4 * sm_mhz * 1e6 / 1e9, 1),
                                        "unit": "Gwarp-inst/s", "frac": round(o_iss / (ALU_SMS * 4 * sm_mhz * 1e6 / 1e9), 5),
                                        "counts_from": cap["file"]}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_step, "ms_per_step_min": ms_min, "ms_per_step_mean": ms_mean,
            "timing": "K steps back to back on one stream, one CUDA event between steps; value on the median step, max over ranks",
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "seed": seed, "n_clusters_per_gpu": N, "n_sectors": ev.n_sectors,
                       "n_rows": ev.n_rows, "cache": "inputs_larger_than_L2" if 8 * N > 126e6 else "working set may fit L2",
                       "parallelism": f"replicas x{world}", "tracks_per_step": int(st.n_tracks),
                       "tracklets_per_step": nT, "start_hits_per_step": int(st.n_start_hits), "tracklet_hits": H},
            "tracks_per_s": float(st.n_tracks) * world / (ms_step * 1e-3),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": ms_e2e, "steps": e2e_steps, "how": "tpcSubmitHost/tpcCollectHost, 2 slots, pinned host buffers"},
            "gpu_launches": int(st.kernel_launches) * K,
            "clocks": clocks, "roofline": roofline, "roofline_second": roofline_second, "stages": stages, "cpu_baseline": cpu}
    if refit_ms is not None:
        ncl = int(st.n_track_clusters)
        rb = 2 * 12 * ncl + 2 * 88 * int(st.n_tracks)       # per pass: index 4 + y,z 8 per cluster; two 88-byte states out
        line["next_refit"] = {"what": "a6 refit of the selected tracks (NEXT-2), not part of `value`", "ms": round(refit_ms, 4),
                              "alg_bytes": rb, "gbs": round(rb / (refit_ms * 1e-3) / 1e9, 1) if refit_ms > 0 else None,
                              "tracks": int(st.n_tracks), "track_clusters": ncl}
        line["next_merge"] = {"what": "a7 segment merger (NEXT-1), not part of `value`", "ms": round(merge_ms, 4),
                              "links": n_links}
        line["next_legs"] = {"what": "a10 pairs of looper legs (rest of NEXT-1), not part of `value`", "ms": round(legs_ms, 4),
                             "pairs": n_legs}
        line["next_merged"] = {"what": "a11 merged tracks and leg labels (O12; rest of NEXT-1, input of NEXT-3), not part of `value`",
                               "ms": round(merged_ms, 4), "tracks_on_secondary_legs": n_two_leg}
        pb = 6 * N + 12 * N       # charge: 4 B in, 2 B out; positions: 8 B in, 4 B out
        line["next_pack"] = {"what": "a9 dynamic-precision charge code and 16-bit position code (NEXT-4), two streaming "
                                     "kernels, not part of `value`",
                             "ms": round(pack_ms, 4), "alg_bytes": pb, "bound": "hbm",
                             "gbs": round(pb / (pack_ms * 1e-3) / 1e9, 1) if pack_ms > 0 else None,
                             "frac_of_hbm_peak": round(pb / (pack_ms * 1e-3) / 1e9 / peak, 4) if pack_ms > 0 else None}
        line["next_flags"] = {"what": "a8 cluster flags and rejection strategies A / B (NEXT-3) with the leg labels of a11 (secondary "
                                      "legs do not protect and are removable by strategy A), not part of `value`",
                              "ms": round(flags_ms, 4), "fractions_of_clusters": flag_frac,
                              "chi2_tube": {"tube_chi2_max": TUBE_CHI2_MAX, "ms": round(flags_chi2_ms, 4) if flags_chi2_ms else None,
                                            "fractions_of_clusters": flag_frac_chi2}}
    print(json.dumps(line), flush=True)


def _spawn(args, argv):
    """`python bench.py --gpus N` without a launcher: start N ranks of this same command under torch.distributed.run
    (one process per GPU, rendezvous on 127.0.0.1) and pass their exit code on."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + argv
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-refit", action="store_true", help="skip the separate timing of the NEXT rows (a6..a10)")
    ap.add_argument("--dry-run", action="store_true", help="N > 1 plumbing only (gloo, no GPU work): for the tests")
    args = ap.parse_args()
    if args.gpus < 1 or args.steps < 1:
        ap.error("--gpus and --steps must be >= 1")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1 and args.impl == "ours":
        sys.exit(_spawn(args, sys.argv[1:]))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and args.impl == "ours":
        print(f"bench.py: --gpus {args.gpus} but the launcher started {world} rank(s)", file=sys.stderr)
        sys.exit(2)
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.dry_run:
        run_dry(args, rank, world)
        return
    run_ours(args, rank, world, local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
