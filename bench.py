#!/usr/bin/env python
"""bench.py -- annihilation photon pairs simulated per second on B200 (BASELINE.json metric).

A *step* is one pass of the whole hot path (gpet_simulate + gpet_digitize: source, panel search, in-panel
Woodcock transport, hits, adder, blur, window, time sort, coincidences) over one batch of synthetic input.
The timed steps run in turn on one stream (the transport kernel with its full CTA (20 warps) per SM).  After the timed
region the same steps are also run as a two-stream pipeline -- the transport kernel of step k+1 (bound by instruction
issue) beside the digitizer of step k (bound by HBM latency) -- and reported under "pipelined";
`--overlap` makes that pipeline the timed headline instead.
Workload at N=1: BASELINE.json configs[1] (C1): 12-panel ring, single layer, centred point source, 0.5 deg
acolinearity, 1e7 pairs, 350-650 keV, 15 % blur, 4 ns window.  With N ranks each rank runs its own 1e7
histories (disjoint history ranges, no data-path collective): weak scaling.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C1] [--pairs P]

Prints ONE JSON line (rank 0).  `--impl reference` times the oracle (oracle/, plain fp64 C on the host
cores) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "annihilation photon pairs simulated/sec"
UNIT = "pairs/s"
SM_COUNT, LANES_PER_SM = 148, 128
# Algorithmic thread-instructions per pair of the transport kernel on C1 (event
# counts of the oracle x audited minimum instruction cost per event).
# C1: SURVEY.md 8(d)'s 740; the others: tests/golden/alg_instr_per_pair.json (written by tests/golden/alg_instr.py from the
# oracle's event counts x the same per-event costs; that audit gives 697 for C1).
AUDITED_C1 = 697.4
ALG_INSTR_PER_PAIR = {"C1": 740.0, "C2": 698.8, "C3": 699.4, "C4": 1104.1, "P1": 999.0, "P2": 999.0, "P3": 999.0,
                      "T1": 1457.4, "T2": 1456.9, "T3": 1460.6}


def digitizer_alg_bytes(n_hits, n_singles, n_coinc, n_buckets):
    """Algorithmic HBM bytes of one gpet_digitize call on the CHUNKED hit layout with coarse time buckets -- the path this
    bench times: every hit's history, ids, energy and time are read once (16 B) and the position of
    each kept single's representative hit (12 B); a kept single is written into its bucket's region (32 B), read by the
    block that sorts the bucket (32 B), written in time order (32 B), read by the window pass (32 B, 1 B flag) and its flag
    by the writer (1 B); a coincidence reads two singles and writes one 36-byte list-mode record; the coarse buckets are
    zeroed, counted and scanned (12 B each)."""
    return 16 * n_hits + (12 + 32 + 32 + 32 + 32 + 2) * n_singles + 100 * n_coinc + 12 * n_buckets


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d.get("hbm_gbs"), sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag, self.proc = index, [], False, None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.samples.append((time.perf_counter(), [x.strip() for x in line.split(",")]))
                if self.stop_flag:
                    break
        except Exception:
            pass

    def finish(self, t0: float, t1: float):
        self.stop_flag = True
        if self.proc:
            self.proc.terminate()
        inside = [s for t, s in self.samples if t0 <= t <= t1] or [s for _, s in self.samples[-3:]]
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": len(inside)}
        try:
            mhz = sorted(float(s[0]) for s in inside)
            out["sm_mhz"] = mhz[len(mhz) // 2]
            out["sm_max_mhz"] = float(inside[0][1])
            out["power_w_max"] = max(float(s[2]) for s in inside)
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            out["reasons"] = [n for i, n in enumerate(names) if any(s[3 + i].lower().startswith("active") for s in inside)]
        except Exception:
            pass
        return out


def workload(config: str, pairs):
    from paper_2603_07327_b200 import workloads as W
    from dataclasses import replace
    if config == "C4" and pairs is None:
        pairs = 62_500_000                                          # one of the 16 time slices of the 1e9-pair run per step
    run = W.config_runs(config, pairs)[0]
    if run.source.half_life_s > 0.0:
        # the bench strings batches together into one long acquisition: constant activity instead of the decay law (12 s of
        # 18F change the activity by 0.1 %), so that every batch is the same 12 s of the paper's Table 1
        run = replace(run, source=replace(run.source, half_life_s=0.0, duration_s=0.0))
    ring = "12-panel ring R=55mm, 2x4 modules of 16x16 LYSO (1.0 mm pitch)"
    tail = "0.5deg acolinearity, 350-650 keV, 15% blur, 4 ns window"
    paper = "the paper's scanner (PAPER.md:47: 10 panels, R=85mm, six 51x51 modules, 1.0 mm pitch)"
    desc = {"C1": f"C1: {ring}, single 10 mm layer, centred point source, {tail}",
            "C2": f"C2: {ring}, two aligned 5 mm layers with a 0.1 mm gap, centred point source, {tail}",
            "C3": f"C3: {ring}, 6 mm front layer offset by half a pitch over a 4 mm back layer, centred point source, {tail}",
            "C4": f"C4: C3's ring, 128^3 x 0.25 mm hot-rod water phantom, pairs from the activity map, one time slice of {run.n_pairs} pairs per step, {tail}",
            "P1": f"P1: {paper}, H2RSPET-1CL, centred point source", "P2": f"P2: {paper}, 1CL-split, centred point source",
            "P3": f"P3: {paper}, 2CL, centred point source",
            "T1": f"T1: {paper}, H2RSPET-1CL, Derenzo source in a 40.25 mm water box, 12 s of decay per step (Table 1, PAPER.md:131-137)",
            "T2": f"T2: {paper}, 1CL-split, Derenzo source, 12 s per step (Table 1)",
            "T3": f"T3: {paper}, 2CL, Derenzo source, 12 s per step (Table 1)"}.get(config, config)
    return run, desc


# ----------------------------------------------------------------------------- reference arm = the oracle
def oracle_pass(run, tables, n, threads, first=0):
    from oracle import gpet_oracle as O
    res = O.simulate(run.geometry, tables, run.source, n, run.seed, first_history=first, threads=threads)
    O.digitize(run.source, run.seed, run.n_pairs, res.hits, run.digitizer)
    return len(res.hits)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import gpet_oracle as O
    from paper_2603_07327_b200 import workloads as W
    O.build()
    run, desc = workload(args.config, args.pairs)
    tables = W.tables()
    threads = os.cpu_count() or 1
    sample = args.ref_pairs
    for w in range(args.warmup):
        oracle_pass(run, tables, min(sample, 50_000), threads)
    t0 = time.perf_counter()
    for k in range(args.steps):
        oracle_pass(run, tables, sample, threads, first=k * sample)
    dt = time.perf_counter() - t0
    value = sample * args.steps / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "pairs_per_step": sample, "note": "oracle (plain fp64 C, oracle/) on the host cores; each step is a "
                   f"bounded sample of {sample} histories of the workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": f"{args.steps} x {sample} pairs of {args.config}"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ----------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2603_07327_b200 import api, sharding, workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    api.lib()                                                   # fails loudly if libgpet.so is missing

    run, desc = workload(args.config, args.pairs)
    n = run.n_pairs
    # Every step simulates its OWN histories: batch b of the job is the time slice [b n world, (b+1) n world) of one long
    # acquisition [R16], rank r takes the r-th n histories of it (disjoint ranges, aligned to time slices: no coincidence
    # window straddles two ranks or two batches).
    from dataclasses import replace
    run = replace(run, source=replace(run.source, pairs_per_time_slice=n))
    n_batches_max = args.warmup + 3 * args.steps + args.e2e_steps + 64
    n_total = sharding.total_pairs(world, n) * n_batches_max
    batch_no = [0]

    def next_first():
        first, _ = sharding.history_range(rank, world, n)
        first += batch_no[0] * sharding.total_pairs(world, n)
        batch_no[0] += 1
        return first

    tables = W.tables()
    geom, mats, src = api.gpet_geometry_create(run.geometry), api.gpet_materials_load(tables), api.DeviceSource(run.source)
    cap = int(n * args.hits_per_pair) + 1024
    # Two batches in flight: gpet_simulate of step k+1 (stream A) runs beside gpet_digitize of step k (stream B); each
    # step is still one full pass of the hot path over its own 1e7 pairs, and every step's work lies in the timed region.
    nbuf = 2 if args.overlap else 1
    # chunked hit layout (include/gpet.h): hits grouped per 512-pair chunk, sorted by history in shared memory by the digitizer
    hits = [api.HitBuffer.allocate_chunked(n, args.hits_per_pair) for _ in range(nbuf)]
    cap = hits[0].capacity
    coinc = [api.CoincBuffer.allocate(cap // 4) for _ in range(nbuf)]
    singles_count = api.SinglesBuffer.allocate(0)                 # NULL arrays, valid counter: the digitizer reports how many singles it kept
    scratch = [torch.empty(api.gpet_digitize_scratch_bytes(n, cap), dtype=torch.uint8, device="cuda") for _ in range(nbuf)]
    s_a = torch.cuda.Stream()
    s_b = torch.cuda.Stream() if args.overlap else s_a
    warps = api.gpet_set_transport_warps(args.transport_warps if args.transport_warps else 0)

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def run_steps(k_steps, record):
        """Enqueues k_steps steps; returns the per-step (transport, digitizer) event pairs when record is set."""
        sim_done = [torch.cuda.Event() for _ in range(nbuf)]
        dig_done = [torch.cuda.Event() for _ in range(nbuf)]
        evs = []
        for k in range(k_steps):
            i = k % nbuf
            if args.overlap and k >= nbuf:
                s_a.wait_event(dig_done[i])                         # hit buffer i has been digitized
            e = [ev() for _ in range(4)] if record else None
            with torch.cuda.stream(s_a):
                hits[i].reset()
                if record:
                    e[0].record(s_a)
                first = next_first()
                api.gpet_simulate(geom, mats, src, first, n, run.seed, hits[i], s_a)
                if record:
                    e[1].record(s_a)
            if args.overlap:
                sim_done[i].record(s_a)
                s_b.wait_event(sim_done[i])
            if record:
                e[2].record(s_b)
            api.gpet_digitize(src, run.seed, n_total, first, n, hits[i], cap, run.digitizer, scratch[i], singles_count, coinc[i], s_b)
            if record:
                e[3].record(s_b)
                evs.append(e)
            if args.overlap:
                dig_done[i].record(s_b)
        if args.overlap:
            s_a.wait_stream(s_b)
        return evs

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    run_steps(args.warmup, False)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.12)
    launches0 = api.gpet_launch_count()
    e0, e1 = ev(), ev()
    barrier()
    w0 = time.perf_counter()
    e0.record(s_a)
    t_events = run_steps(args.steps, True)
    e1.record(s_a)
    barrier()
    w1 = time.perf_counter()
    launches = api.gpet_launch_count() - launches0
    ms_total = sharding.max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.finish(w0, w1) if rank == 0 else None
    transport_ms = sum(e[0].elapsed_time(e[1]) for e in t_events) / len(t_events)
    digitize_ms = sum(e[2].elapsed_time(e[3]) for e in t_events) / len(t_events)
    n_hits, n_coinc, n_singles = hits[0].count(), int(coinc[0].n_coinc.item()), int(singles_count.n_singles.item())
    for hb, cb in zip(hits, coinc):
        if hb.dropped():
            raise SystemExit(f"hit buffer overflow ({hb.dropped()} hits dropped); raise --hits-per-pair")
        if int(cb.n_coinc.item()) > cb.capacity:
            raise SystemExit("coincidence buffer overflow")
    value = sharding.total_pairs(world, n) * args.steps / (ms_total * 1e-3)

    # ---- the two halves alone (untimed extra, not part of `value`): serial steps with the full transport CTA
    alone = None
    if args.overlap:
        api.gpet_set_transport_warps(0)
        st = torch.cuda.current_stream()
        ta, tb = [], []
        for k in range(8):
            hits[0].reset()
            x, y, z = ev(), ev(), ev()
            first = next_first()
            x.record(st); api.gpet_simulate(geom, mats, src, first, n, run.seed, hits[0], st); y.record(st)
            api.gpet_digitize(src, run.seed, n_total, first, n, hits[0], cap, run.digitizer, scratch[0], None, coinc[0], st); z.record(st)
            torch.cuda.synchronize()
            if k >= 3:
                ta.append(x.elapsed_time(y)); tb.append(y.elapsed_time(z))
        alone = {"transport_ms": sum(ta) / len(ta), "digitize_ms": sum(tb) / len(tb)}
    # ---- the same steps as a two-stream pipeline (extra, after the timed region; not part of `value`)
    pipelined = None
    if not args.overlap and not args.no_pipelined:
        pw = api.gpet_set_transport_warps(args.transport_warps if args.transport_warps else 0)
        hits.append(api.HitBuffer.allocate_chunked(n, args.hits_per_pair)); coinc.append(api.CoincBuffer.allocate(cap // 4))
        scratch.append(torch.empty(api.gpet_digitize_scratch_bytes(n, cap), dtype=torch.uint8, device="cuda"))
        s_b2 = torch.cuda.Stream()
        sim_done = [torch.cuda.Event() for _ in range(2)]; dig_done = [torch.cuda.Event() for _ in range(2)]

        def pipe(k_steps):
            for k in range(k_steps):
                i = k & 1
                if k >= 2:
                    s_a.wait_event(dig_done[i])
                with torch.cuda.stream(s_a):
                    hits[i].reset()
                    first = next_first()
                    api.gpet_simulate(geom, mats, src, first, n, run.seed, hits[i], s_a)
                sim_done[i].record(s_a)
                s_b2.wait_event(sim_done[i])
                api.gpet_digitize(src, run.seed, n_total, first, n, hits[i], cap, run.digitizer, scratch[i], None, coinc[i], s_b2)
                dig_done[i].record(s_b2)
            s_a.wait_stream(s_b2)

        pipe(4)
        barrier()
        p0, p1 = ev(), ev()
        p0.record(s_a); pipe(args.steps); p1.record(s_a)
        barrier()
        p_ms = sharding.max_over_ranks(p0.elapsed_time(p1))
        assert hits[1].dropped() == 0 and 0 < int(coinc[1].n_coinc.item()) <= coinc[1].capacity
        pipelined = {"value": sharding.total_pairs(world, n) * args.steps / (p_ms * 1e-3), "unit": UNIT, "ms_per_step": p_ms / args.steps, "steps": args.steps,
                     "transport_warps_per_sm": pw,
                     "note": "gpet_simulate(k+1) on one stream beside gpet_digitize(k) on another, two hit buffers; same results"}
    api.gpet_set_transport_warps(0)                             # the host-buffer path below is one batch at a time

    # ---- end to end through the C ABI with HOST buffers (gpet_pipeline_*: the call a user makes for a stream of batches):
    # every step's list-mode coincidences are copied to pinned host memory inside the timed region; two batches in flight
    # (the copy of step k rides a copy stream while step k+1 computes)
    pipe = api.Pipeline(geom, mats, run.source, run.digitizer, n_total, n, args.hits_per_pair, 0, 2)
    host = [api.HostOutputs(int(n * 0.25) + 1024) for _ in range(2)]

    def e2e_steps(k_steps):
        pipe.submit(next_first(), n, run.seed)
        cnt = None
        for k in range(k_steps):
            if k + 1 < k_steps:
                pipe.submit(next_first(), n, run.seed)
            cnt = pipe.collect(host[k & 1])
            if cnt["n_coinc"] > host[k & 1].cap:
                raise SystemExit("host coincidence buffer too small")
        return cnt

    e2e_steps(max(2, min(args.warmup, 3)))
    barrier()
    t0 = time.perf_counter()
    counts = e2e_steps(args.e2e_steps)
    barrier()
    e2e_s = sharding.max_over_ranks(time.perf_counter() - t0)
    e2e_value = sharding.total_pairs(world, n) * args.e2e_steps / e2e_s
    h2d = 104 + 32 + (run.source.phantom_material.size if run.source.phantom_material is not None else 0)
    d2h = 28 + counts["n_coinc"] * 40
    del pipe

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = load_peaks()
    clock_hz = (peaks["sm_max_mhz"] or 1965.0) * 1e6
    peak_alu = SM_COUNT * LANES_PER_SM * clock_hz
    alg = ALG_INSTR_PER_PAIR.get(args.config)
    achieved = alg * n / (transport_ms * 1e-3) if alg else None
    traffic = None
    tp = os.path.join(ROOT, "profiles", "transport_traffic.txt")
    if os.path.exists(tp) and args.config == "C1":
        try:
            traffic = json.load(open(tp)).get("dram_bytes_per_launch")
        except Exception:
            traffic = None
    roofline = {"kernel": "transport (gpet_simulate)", "bound": "alu", "achieved": achieved, "peak": peak_alu, "unit": "thread-instr/s",
                "frac": achieved / peak_alu if achieved else None, "traffic": traffic,
                # the same fraction on the audited instruction count of tests/golden/alg_instr_per_pair.json (C1: 697 instead of
                # SURVEY's 740), the count every other config is reported on: comparable across configs
                "frac_audited": (AUDITED_C1 / alg * achieved / peak_alu if args.config == "C1" else achieved / peak_alu) if achieved else None,
                "alone": ({"transport_ms": alone["transport_ms"], "achieved": alg * n / (alone["transport_ms"] * 1e-3),
                           "frac": alg * n / (alone["transport_ms"] * 1e-3) / peak_alu,
                           "note": "same kernel with its full CTA (20 warps) and nothing else on the GPU (8 serial steps after the timed region)"}
                          if alone and alg else None),
                "note": f"{alg} algorithmic thread-instr/pair (DESIGN.md 6) x {n} pairs / {transport_ms:.3f} ms; peak = 148 SMs x 128 lanes x "
                        f"{peaks['sm_max_mhz']} MHz ({peaks['source']} max SM clock); hbm {peaks['hbm_gbs']} GB/s of {peaks['source']}",
                "transport_ms": transport_ms, "digitize_ms": digitize_ms, "transport_warps_per_sm": warps,
                "overlap": bool(args.overlap),
                "hit_bytes_gbs": n_hits * 28 / (transport_ms * 1e-3) / 1e9}
    digi_ms = digitize_ms
    roofline_digi = None
    if peaks["hbm_gbs"]:
        dbytes = digitizer_alg_bytes(n_hits, n_singles, n_coinc, (cap + 511) // 512)
        dach = dbytes / (digi_ms * 1e-3) / 1e9
        dtraffic = None
        dp = os.path.join(ROOT, "profiles", "digitizer_traffic.txt")
        if os.path.exists(dp) and args.config == "C1":
            try:
                dtraffic = json.load(open(dp)).get("dram_bytes_per_call")
            except Exception:
                dtraffic = None
        roofline_digi = {"kernel": "digitizer (gpet_digitize on the chunked hit layout: 6 kernels)", "bound": "hbm", "achieved": dach, "peak": peaks["hbm_gbs"],
                         "unit": "GB/s", "frac": dach / peaks["hbm_gbs"], "traffic": dtraffic,
                         "alone": ({"digitize_ms": alone["digitize_ms"], "achieved": dbytes / (alone["digitize_ms"] * 1e-3) / 1e9,
                                    "frac": dbytes / (alone["digitize_ms"] * 1e-3) / 1e9 / peaks["hbm_gbs"]} if alone else None),
                         "note": f"{dbytes / n:.1f} algorithmic B/pair of the chunked path (DESIGN.md 6: {n_hits} hits, {n_singles} kept singles, {n_coinc} "
                                 f"coincidences) / {digi_ms:.3f} ms; peak = hbm_gbs of {peaks['source']}.  Per kernel (profiles/README.md): chunk_adder is bound by "
                                 "instruction issue, the bucket sort by barrier and load latency in its short blocks, the coincidence passes by the 32-byte records they read 8 bytes of; none by bandwidth"}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import gpet_oracle as O
        O.build()
        threads = os.cpu_count() or 1
        oracle_pass(run, tables, 20_000, threads)
        t0 = time.perf_counter()
        oracle_pass(run, tables, args.cpu_pairs, threads)
        dt = time.perf_counter() - t0
        cpu = {"value": args.cpu_pairs / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"first {args.cpu_pairs} histories of {args.config} (transport + digitizer), {dt:.1f} s wall"}

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": desc, "pairs_per_step_per_gpu": n, "seed": run.seed, "parallelism": f"{world} x independent history ranges",
                   "pipeline": (f"two batches in flight: gpet_simulate(k+1) on one stream beside gpet_digitize(k) on another, transport CTA of {warps} warps"
                                if args.overlap else "serial: simulate then digitize on one stream"),
                   "l2": f"inputs larger than L2: the hit buffer ({n_hits * 28 / 1e6:.0f} MB/step) and digitizer scratch exceed the 126 MB L2",
                   "hits_per_step": n_hits, "singles_per_step": n_singles, "coincidences_per_step": n_coinc,
                   "outputs": "timed steps leave list-mode coincidences (and the singles count) in device memory; the caller-visible singles "
                              "arrays are not requested; e2e copies every step's coincidence list to the host"},
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "steps": args.e2e_steps,
                "api": "gpet_pipeline_submit / gpet_pipeline_collect (host outputs per step: coincidence list-mode + counters; two batches in flight)"},
        "roofline": roofline, "roofline_digitizer": roofline_digi, "pipelined": pipelined, "cpu_baseline": cpu,
    }))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C1")
    ap.add_argument("--pairs", type=int, default=None, help="pairs per step per GPU (default: the config's own, 1e7 for C1)")
    ap.add_argument("--hits-per-pair", type=float, default=None, help="hit buffer size per pair (default: 1.2 for C1-C4, 2.0 for P1-P3, 3.0 for T1-T3)")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--cpu-pairs", type=int, default=10_000_000)
    ap.add_argument("--ref-pairs", type=int, default=2_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-pipelined", action="store_true", help="skip the extra two-stream pipeline measurement")
    ap.add_argument("--overlap", action="store_true", help="time the two-stream pipeline as the headline instead of the serial steps")
    ap.add_argument("--transport-warps", type=int, default=0, help="warps per transport CTA (default 20; fewer leave more of each SM to the other stream in the pipeline)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.hits_per_pair is None:
        args.hits_per_pair = {"P": 2.0, "T": 3.0}.get(args.config[0].upper(), 1.2)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
