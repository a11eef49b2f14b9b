#!/usr/bin/env python
"""Benchmark of the photon-propagation hot path (BASELINE.json metric: photons propagated/s on one
B200, layered ice, 5160 DOMs).

  python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path
  python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands

A step = one pass of the whole hot path (a1..a9) over one batch of synthetic input: configuration C1
(BASELINE.json configs[1]: 200 cascades on one 1 km muon, ~1.96e9 photons, 86x60 DOMs, 100 ice layers).
`value` is measured with the sources already resident in HBM (pp_run_resident) and CUDA events;
`e2e` goes through pp_submit / pp_flush / pp_collect with host buffers, copies included.
N > 1 runs N independent replicas ("replicas only", no collective on the data path).
Prints ONE JSON line on rank 0.
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

METRIC = "photons propagated/s on 1 B200, layered ice 5160 DOMs; % of SM FP32 roofline"
UNIT = "photons/s"
WORKLOAD = "C1: BASELINE.json configs[1], 200 cascades E^-1 1 GeV-10 TeV on a 1 km muon, 86x60 DOMs, 100 layers"

# Thread-level instructions the propagation kernel executes per simulated flight (scattering step):
# smsp__thread_inst_executed.sum / flights from the ncu capture named in profiles/ (DESIGN.md section 6).
INSTR_PER_FLIGHT_FILE = os.path.join(ROOT, "profiles", "instr_per_flight.json")


KERNEL_SOURCES = ["pp_kernels.cu", "pp_device.cuh", "pp_types.h"]
FIXED_BUDGET_INSTR_PER_FLIGHT = 240.0  # ~220-260 thread instructions per scattering step


def kernel_source_hash():
    """SHA-256 over the kernel sources and the nvcc flags: what the stored instructions-per-flight was measured on."""
    import hashlib
    from paper_2405_05700_b200 import build as pp_build
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(pp_build.CSRC, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read() + b"\0")
    h.update(" ".join(pp_build.NVCC_FLAGS + os.environ.get("PP_NVCC_EXTRA", "").split()).encode())
    return h.hexdigest()


def load_instr_per_flight():
    """The per-unit figure of the roofline.  Valid only for the exact kernel sources + flags it was measured on:
    returns (None, ..., reason) if the stored SHA-256 differs from the sources in the tree."""
    try:
        with open(INSTR_PER_FLIGHT_FILE) as f:
            d = json.load(f)
        have = kernel_source_hash()
        if d.get("kernel_sources_sha256") != have:
            return None, None, (f"stale: profiles/instr_per_flight.json was measured on sources {str(d.get('kernel_sources_sha256'))[:12]}, "
                                f"the tree holds {have[:12]}; re-measure (bench.py --update-instr-per-flight)"), None
        return float(d["thread_instructions_per_flight"]), d.get("dram_bytes_per_launch"), d.get("source", ""), \
            d.get("fp32_flops_per_flight")
    except Exception as e:
        return None, None, f"unreadable: {e!r}", None


def update_instr_per_flight(args):
    """`bench.py --update-instr-per-flight NCU.csv --flights N [--fp32-per-thread-instr X]`: store the per-unit figure
    from an ncu --csv log of `bench.py --steps 1 --warmup 0 --no-cpu-baseline` taken with the metrics
    smsp__thread_inst_executed.sum, smsp__inst_executed.sum, dram__bytes_read.sum, dram__bytes_write.sum (all propagate
    launches of the run; N = flights those launches simulated, printed by the same bench line)."""
    import csv
    tot = {}
    n_launch = 0
    with open(args.update_instr_per_flight) as f:
        rows = [r for r in csv.reader(f) if len(r) > 5]
    hdr = rows[0]
    i_k, i_m, i_v = hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Value")
    for r in rows[1:]:
        if "propagate_kernel" not in r[i_k]:
            continue
        v = float(r[i_v].replace(",", ""))
        tot[r[i_m]] = tot.get(r[i_m], 0.0) + v
        n_launch += r[i_m] == "smsp__inst_executed.sum"
    thr, warp = tot["smsp__thread_inst_executed.sum"], tot["smsp__inst_executed.sum"]
    d = {"thread_instructions_per_flight": thr / args.flights, "warp_instructions_per_flight": warp / args.flights,
         "mean_active_lanes": thr / warp,
         "fp32_flops_per_flight": (args.fp32_per_thread_instr * thr / args.flights) if args.fp32_per_thread_instr else None,
         "dram_bytes_per_launch": (tot.get("dram__bytes_read.sum", 0.0) + tot.get("dram__bytes_write.sum", 0.0)) / max(1, n_launch),
         "propagate_launches": n_launch, "flights": args.flights, "kernel_sources_sha256": kernel_source_hash(),
         "kernel": "pp::propagate_kernel<false,false,false,false>", "source": args.note}
    with open(INSTR_PER_FLIGHT_FILE, "w") as f:
        json.dump(d, f, indent=2)
        f.write("\n")
    print(json.dumps(d))
    return 0


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


class ClockSampler:
    """Samples SM clock and throttle reasons with nvidia-smi while the timed region runs."""

    def __init__(self, index: int):
        self.index = index
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._th = None

    def _run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip().split("\n")[0]
                f = [x.strip() for x in out.split(",")]
                self.samples.append(float(f[0]))
                self.max_mhz = float(f[1])
                for nm, v in zip(names, f[2:6]):
                    if v.lower().startswith("active"):
                        self.reasons.add(nm)
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._th = threading.Thread(target=self._run, daemon=True)
        self._th.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._th.join(timeout=6)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def workload():
    from paper_2405_05700_b200 import workloads as W
    return W.geometry_full(), W.ice_layered(), W.sources_c1()


# ------------------------------------------------------------------------------------------------
# CPU oracle legs
# ------------------------------------------------------------------------------------------------
def oracle_rate(geo, ice, src, seed, budget_s, n_threads=0):
    """Times the oracle, as it stands, on a strided sample of the workload sized for ~budget_s (n_threads = 0: all
    host cores)."""
    from oracle import oracle as O
    t = time.perf_counter()
    r = O.propagate(geo, ice, src, seed=seed, stride=8192, n_threads=n_threads)
    dt = time.perf_counter() - t
    rate = r.photons / max(dt, 1e-9)
    total = sum(O.photon_count(e, ice.photons_per_GeV) for e in src.src[:, 7])
    stride = 8192
    while stride > 1 and (total / (stride // 2)) / rate < budget_s:
        stride //= 2
    t = time.perf_counter()
    r = O.propagate(geo, ice, src, seed=seed, stride=stride, n_threads=n_threads)
    dt = time.perf_counter() - t
    return {"photons": r.photons, "seconds": dt, "value": r.photons / dt, "flights_per_s": r.flights / dt,
            "stride": stride, "hits": r.hit}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    geo, ice, src = workload()
    cores = os.cpu_count() or 1
    per_step_budget = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_rate(geo, ice, src, 0, 0.5)
    photons = 0
    secs = 0.0
    last = None
    for k in range(args.steps):
        last = oracle_rate(geo, ice, src, k, per_step_budget)
        photons += last["photons"]
        secs += last["seconds"]
    value = photons / secs
    sample = f"C1 photons with photon_idx % {last['stride']} == 0 ({last['photons']} photons per step)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# this repo's CUDA path
# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2405_05700_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    from paper_2405_05700_b200 import replicas
    geo, ice, src = workload()
    seed = replicas.replica_seed(0, rank)  # independent replicas
    target = 10 ** 8
    prop = B.Propagator(geo, ice, seed=seed, launch_photons_target=target)
    d = prop.upload(src.src, src.event_id, src.source_id)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def l2_flush():
        flush_buf.fill_(1)

    s0, s1 = prop.streams
    # ---- device-resident throughput (`value`) ----
    for _ in range(args.warmup):
        prop.run_resident(*d)
        prop.drain()
    st_before = prop.stats()
    launches_before = B.kernel_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    photons = 0
    hits = 0
    barrier()
    with ClockSampler(local) as clk:
        t_wall0 = time.perf_counter()
        for k in range(args.steps):
            l2_flush()
            torch.cuda.synchronize()
            ev[k][0].record(s0)
            ph, _, _ = prop.run_resident(*d)
            s0.wait_stream(s1)
            ev[k][1].record(s0)
            photons += ph
            hits += len(prop.drain())
        barrier()
        t_wall = time.perf_counter() - t_wall0
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    launches = B.kernel_launch_count() - launches_before
    st_after = prop.stats()
    flights = st_after.flights - st_before.flights
    busy_ms = st_after.kernel_busy_ms - st_before.kernel_busy_ms
    n_prop_launches = st_after.launches - st_before.launches

    # ---- end to end through pp_submit / pp_flush / pp_collect with host buffers (`e2e`) ----
    pinned_src = torch.from_numpy(src.src.copy()).pin_memory().numpy()
    for _ in range(min(args.warmup, 2)):
        prop.run(pinned_src, src.event_id, src.source_id)
    barrier()
    e2e_hits = 0
    t0 = time.perf_counter()
    for k in range(args.steps):
        e2e_hits += len(prop.run(pinned_src, src.event_id, src.source_id))
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    st_e2e = prop.stats()
    e2e_launches = st_e2e.launches - st_after.launches

    # ---- device-busy fraction THROUGH THE BATCHING SERVER (north_star: >= 90 %; "> 90 %", PAPER.md:86
    # 45 % -> 80 %): C2 x 10 re-numbered replicas shipped by 8 producer threads in blocks of 8192 sources through
    # pp_submit while one consumer collects.  The headline is ONE continuous stream of 8 passes over those blocks
    # (>= 0.5 s, no flush or pause in between: the steady state PAPER.md:59 describes); beside it the figure of a
    # single short job (one pass, ~80 ms, of which the ramp-up and the drain are several ms) ----
    server = None
    if world == 1 and not args.no_server_leg:
        c2, packed, n_events = pack_stream_blocks(10, 8, 8192)
        with B.Propagator(geo, ice, seed=seed, launch_photons_target=target) as sp:
            sp.run(c2.src, c2.event_id, c2.source_id)  # warm-up
            short = stream_job(sp, packed)
            r = stream_job(sp, packed, passes=8, id_stride=10 * n_events + 1000000)  # (ids clear of the short job's)
        server = {"device_busy_frac": r["kernel_s"] / r["wall_s"], "photons_per_s": r["photons"] / r["wall_s"],
                  "threads": 8, "launches": r["launches"], "jobs": 1, "passes": 8, "photons": r["photons"],
                  "wall_s": r["wall_s"], "hits": r["hits"],
                  "workload": f"one continuous stream: 8 passes over C2 x 10 replicas of {n_events} events "
                              f"({sum(len(b) for b in packed)} blocks of >= 8192 sources per pass) through pp_submit / pp_collect",
                  "short_job": {"device_busy_frac": short["kernel_s"] / short["wall_s"],
                                "photons_per_s": short["photons"] / short["wall_s"], "wall_s": short["wall_s"],
                                "photons": short["photons"], "launches": short["launches"],
                                "workload": "one pass (C2 x 10), submit to drain"},
                  "paper": "GPU utilisation > 90 % (PAPER.md:5); 45 % -> 80 % (PAPER.md:86); hardware not stated"}

    # ---- max over ranks ----
    tmax, wsum = replicas.reduce_results(dist, torch.device("cuda", local), {"dev_ms": dev_ms, "e2e_s": e2e_s},
                                         {"photons": float(photons)})
    dev_ms_max, e2e_s_max, photons_all = tmax["dev_ms"], tmax["e2e_s"], wsum["photons"]
    value = photons_all / (dev_ms_max * 1e-3)
    e2e_value = photons_all / e2e_s_max

    if rank == 0:
        peaks = measured_peaks()
        clocks = clk.summary()
        ipf, dram_bytes, ipf_src, fpf = load_instr_per_flight()
        sm_max = peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0
        n_sm = torch.cuda.get_device_properties(local).multi_processor_count
        roofline = None
        if ipf is not None and busy_ms > 0:
            # issue-slot roofline: every SM sub-partition issues at most one warp instruction (32 thread
            # instructions) per clock: peak = SMs * 4 * 32 * f; f = max SM clock.
            peak = n_sm * 4 * 32 * sm_max * 1e6 / 1e9  # G thread-instr/s
            achieved = flights * ipf / (busy_ms * 1e-3) / 1e9
            roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Ginstr/s (thread-level)",
                        "frac": achieved / peak, "traffic": dram_bytes,
                        "kernel": "pp::propagate_kernel<false,false,false,false>",
                        "kernel_ms_per_launch": busy_ms / max(1, n_prop_launches),
                        "units_per_launch": {"flights": flights / max(1, n_prop_launches)},
                        "thread_instructions_per_flight": ipf, "per_unit_source": ipf_src,
                        "peak_source": f"{n_sm} SMs x 4 issue slots x 32 lanes x {sm_max:.0f} MHz (max SM clock; "
                                       "MEASURED_PEAKS.json sm_max_mhz)",
                        "frac_at_observed_clock": (achieved / (n_sm * 4 * 32 * clocks["sm_mhz"] * 1e-3)
                                                   if clocks.get("sm_mhz") else None)}
            # the same flights/s against a FIXED instruction budget per flight (~240): unlike
            # `frac`, this one cannot rise by executing more instructions per flight
            roofline["frac_fixed_budget"] = flights * FIXED_BUDGET_INSTR_PER_FLIGHT / (busy_ms * 1e-3) / 1e9 / peak
            roofline["fixed_budget_thread_instructions_per_flight"] = FIXED_BUDGET_INSTR_PER_FLIGHT
            if fpf:
                # the metric's "% of SM FP32 roofline": FP32 flops (FFMA = 2, FMUL/FADD = 1) per flight from the same
                # ncu capture, against SMs x 128 lanes x 2 x f; capped near 30 % by the integer/control share of the mix
                fp32_peak = n_sm * 128 * 2 * sm_max * 1e6 / 1e12
                fp32 = flights * float(fpf) / (busy_ms * 1e-3) / 1e12
                roofline["fp32"] = {"achieved_tflops": fp32, "peak_tflops": fp32_peak, "frac": fp32 / fp32_peak,
                                    "fp32_flops_per_flight": float(fpf)}
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            o = oracle_rate(geo, ice, src, 0, 12.0)
            o1 = oracle_rate(geo, ice, src, 0, 6.0, n_threads=1)  # 1 thread and all cores
            cpu = {"value": o["value"], "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                   "sample": f"C1 photons with photon_idx % {o['stride']} == 0 ({o['photons']} photons, {o['seconds']:.1f} s)",
                   "flights_per_s": o["flights_per_s"],
                   "one_thread": {"value": o1["value"], "cores": 1, "flights_per_s": o1["flights_per_s"],
                                  "sample": f"photon_idx % {o1['stride']} == 0 ({o1['photons']} photons, {o1['seconds']:.1f} s)"}}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": dev_ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": WORKLOAD, "photons_per_step": photons / args.steps, "launch_photons_target": target,
                           "l2": "flushed between timed steps (256 MB write); inputs are 9.6 KB, the path is issue-bound",
                           "parallelism": "replicas only" if world > 1 else "single GPU",
                           "hits_per_step": hits / args.steps},
                "flights_per_s": flights / (dev_ms * 1e-3) * world, "flights_per_step": flights / args.steps,
                "propagate_launches_per_step": n_prop_launches / args.steps, "device_busy_frac_resident": busy_ms / dev_ms,
                "wall_s_timed_region": t_wall,
                "e2e": {"value": e2e_value, "unit": UNIT,
                        "h2d_bytes_per_step": int(len(src) * 48 + 0),
                        "d2h_bytes_per_step": int(e2e_hits / args.steps * 32 + e2e_launches / args.steps * 64),
                        "hits_per_step": e2e_hits / args.steps},
                "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "server": server, "cpu_baseline": cpu}
        if roofline is None:
            line["roofline_note"] = ipf_src or "no per-unit figure"
        print(json.dumps(line))
    prop.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------------
# C3: launch-size sweep; C2: streaming from worker threads (report modes, one JSON line per point)
# ------------------------------------------------------------------------------------------------
def run_sweep(args):
    """BASELINE.json configs[3]: photons per launch 1e5..1e9 on C1's geometry and ice; one pp_submit + pp_flush +
    drain per launch with launch_photons_target = N.  Reports photons/s (wall clock, host buffers in and out) and the
    device-busy fraction (kernel time / wall time) per launch size."""
    import torch
    from paper_2405_05700_b200 import binding as B
    from paper_2405_05700_b200 import workloads as W
    torch.cuda.set_device(0)
    geo, ice = W.geometry_full(), W.ice_layered()
    sizes = [10 ** k for k in range(5, 10)] if not args.sweep_sizes else [int(float(x)) for x in args.sweep_sizes.split(",")]
    for n in sizes:
        src = W.sources_c3(float(n), seed=3)
        reps = int(max(3, min(50, 2e9 // n)))
        with B.Propagator(geo, ice, seed=0, launch_photons_target=n) as prop:
            for _ in range(2):
                prop.run(src.src, src.event_id, src.source_id)
            st0 = prop.stats()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            hits = 0
            for _ in range(reps):
                hits += len(prop.run(src.src, src.event_id, src.source_id))
            wall = time.perf_counter() - t0
            st1 = prop.stats()
        ph = st1.photons_done - st0.photons_done
        busy = (st1.kernel_busy_ms - st0.kernel_busy_ms) * 1e-3
        print(json.dumps({"mode": "sweep", "workload": "C3: cascades uniform in the instrumented volume, 1-100 TeV, cut at N photons",
                          "photons_per_launch": n, "sources": len(src), "launches": st1.launches - st0.launches, "reps": reps,
                          "photons_per_s": ph / wall, "kernel_photons_per_s": ph / busy, "device_busy_frac": busy / wall,
                          "ms_per_launch_wall": 1e3 * wall / reps, "ms_per_launch_kernel": 1e3 * busy / reps,
                          "hits_per_launch": hits / reps, "flights_per_photon": (st1.flights - st0.flights) / ph}), flush=True)
    return 0


def pack_stream_blocks(replicas, n_thr, block_sources):
    """C2 re-numbered `replicas` times and dealt to `n_thr` clients: client t owns events g with g % n_thr == t of
    every replica and ships a block whenever >= block_sources sources have piled up (blocks end on event boundaries)."""
    from paper_2405_05700_b200 import binding as B
    from paper_2405_05700_b200 import workloads as W
    src = W.sources_c2()
    order = np.argsort(src.event_id, kind="stable")
    rec = B.pack_sources(src.src[order])
    ev, sid = src.event_id[order], src.source_id[order]
    n_events = int(ev.max()) + 1
    first = np.searchsorted(ev, np.arange(n_events + 1))  # sources of event g: [first[g], first[g+1])
    blocks = [[] for _ in range(n_thr)]
    for t in range(n_thr):
        cur, cur_n = [], 0
        for r in range(replicas):
            for g in range(t, n_events, n_thr):
                a, b = int(first[g]), int(first[g + 1])
                if b > a:
                    cur.append((r, a, b))
                    cur_n += b - a
                if cur_n >= block_sources:
                    blocks[t].append(cur)
                    cur, cur_n = [], 0
        if cur:
            blocks[t].append(cur)
    packed = [[(np.concatenate([rec[a:b] for _, a, b in blk]),
                np.concatenate([ev[a:b] + np.uint32(r * n_events) for r, a, b in blk]),
                np.concatenate([sid[a:b] for _, a, b in blk])) for blk in bl] for bl in blocks]
    return src, packed, n_events


def stream_job(prop, packed, passes: int = 1, id_stride: int = 0):
    """Producer threads (the paper's propagation clients) ship their packed blocks through pp_submit
    while one consumer thread collects hits; returns wall seconds, photons, kernel-busy seconds, launches, hits between
    the first submit and the drain.  `passes` > 1: every producer ships its blocks that many times over without a
    pause or a flush in between -- one continuous stream --, the event ids of pass q moved up by q * id_stride so that
    no (event, source) pair recurs."""
    import torch
    st0 = prop.stats()

    def producer(t):
        for q in range(passes):
            for r_, e_, s_ in packed[t]:
                prop.submit(r_, e_ if q == 0 else e_ + np.uint32(q * id_stride), s_)

    n_hits = [0]
    done = threading.Event()

    def consumer():
        while True:
            h = prop.collect(1 << 20, block=True)
            if len(h) == 0:
                if done.is_set():
                    return
                time.sleep(0.0005)
                continue
            n_hits[0] += len(h)

    torch.cuda.synchronize()
    t0 = time.perf_counter()
    cons = threading.Thread(target=consumer)
    cons.start()
    th = [threading.Thread(target=producer, args=(t,)) for t in range(len(packed))]
    for t in th:
        t.start()
    for t in th:
        t.join()
    prop.flush()
    done.set()
    cons.join()
    n_hits[0] += len(prop.collect_all())
    wall = time.perf_counter() - t0
    st1 = prop.stats()
    return {"wall_s": wall, "photons": int(st1.photons_done - st0.photons_done),
            "kernel_s": (st1.kernel_busy_ms - st0.kernel_busy_ms) * 1e-3, "launches": int(st1.launches - st0.launches),
            "hits": int(n_hits[0]), "source_ring_high_water": int(st1.source_ring_high_water)}


def run_stream(args):
    """BASELINE.json configs[2] through the batching server.  `--threads` producer threads play the paper's
    propagation clients: each owns a share of the events of `--replicas` re-numbered replicas of
    C2, queues their light sources and ships a block to the server whenever `--block-sources` sources have piled up
    ("when the step queue is sufficiently full, a block of steps is sent"); one consumer thread collects hits
    meanwhile; the server cuts launches at 1e8 photons.  The blocks are packed before the clock starts (producing the
    sources is the CPU stages' work, not this path's).  Reports photons/s and the device-busy fraction between the
    first submit and the drain."""
    import torch
    from paper_2405_05700_b200 import binding as B
    from paper_2405_05700_b200 import workloads as W
    torch.cuda.set_device(0)
    geo, ice = W.geometry_full(), W.ice_layered()
    replicas, n_thr = args.replicas, max(1, args.threads)
    src, packed, n_events = pack_stream_blocks(replicas, n_thr, args.block_sources)
    with B.Propagator(geo, ice, seed=0, launch_photons_target=10 ** 8) as prop:
        prop.run(src.src, src.event_id, src.source_id)  # warm-up
        r = stream_job(prop, packed)
    print(json.dumps({"mode": "stream", "workload": f"C2 x {replicas} replicas of {n_events} events, shipped in blocks of >= "
                      f"{args.block_sources} sources by {n_thr} client threads", "threads": n_thr,
                      "blocks": sum(len(b) for b in packed), "sources": int(len(src) * replicas), "photons": r["photons"],
                      "launches": r["launches"], "photons_per_s": r["photons"] / r["wall_s"],
                      "device_busy_frac": r["kernel_s"] / r["wall_s"], "wall_s": r["wall_s"], "kernel_s": r["kernel_s"],
                      "hits": r["hits"], "source_ring_high_water": r["source_ring_high_water"]}), flush=True)
    return 0


def _ipc_client_main(name, client, n_clients, replicas, block_sources, barrier, q):
    """One propagation client process of `--stream --ipc-clients` (no CUDA, no torch in here)."""
    try:
        from paper_2405_05700_b200 import binding as B
        from paper_2405_05700_b200 import ipc
        from paper_2405_05700_b200 import workloads as W
        src = W.sources_c2()
        order = np.argsort(src.event_id, kind="stable")
        rec, ev, sid = B.pack_sources(src.src[order]), src.event_id[order], src.source_id[order]
        n_events = int(ev.max()) + 1
        mine = (ev % n_clients) == client
        rec, ev, sid = rec[mine], ev[mine], sid[mine]
        blocks = []
        for r in range(replicas):
            e_r = ev + np.uint32(r * n_events)
            for a in range(0, len(ev), block_sources):
                blocks.append((rec[a:a + block_sources], e_r[a:a + block_sources], sid[a:a + block_sources]))
        n_hits = 0
        with ipc.IpcClient(name) as c:
            barrier.wait()
            t_first = time.time()  # (wall-clock stamps: comparable across the client processes)
            for r_, e_, s_ in blocks:
                c.submit(r_, e_, s_)
                n_hits += len(c.collect(block=False))
            n_hits += len(c.collect_all())
            t_drained = time.time()
        q.put((client, n_hits, len(blocks), t_first, t_drained))
    except Exception as e:  # pragma: no cover
        q.put((client, repr(e), 0, 0.0, 0.0))


def run_stream_ipc(args):
    """`--stream --ipc-clients N`: the paper's instance-count scan (1, 2, 4, 8, 16 client instances share
    ONE photon server).  N client PROCESSES ship blocks of C2's light sources through shared memory (include/pp_ipc.h)
    to this process, which owns the propagator; photons/s and device-busy between the start signal and the last
    client's drain."""
    import multiprocessing as mp
    import torch
    from paper_2405_05700_b200 import binding as B
    from paper_2405_05700_b200 import ipc
    from paper_2405_05700_b200 import workloads as W
    torch.cuda.set_device(0)
    geo, ice = W.geometry_full(), W.ice_layered()
    src = W.sources_c2()
    n = args.ipc_clients
    name = f"/pp_bench_{os.getpid()}"
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    barrier = ctx.Barrier(n + 1)
    with B.Propagator(geo, ice, seed=0, launch_photons_target=10 ** 8) as prop:
        prop.run(src.src, src.event_id, src.source_id)  # warm-up
        with ipc.IpcServer(prop, name, max_clients=n, ingest_threads=args.ingest_threads) as srv:
            procs = [ctx.Process(target=_ipc_client_main, args=(name, c, n, args.replicas, args.block_sources, barrier, q))
                     for c in range(n)]
            for p in procs:
                p.start()
            st0 = prop.stats()  # (before the start signal: the server is idle now, and the clients start at once)
            barrier.wait()  # every client has packed its blocks and attached
            t0 = time.perf_counter()
            res = [q.get(timeout=600) for _ in procs]
            wall = time.perf_counter() - t0
            st1 = prop.stats()
            for p in procs:
                p.join(timeout=60)
            ist = srv.stats()
    bad = [r for r in res if not isinstance(r[1], int)]
    if bad:
        raise SystemExit(f"ipc client failed: {bad}")
    ph = st1.photons_done - st0.photons_done
    busy = (st1.kernel_busy_ms - st0.kernel_busy_ms) * 1e-3
    # the job as the clients see it: from the first client's first submit to the last client's drain (the outer clock
    # also counts the wake-up from the start barrier and the result queue of N Python processes)
    wall_outer, wall = wall, max(r[4] for r in res) - min(r[3] for r in res)
    print(json.dumps({"mode": "stream-ipc", "workload": f"C2 x {args.replicas} replicas shipped in blocks of {args.block_sources} "
                      f"sources by {n} client processes over shared memory", "client_processes": n,
                      "blocks": int(sum(r[2] for r in res)), "photons": int(ph), "launches": st1.launches - st0.launches,
                      "photons_per_s": ph / wall, "device_busy_frac": busy / wall, "wall_s": wall, "kernel_s": busy,
                      "wall_s_outer": wall_outer, "device_busy_frac_outer": busy / wall_outer,
                      "hits": int(sum(r[1] for r in res)), "hits_unrouted": ist["hits_unrouted"],
                      "server_blocks_ingested": ist["blocks_ingested"]}), flush=True)
    return 0


def run_multi(args):
    """`python bench.py --gpus N` WITHOUT torchrun: ONE server process, N devices behind one front (include/pp_multi.h,
    NEXT-4): C1 is shipped through pp_multi_submit, dealt in batches of 1e8 photons to the least-loaded device, and
    collected through one pp_multi_collect.  Prints the contract's JSON line (value = whole-job photons/s; wall clock
    between the first submit and the drain, host buffers in and out).  With `--same-device` all N handles sit on
    cuda:0 (what a 1-GPU box can run: checks the plumbing, says nothing about scaling)."""
    import torch
    from paper_2405_05700_b200 import multi
    n = args.gpus
    have = torch.cuda.device_count()
    devices = [0] * n if args.same_device else list(range(n))
    if not args.same_device and have < n:
        raise SystemExit(f"bench.py: --gpus {n} but only {have} CUDA devices (use --same-device for a plumbing check)")
    geo, ice, src = workload()
    target = 10 ** 8
    with multi.MultiFront.over_devices(geo, ice, devices, seed=0, launch_photons_target=target, deal_photons=target) as m:
        for _ in range(args.warmup):
            m.run(src.src, src.event_id, src.source_id)
        for d in set(devices):
            torch.cuda.synchronize(d)
        st0 = [p.stats() for p in m._props]
        hits = 0
        with ClockSampler(0) as clk:
            t0 = time.perf_counter()
            for _ in range(args.steps):
                hits += len(m.run(src.src, src.event_id, src.source_id))
            wall = time.perf_counter() - t0
        st1 = [p.stats() for p in m._props]
        mst = m.stats()
    ph = sum(b.photons_done - a.photons_done for a, b in zip(st0, st1))
    busy = [(b.kernel_busy_ms - a.kernel_busy_ms) * 1e-3 for a, b in zip(st0, st1)]
    flights = sum(b.flights - a.flights for a, b in zip(st0, st1))
    n_launch = int(sum(b.launches - a.launches for a, b in zip(st0, st1)))
    # the issue-slot roofline of the propagation kernel, as in the single-GPU line, averaged over the devices:
    # (sum of flights x instructions per flight) / (sum of the devices' kernel-busy time), against ONE device's peak
    roofline = None
    ipf, dram_bytes, ipf_src, _ = load_instr_per_flight()
    clocks = clk.summary()
    if ipf is not None and sum(busy) > 0:
        sm_max = measured_peaks().get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0
        n_sm = torch.cuda.get_device_properties(devices[0]).multi_processor_count
        peak = n_sm * 4 * 32 * sm_max * 1e6 / 1e9
        achieved = flights * ipf / sum(busy) / 1e9
        roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Ginstr/s (thread-level), per device",
                    "frac": achieved / peak, "traffic": dram_bytes, "kernel": "pp::propagate_kernel<false,false,false,false>",
                    "kernel_ms_per_launch": 1e3 * sum(busy) / max(1, n_launch),
                    "units_per_launch": {"flights": flights / max(1, n_launch)},
                    "thread_instructions_per_flight": ipf, "per_unit_source": ipf_src,
                    "frac_fixed_budget": flights * FIXED_BUDGET_INSTR_PER_FLIGHT / sum(busy) / 1e9 / peak,
                    "note": "kernel-busy time summed over the devices; the job's wall clock is in value / ms_per_step"}
    cpu = None
    if not args.no_cpu_baseline:
        o = oracle_rate(geo, ice, src, 0, 12.0)
        cpu = {"value": o["value"], "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
               "sample": f"C1 photons with photon_idx % {o['stride']} == 0 ({o['photons']} photons, {o['seconds']:.1f} s)"}
    print(json.dumps({"metric": METRIC, "value": ph / wall, "unit": UNIT, "n_gpus": n, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * wall / args.steps, "higher_is_better": True,
                      "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": WORKLOAD, "parallelism": f"one server process, {n} devices behind one front "
                                 "(pp_multi.h): replicas only, no collective", "devices": devices,
                                 "deal_photons": target, "photons_per_step": ph / args.steps},
                      "device_busy_frac_per_device": [b / wall for b in busy],
                      "photons_per_device": [b.photons_done - a.photons_done for a, b in zip(st0, st1)],
                      "batches_per_device": mst["batches"], "hits_per_step": hits / args.steps,
                      "e2e": {"value": ph / wall, "unit": UNIT, "h2d_bytes_per_step": int(len(src) * 48),
                              "d2h_bytes_per_step": int(hits / args.steps * 32)},
                      "gpu_launches": n_launch, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu}))
    return 0


def run_c4(args):
    """BASELINE.json configs[4]: one 1e8 GeV bundle (500 muons, ~5e9 photons) with the hit ring capped at 2 GB, and
    the same event with a 256 KiB ring (stop/replay relaunches all the time): time, device memory, hits."""
    import torch
    from paper_2405_05700_b200 import binding as B
    from paper_2405_05700_b200 import workloads as W
    torch.cuda.set_device(0)
    geo, ice, src = W.geometry_full(), W.ice_layered(), W.sources_c4()
    for ring in (2 << 30, 256 << 10):
        torch.cuda.synchronize()
        torch.cuda.reset_peak_memory_stats()
        mem0 = torch.cuda.memory_allocated()
        with B.Propagator(geo, ice, seed=0, launch_photons_target=5 * 10 ** 8, hit_ring_bytes=ring,
                          source_ring_bytes=16 << 20) as prop:
            prop.run(src.src[:64], src.event_id[:64], src.source_id[:64])  # warm-up
            st0 = prop.stats()
            t0 = time.perf_counter()
            hits = prop.run(src.src, src.event_id, src.source_id)
            wall = time.perf_counter() - t0
            st1 = prop.stats()
            peak = torch.cuda.max_memory_allocated() - mem0
            ws, pin = prop.device_workspace_bytes, prop.pinned_workspace_bytes
        ph = st1.photons_done - st0.photons_done
        busy = (st1.kernel_busy_ms - st0.kernel_busy_ms) * 1e-3
        print(json.dumps({"mode": "c4", "workload": "C4: one 1e8 GeV bundle, 500 muons", "sources": len(src), "photons": int(ph),
                          "hit_ring_bytes": ring, "device_workspace_bytes": int(ws), "pinned_workspace_bytes": int(pin),
                          "peak_device_bytes_over_baseline": int(peak), "hits": int(len(hits)),
                          "hit_bytes": int(len(hits) * 32), "launches": st1.launches - st0.launches,
                          "relaunches": st1.relaunches - st0.relaunches, "photons_per_s": ph / wall,
                          "device_busy_frac": busy / wall, "wall_s": wall,
                          "hit_ring_high_water_bytes": int(st1.hit_ring_high_water)}), flush=True)
    return 0


def run_ext(args):
    """C1 with the optional physics on (report mode): the stand-in wavelength bins (R-21), weighted DOM acceptance
    (R-17) and C1's cascades given a 5 m length (R-18), through the device-resident path, next to the plain run."""
    import torch
    from paper_2405_05700_b200 import binding as B
    from paper_2405_05700_b200 import workloads as W
    torch.cuda.set_device(0)
    geo, ice, src = workload()
    for name in ("plain", "acceptance", "spectrum", "acceptance+spectrum+segments"):
        with B.Propagator(geo, ice, seed=0, launch_photons_target=10 ** 8) as prop:
            if "acceptance" in name:
                prop.set_acceptance("weighted", W.ACCEPTANCE_COEF)
            if "spectrum" in name:
                prop.set_spectrum(W.spectrum_standin())
            ln = np.full(len(src), 5.0, np.float32) if "segments" in name else None
            for _ in range(2):
                prop.run(src.src, src.event_id, src.source_id, ln)
            st0 = prop.stats()
            t0 = time.perf_counter()
            hits = 0
            for _ in range(args.steps):
                hits += len(prop.run(src.src, src.event_id, src.source_id, ln))
            wall = time.perf_counter() - t0
            st1 = prop.stats()
        ph = st1.photons_done - st0.photons_done
        busy = (st1.kernel_busy_ms - st0.kernel_busy_ms) * 1e-3
        print(json.dumps({"mode": "ext", "physics": name, "photons_per_step": ph / args.steps, "photons_per_s": ph / wall,
                          "kernel_photons_per_s": ph / busy, "flights_per_photon": (st1.flights - st0.flights) / ph,
                          "hits_per_step": hits / args.steps,
                          "rejected_per_step": (st1.photons_rejected - st0.photons_rejected) / args.steps}), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--same-device", action="store_true",
                    help="with --gpus N and no torchrun: put all N handles of the multi-device front on cuda:0")
    ap.add_argument("--no-server-leg", action="store_true", help="skip the device-busy-through-the-server leg")
    ap.add_argument("--update-instr-per-flight", default="", metavar="NCU_CSV",
                    help="store profiles/instr_per_flight.json from an ncu --csv log (see update_instr_per_flight)")
    ap.add_argument("--flights", type=float, default=0.0, help="with --update-instr-per-flight: flights the launches simulated")
    ap.add_argument("--fp32-per-thread-instr", type=float, default=0.0,
                    help="with --update-instr-per-flight: FP32 flops per thread instruction from the ncu source page")
    ap.add_argument("--note", default="", help="with --update-instr-per-flight: where the numbers come from")
    ap.add_argument("--ext", action="store_true", help="C1 with the optional physics on (report mode)")
    ap.add_argument("--c4", action="store_true", help="C4 memory-bounded extreme event (report mode)")
    ap.add_argument("--sweep", action="store_true", help="C3 launch-size sweep (report mode)")
    ap.add_argument("--sweep-sizes", default="", help="comma-separated photons per launch (default 1e5..1e9)")
    ap.add_argument("--stream", action="store_true", help="C2 replicas through the batching server from worker threads")
    ap.add_argument("--threads", type=int, default=8)
    ap.add_argument("--replicas", type=int, default=10)
    ap.add_argument("--ipc-clients", type=int, default=0, help="with --stream: N client processes over include/pp_ipc.h")
    ap.add_argument("--block-sources", type=int, default=8192, help="sources a client queues before it ships a block")
    ap.add_argument("--ingest-threads", type=int, default=0, help="with --ipc-clients: ingest threads of the server (0 = default)")
    args = ap.parse_args()
    if args.update_instr_per_flight:
        return update_instr_per_flight(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.ext:
        return run_ext(args)
    if args.c4:
        return run_c4(args)
    if args.sweep:
        return run_sweep(args)
    if args.stream:
        return run_stream_ipc(args) if args.ipc_clients > 0 else run_stream(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return run_multi(args)  # one server process, N devices (NEXT-4); under torchrun: N independent replicas
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
