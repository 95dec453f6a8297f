#!/usr/bin/env python
"""bench.py -- events/s of the LST hot path on B200 (BASELINE.json metric), with roofline and
CPU-oracle baseline.  One JSON line on stdout (rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Workload (config.workload): BASELINE.json configs[2] = 64 independent PU200-like events
(configs[1] recipe, seeds 0..63), pipelined on 4 CUDA streams, 16-event batched launches, the
arena allocated once.  A "step" is one pass of the WHOLE hot path (a0 bin/sort, a1 MD, a2 LS,
a3 T3, a4 T5) over these 64 events.  `value` = events/s with the hit SoA already resident in
HBM; `e2e` = the same through the C-ABI with HOST (pinned) buffers: H2D of the hits and D2H of
the quintuplets inside the timed region.  N > 1: independent replicas (events are independent,
PAPER.md:147), one process per GPU, no data-path collective.

--impl reference times the CPU oracle (the tier's reference arm) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "events/sec at PU200-like density (1 B200)"
UNIT = "events/s"
N_EVENTS = 64
NOMINAL_HBM_GBS = 8000.0           # the "about 8 TB/s" of BASELINE.json's north_star; fractions are reported against the measured peak AND this
N_STREAMS = int(os.environ.get("LST_BENCH_STREAMS", "4"))   # BASELINE.json configs[2]: 4 streams (override: experiments only)
# SURVEY.md 8(d) algorithmic bytes per unit (each input read once, each output written once)
MAP_BYTES = 4 * (69630 + 6121)
# SPEC operations per candidate (every sqrt and div counted as one)
FLOPS_PER_CAND = (34, 51, 45, 255)
HEADER_BYTES = 424   # per-slot counter block that lst_sync_batch reads back (csrc/lst_device.cuh SlotHeader)
A0_KERNELS = ("bin_count", "bin_scatter", "bin_order")               # lst_stats.kernel_ms[0..2]


def algorithmic_bytes(stage: int, n_hits, needed):
    md, ls, t3, t5 = needed
    return (37 * n_hits,
            16 * n_hits + 40 * md,
            24 * md + MAP_BYTES + 24 * ls,
            8 * ls + 16 * md + 16 * t3,
            12 * t3 + 16 * md + 28 * t5)[stage]


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [v.strip() for v in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def rank_seed0(rank: int) -> int:
    """First event seed of a rank: replicas work on disjoint events (rank r: seeds 64 r .. 64 r + 63)."""
    return rank * N_EVENTS


def max_over_ranks(value: float, dist, device) -> float:
    """The slowest rank's time (the job is over when the last replica is)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_events_per_s(world: int, steps: int, total_ms: float) -> float:
    """Events all ranks processed / the slowest rank's time."""
    return world * N_EVENTS * steps / (total_ms * 1e-3)


def make_map(geom, device=None):
    """The module map (rule [B]), the step before the path: our arm builds it with the library's own GPU
    builder (lst_build_module_map), the reference arm with the oracle's (device=None)."""
    from paper_2207_08207_b200 import synth
    mg = synth.map_geometry(geom)
    margs = (mg["layer"], mg["phi"], mg["rho"], mg["gap"], mg["hw"], mg["zlo"], mg["zhi"])
    if device is None:
        from oracle import oracle
        offs, tg = oracle.load("f64").build_map(*margs)
    else:
        from paper_2207_08207_b200 import lst
        offs, tg, _ = lst.build_module_map(*margs, device=device)
    return synth.ModuleMap(geom.n_modules, offs, tg)


def make_events(seed0: int, n: int, device=None):
    from paper_2207_08207_b200 import synth
    geom = synth.make_geometry()
    return geom, make_map(geom, device), [synth.generate_event(geom, 1, seed0 + i) for i in range(n)]


# ------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on a bounded sample
# ------------------------------------------------------------------------------------------
def oracle_events_per_s(geom, mmap, events, check=None):
    """Times the oracle over `events`.  check: per event, the quintuplet hit tuples the GPU arm downloaded end to end; they
    are compared with the oracle's (outside the timed intervals)."""
    from oracle import oracle
    o = oracle.load("f32")
    dt = 0.0
    for k, ev in enumerate(events):
        t0 = time.perf_counter()
        r = o.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side)
        dt += time.perf_counter() - t0
        if check is not None:
            want, got = r.t5_hits(), check[k]
            assert got.shape == want.shape and set(map(tuple, got.tolist())) == set(map(tuple, want.tolist())), \
                f"end-to-end quintuplets of event {k} differ from the oracle's"
    return len(events) / dt, dt


def _oracle_with_seeds(geom, mmap, ev, sd):
    from oracle import oracle
    return oracle.load("f32").run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side, seeds=sd.arrays())


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    per_step = 4                                     # bounded sample: 4 of the 64 events per step
    geom, mmap, events = make_events(0, per_step)
    for _ in range(args.warmup):
        oracle_events_per_s(geom, mmap, events[:1])
    tot = 0.0
    for _ in range(args.steps):
        tot += oracle_events_per_s(geom, mmap, events)[1]
    value = per_step * args.steps / tot
    cpu = {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"{per_step} events (seeds 0..{per_step - 1}) of the 64-event workload per step, single thread"}
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                      "data": "synthetic", "config": workload_config(), "cpu_baseline": cpu,
                      "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                      "gpu_launches": 0}))


def workload_config():
    return {"workload": "BASELINE.json configs[2]: 64 PU200-like events (configs[1] recipe, seeds 0..63), "
                        "4 CUDA streams x 16-event batched launches, arena reused",
            "events_per_step": N_EVENTS, "streams": N_STREAMS, "geometry": "6-layer barrel, 6120 pT modules",
            "l2": "explicit L2 flush (256 MiB memset) between timed steps, outside the timed intervals"}


# ------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2207_08207_b200 import build as lst_build, lst

    rank = int(os.environ.get("RANK", "0"))
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        lst_build.build()                       # no-op when liblst.so is up to date (it travels in-tree); never a fallback
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    geom, mmap, events = make_events(rank_seed0(rank), N_EVENTS, device=local)
    per_stream = N_EVENTS // N_STREAMS
    cfg = lst.default_config()
    cfg.device, cfg.n_slots = local, 2 * N_EVENTS          # second half: the other buffer set of the end-to-end pipeline
    ctx = lst.Lst.from_synth(geom, mmap, cfg)
    streams = [torch.cuda.Stream(dev) for _ in range(N_STREAMS)]
    main = torch.cuda.current_stream(dev)
    d_in = [[torch.from_numpy(a).to(dev) for a in (e.x, e.y, e.z, e.module, e.side)] for e in events]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    torch.cuda.synchronize(dev)

    def step_device():
        for s, st in enumerate(streams):
            ctx.load_events(s * per_stream, d_in[s * per_stream:(s + 1) * per_stream], stream=st)
            ctx.run_batch(s * per_stream, per_stream, st)

    def timed(step_fn, n_steps):
        """n_steps steps, each bracketed by CUDA events on the launching streams, L2 flushed between."""
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(n_steps)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(n_steps)]
        done = [torch.cuda.Event() for _ in streams]
        for i in range(n_steps):
            flush.zero_()
            e0[i].record(main)
            for st in streams:
                st.wait_event(e0[i])
            step_fn()
            for st, d in zip(streams, done):
                d.record(st)
                main.wait_event(d)
            e1[i].record(main)
        torch.cuda.synchronize(dev)
        return [a.elapsed_time(b) for a, b in zip(e0, e1)]

    def barrier():
        torch.cuda.synchronize(dev)
        if dist:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # warm-up, then check every slot finished without overflow / bad input
    timed(step_device, max(3, args.warmup))
    stats = []
    for k in range(N_EVENTS):
        ctx.sync(k, streams[k // per_stream])
        stats.append(ctx.stats(k))
    n_hits = sum(s["n_hits"] for s in stats)
    needed = [sum(s["needed"][j] for s in stats) for j in range(4)]
    cands = [sum(s["candidates"][j] for s in stats) for j in range(4)]
    evals = [sum(s["evaluated"][j] for s in stats) for j in range(4)]
    rewalks = [sum(s["rewalks"][j] for s in stats) for j in range(4)]

    # ---- the timed region ---------------------------------------------------------------
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = ctx.launch_count()
    w0 = time.perf_counter()
    ms = timed(step_device, args.steps)
    barrier()
    wall = time.perf_counter() - w0
    launches = ctx.launch_count() - l0
    clocks = sampler.stop()
    total_ms = max_over_ranks(sum(ms), dist, dev)
    value = whole_job_events_per_s(world, args.steps, total_ms)

    if args.profile and args.with_optional:
        # the optional stages [D] and [P] in the profiled step too, so that one ncu capture covers every kernel
        from paper_2207_08207_b200 import synth as _synth
        d_sd = [[torch.from_numpy(a).to(dev) for a in _synth.generate_seeds(e, rank_seed0(rank) + i).arrays()] for i, e in enumerate(events)]

        def step_all():
            for s, st in enumerate(streams):
                ctx.load_events(s * per_stream, d_in[s * per_stream:(s + 1) * per_stream], stream=st)
                ctx.load_seeds(s * per_stream, d_sd[s * per_stream:(s + 1) * per_stream], stream=st)
                ctx.run_batch(s * per_stream, per_stream, st)
                ctx.run_stage(s * per_stream, per_stream, lst.CLEAN, st)
                ctx.run_stage(s * per_stream, per_stream, lst.PIXEL, st)
        timed(step_all, 2)
    if args.profile:
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                              "ms_per_step": total_ms / args.steps, "gpu_launches": int(launches), "profile_mode": True}))
        ctx.close()
        return

    # ---- end to end: pinned host hits in, quintuplets out, through the C-ABI -------------
    # Host input in the "packed" layout of include/lst.h (the five arrays of an event in ONE pinned block): an event
    # travels as one copy-engine transfer while the results come back through k_fetch_direct (SM writes over PCIe), so
    # the two directions do not queue on one engine.  LST_BENCH_E2E_INPUT=arrays: five separate pinned arrays per event
    # (read by the binning kernel itself), for comparison.
    e2e_input = os.environ.get("LST_BENCH_E2E_INPUT", "packed")
    if e2e_input == "packed":
        keep_blocks, np_in = [], []
        for e in events:
            bufs = lst.packed_event_buffers(e.n)
            for dst, src in zip(bufs[:5], (e.x, e.y, e.z, e.module, e.side)):
                dst[:] = src
            np_in.append(list(bufs[:5]))
            keep_blocks.append(bufs[5])
    else:
        h_in = [[torch.from_numpy(a).pin_memory() for a in (e.x, e.y, e.z, e.module, e.side)] for e in events]
        np_in = [[t.numpy() for t in ev] for ev in h_in]
    cap5 = max(s["needed"][3] for s in stats) * 2 + 1024
    # Two buffer sets (slots, streams, pinned result buffers): step i + 1 is loaded and run while the results of
    # step i travel back -- H2D and D2H share the PCIe link in opposite directions, as in a continuously fed pipeline.
    sets = []
    for p in range(2):
        out = [(torch.empty((cap5, 10), dtype=torch.int32).pin_memory().numpy(), torch.empty((cap5, 5), dtype=torch.float32).pin_memory().numpy())
               for _ in range(N_EVENTS)]
        sets.append({"base": p * N_EVENTS, "streams": streams if p == 0 else [torch.cuda.Stream(dev) for _ in range(N_STREAMS)],
                     "idx": [[out[k][0] for k in range(s * per_stream, (s + 1) * per_stream)] for s in range(N_STREAMS)],
                     "val": [[out[k][1] for k in range(s * per_stream, (s + 1) * per_stream)] for s in range(N_STREAMS)],
                     # the same pinned memory seen as binary16 rows, for the reduced-precision store
                     "val_h": [[out[k][1].view(np.float16).reshape(-1)[:cap5 * 5].reshape(cap5, 5) for k in range(s * per_stream, (s + 1) * per_stream)]
                               for s in range(N_STREAMS)],
                     "counts": None})

    e2e_kind = [lst.T5]                             # lst.CLEAN: the path + cleaning stage, only the kept quintuplets travel back
    e2e_ctx = [ctx, "val"]                          # the context the end-to-end arm drives and the result buffers it fills

    def e2e_launch(i):                              # H2D of the pinned hit SoA + a0..a4 of step i, all asynchronous
        S = sets[i % 2]
        for s, st in enumerate(S["streams"]):
            e2e_ctx[0].load_events(S["base"] + s * per_stream, np_in[s * per_stream:(s + 1) * per_stream], stream=st)
            e2e_ctx[0].run_batch(S["base"] + s * per_stream, per_stream, st)
            if e2e_kind[0] == lst.CLEAN:
                e2e_ctx[0].run_stage(S["base"] + s * per_stream, per_stream, lst.CLEAN, st)

    def e2e_collect(i):                             # counters back (one sync per stream), then gathers + D2H enqueued
        S = sets[i % 2]
        S["counts"] = [e2e_ctx[0].fetch_batch(S["base"] + s * per_stream, e2e_kind[0], S["idx"][s], S[e2e_ctx[1]][s], stream=st, wait=False)
                       for s, st in enumerate(S["streams"])]

    def e2e_run(n):
        e2e_launch(0)
        for i in range(1, n):
            e2e_launch(i)
            e2e_collect(i - 1)
        e2e_collect(n - 1)
        for S in sets:
            for st in S["streams"]:
                st.synchronize()

    e2e_steps = max(4, min(args.steps, 40))
    e2e_run(3)
    barrier()
    t0 = time.perf_counter()
    e2e_run(e2e_steps)
    torch.cuda.synchronize(dev)
    e2e_s = max_over_ranks(time.perf_counter() - t0, dist, dev)
    # the results are on the host: both buffer sets hold every event's quintuplets (all counts checked here; every tuple is
    # compared with the ORACLE's in the cpu_baseline leg below, where the oracle runs over these events anyway)
    for S in sets:
        got = [c for per in S["counts"] for c in per]
        assert got == [st_["needed"][3] for st_ in stats], "end-to-end results incomplete"
    e2e_tuples = [np.array(sets[0]["idx"][k // per_stream][k % per_stream][:stats[k]["needed"][3]]) for k in range(N_EVENTS)]
    # the same with the cleaning stage [D] in the step and only the kept quintuplets (the track candidates) downloaded
    e2e_kind[0] = lst.CLEAN
    e2e_run(3)
    barrier()
    t0 = time.perf_counter()
    e2e_run(e2e_steps)
    torch.cuda.synchronize(dev)
    e2e_tc_s = max_over_ranks(time.perf_counter() - t0, dist, dev)
    kept_e2e = sum(c for S in sets[:1] for per in S["counts"] for c in per)
    e2e_kind[0] = lst.T5
    h2d = sum(sum(a.nbytes for a in ev) for ev in np_in)
    d2h = needed[3] * (40 + 20) + N_EVENTS * HEADER_BYTES
    # What the link itself allows for these byte counts: the same number and sizes of transfers as plain copies, both
    # directions at once on two streams, nothing else on the GPU (same box, same pinned buffers).
    pcie = pcie_ceiling(torch, dev, [[blk] for blk in keep_blocks] if e2e_input == "packed" else np_in,
                        [(stats[k]["needed"][3] * 40, stats[k]["needed"][3] * 20) for k in range(N_EVENTS)], sets[0])
    step_s = e2e_s / e2e_steps
    e2e = {"value": world * N_EVENTS * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
           "d2h_bytes_per_step": int(d2h), "steps": e2e_steps, "ms_per_step": 1e3 * step_s,
           "h2d_gbs": h2d / step_s / 1e9, "d2h_gbs": d2h / step_s / 1e9, "input_layout": e2e_input,
           "pcie_ceiling": pcie,
           "how": "per stream: lst_load_events(16 x pinned host event, packed layout: one copy-engine transfer each) + lst_run_batch + "
                  "lst_fetch_batch(T5 hit indices + values to pinned host buffers); two buffer sets, step i + 1 is loaded and run while "
                  "step i's results travel back; the timed region ends with every step's results on the host",
           "track_candidates": {"value": world * N_EVENTS * e2e_steps / e2e_tc_s, "unit": UNIT, "d2h_bytes_per_step": int(kept_e2e * 60 + N_EVENTS * HEADER_BYTES),
                                "what": "the same pipeline with LST_CLEAN in the step and lst_fetch_batch(kind = LST_CLEAN): only the kept "
                                        "quintuplets (T5-only track candidates) travel back"}}

    # ---- per-kernel times (CUDA events inside the library, timing mode), one 64-event batch ----
    kernel_ms, launches_per_step = per_kernel_times(lst, geom, mmap, d_in, local)
    lp = launches_per_step                      # per-launch quantities: one launch covers 64 / lp events
    alone_ms, _ = per_kernel_times(lst, geom, mmap, d_in, local, alone=True)
    for k in lst.KERNEL_NAMES[7:]:
        kernel_ms.pop(k)
        alone_ms.pop(k)
    with_clean_ms, _ = per_kernel_times(lst, geom, mmap, d_in, local, with_clean=True)
    clean_alone_ms, _ = per_kernel_times(lst, geom, mmap, d_in, local, with_clean=True, alone=True, reps=3)
    clean_ms = {k: {"in_step": with_clean_ms[k], "alone": clean_alone_ms[k]} for k in lst.KERNEL_NAMES[7:]}
    peaks = measured_peaks()
    roof, per_stage = roofline(kernel_ms, alone_ms, n_hits / lp, [v / lp for v in needed], [v / lp for v in evals], peaks, N_EVENTS // lp)
    spec_flops_step = sum(evals[i] * FLOPS_PER_CAND[i] for i in range(4))
    alu_peak = 148 * 128 * peaks["sm_max_mhz"] * 1e6 / 1e12
    path = {"what": "whole path a0..a4 over the timed region: SPEC flops of all evaluated candidates and algorithmic bytes "
                    "of all stages per step / ms_per_step",
            "alu_tflops": spec_flops_step / (total_ms / args.steps * 1e-3) / 1e12, "alu_peak_tflops": alu_peak,
            "alu_frac": spec_flops_step / (total_ms / args.steps * 1e-3) / 1e12 / alu_peak,
            "hbm_gbs": sum(algorithmic_bytes(i, n_hits, needed) for i in range(5)) / (total_ms / args.steps * 1e-3) / 1e9,
            "hbm_frac": sum(algorithmic_bytes(i, n_hits, needed) for i in range(5)) / (total_ms / args.steps * 1e-3) / 1e9 / peaks["hbm_gbs"],
            "hbm_frac_nominal": sum(algorithmic_bytes(i, n_hits, needed) for i in range(5)) / (total_ms / args.steps * 1e-3) / 1e9 / NOMINAL_HBM_GBS}

    # ---- the path followed by the optional duplicate-cleaning stage [D], same timing rules ----
    def step_device_clean():
        for s, st in enumerate(streams):
            ctx.load_events(s * per_stream, d_in[s * per_stream:(s + 1) * per_stream], stream=st)
            ctx.run_batch(s * per_stream, per_stream, st)
            ctx.run_stage(s * per_stream, per_stream, lst.CLEAN, st)
    timed(step_device_clean, 3)
    clean_total_ms = max_over_ranks(sum(timed(step_device_clean, args.steps)), dist, dev)
    for s, st in enumerate(streams):
        ctx.sync_batch(s * per_stream, per_stream, st)
    kept = sum(ctx.stats(k)["n_kept"] for k in range(N_EVENTS))
    clean = {"events_per_s_with_clean": whole_job_events_per_s(world, args.steps, clean_total_ms),
             "ms_per_step_with_clean": clean_total_ms / args.steps, "kernels_ms_per_launch": clean_ms,
             "t5_in": needed[3], "t5_kept": kept,
             "what": "a0..a4 + LST_CLEAN per step; `value` above is a0..a4 only (the BASELINE.json path)"}

    # ---- the path followed by the optional pixel-linking stage [P]: the stand-in seed
    # model of DESIGN.md section 3, seeds resident in HBM like the hits, same timing rules ----
    from paper_2207_08207_b200 import synth as _synth
    seeds = [_synth.generate_seeds(e, rank_seed0(rank) + i) for i, e in enumerate(events)]
    d_seeds = [[torch.from_numpy(a).to(dev) for a in sd.arrays()] for sd in seeds]

    def step_device_pixel():
        for s, st in enumerate(streams):
            ctx.load_events(s * per_stream, d_in[s * per_stream:(s + 1) * per_stream], stream=st)
            ctx.load_seeds(s * per_stream, d_seeds[s * per_stream:(s + 1) * per_stream], stream=st)
            ctx.run_batch(s * per_stream, per_stream, st)
            ctx.run_stage(s * per_stream, per_stream, lst.PIXEL, st)
    timed(step_device_pixel, 3)
    pix_total_ms = max_over_ranks(sum(timed(step_device_pixel, args.steps)), dist, dev)
    for s, st in enumerate(streams):
        ctx.sync_batch(s * per_stream, per_stream, st)
    pst = [ctx.stats(k) for k in range(N_EVENTS)]
    pix_links0 = [ctx.fetch_pixel_links(0, kind)[0] for kind in (0, 1)]
    pix_objs0 = [ctx.fetch_hit_indices(0, lst.T3), ctx.fetch_hit_indices(0, lst.T5)]
    pix_in, _ = per_kernel_times(lst, geom, mmap, d_in, local, d_seeds=d_seeds)
    pix_alone, _ = per_kernel_times(lst, geom, mmap, d_in, local, d_seeds=d_seeds, alone=True, reps=3)
    pix_sum = lambda key, k: int(sum(q[key][k] for q in pst))
    n_seeds_step = int(sum(q["n_seeds"] for q in pst))
    # algorithmic bytes (each input read once, each output written once): seeds 20 B in + 24 B ordered; per outer object its
    # record (T3 16 B, T5 20 + 4 B) + 16 B per anchor + 4 B offset; 20 B per link
    pix_bytes = [(16 + 3 * 16 + 4) * needed[2] + 20 * pix_sum("pix_needed", 0) + 44 * n_seeds_step,
                 (24 + 5 * 16 + 4) * needed[3] + 20 * pix_sum("pix_needed", 1) + 24 * n_seeds_step]
    pixel = {"events_per_s_with_pixel": whole_job_events_per_s(world, args.steps, pix_total_ms), "ms_per_step_with_pixel": pix_total_ms / args.steps,
             "seeds_per_step": n_seeds_step,
             "links_per_step": {"pt3": pix_sum("pix_needed", 0), "pt5": pix_sum("pix_needed", 1)},
             "candidates_per_step": {"pt3": pix_sum("pix_candidates", 0), "pt5": pix_sum("pix_candidates", 1)},
             "evaluated_per_step": {"pt3": pix_sum("pix_evaluated", 0), "pt5": pix_sum("pix_evaluated", 1)},
             "rewalks_per_step": {"pt3": pix_sum("pix_rewalks", 0), "pt5": pix_sum("pix_rewalks", 1)},
             "kernels_ms_per_launch": {k: {"in_step": pix_in[k], "alone": pix_alone[k]} for k in ("seed_bin", "pt3", "pt5")},
             "hbm_frac_alone": {k: pix_bytes[i] / lp / (pix_alone[k] * 1e-3) / 1e9 / measured_peaks()["hbm_gbs"] for i, k in enumerate(("pt3", "pt5"))},
             "what": "a0..a4 + lst_load_seeds + LST_PIXEL per step (hits and seeds resident in HBM); `value` above is a0..a4 only. The method's "
                     "search space is the full (outer object, seed) product (candidates); the kernels evaluate the window of each "
                     "object's first anchor (evaluated) and link sets equal the oracle's (tests/test_gpu_pixel.py)"}

    arena_mib = ctx.arena_bytes()[0] / 2 ** 20
    # ---- reduced-precision object store [H]: the same measurements with
    # lst_config.store_half: output floats that no selection reads kept as binary16, everything else unchanged ----
    ctx.close()
    cfg_h = lst.default_config()
    cfg_h.device, cfg_h.n_slots, cfg_h.store_half = local, 2 * N_EVENTS, 1
    ctx_h = lst.Lst.from_synth(geom, mmap, cfg_h)

    def step_device_half():
        for s, st in enumerate(streams):
            ctx_h.load_events(s * per_stream, d_in[s * per_stream:(s + 1) * per_stream], stream=st)
            ctx_h.run_batch(s * per_stream, per_stream, st)
    timed(step_device_half, 3)
    half_total_ms = max_over_ranks(sum(timed(step_device_half, args.steps)), dist, dev)
    for s, st in enumerate(streams):
        ctx_h.sync_batch(s * per_stream, per_stream, st)
    assert [ctx_h.stats(k)["needed"] for k in range(N_EVENTS)] == [st_["needed"] for st_ in stats], "half store changed the object counts"
    e2e_ctx[0], e2e_ctx[1] = ctx_h, "val_h"
    e2e_run(3)
    barrier()
    t0 = time.perf_counter()
    e2e_run(e2e_steps)
    torch.cuda.synchronize(dev)
    e2e_h_s = max_over_ranks(time.perf_counter() - t0, dist, dev)
    ctx_h.close()
    half_ms, _ = per_kernel_times(lst, geom, mmap, d_in, local, store_half=True)
    half_alone_ms, _ = per_kernel_times(lst, geom, mmap, d_in, local, alone=True, reps=3, store_half=True)
    stored = lambda h: needed[0] * (8, 4)[h] + needed[1] * (16, 8)[h] + needed[2] * (4, 2)[h] + needed[3] * ((20, 10)[h] + 4)
    half = {"what": "lst_config.store_half = 1: MD (dphi, dphichange), LS (sinS, z0, dphi, dphichange), T3 chi2rz, T5 (5 values) stored and "
                    "downloaded as binary16 (round to nearest even of the fp32 result); selections, sets and [D] unchanged (DESIGN.md [H])",
            "events_per_s": whole_job_events_per_s(world, args.steps, half_total_ms), "events_per_s_fp32": value,
            "ms_per_step": half_total_ms / args.steps, "ms_per_step_fp32": total_ms / args.steps,
            "kernels_ms_in_step": {k: {"fp32": kernel_ms[k], "half": half_ms[k]} for k in ("md", "seg", "t3", "t5")},
            "kernels_ms_alone": {k: {"fp32": alone_ms[k], "half": half_alone_ms[k]} for k in ("md", "seg", "t3", "t5")},
            "output_float_bytes_per_step": {"fp32": int(stored(0)), "half": int(stored(1))},
            "algorithmic_bytes_per_step_fp32": int(sum(algorithmic_bytes(i, n_hits, needed) for i in range(5))),
            "e2e": {"value": world * N_EVENTS * e2e_steps / e2e_h_s, "value_fp32": e2e["value"], "unit": UNIT,
                    "d2h_bytes_per_step": int(needed[3] * (40 + 10) + N_EVENTS * HEADER_BYTES), "d2h_bytes_per_step_fp32": int(d2h)}}

    # ---- the same step with lst_config.launches_in_flight = N_STREAMS (include/lst.h): stage grids sized so that the four
    # launches of a stage together fill whole residency waves.  Reported beside `value`, which stays the default sizing ----
    cfg_w = lst.default_config()
    cfg_w.device, cfg_w.n_slots, cfg_w.launches_in_flight = local, N_EVENTS, N_STREAMS
    ctx_w = lst.Lst.from_synth(geom, mmap, cfg_w)

    def step_device_waves():
        for s, st in enumerate(streams):
            ctx_w.load_events(s * per_stream, d_in[s * per_stream:(s + 1) * per_stream], stream=st)
            ctx_w.run_batch(s * per_stream, per_stream, st)
    timed(step_device_waves, 3)
    waves_total_ms = max_over_ranks(sum(timed(step_device_waves, args.steps)), dist, dev)
    for s, st in enumerate(streams):
        ctx_w.sync_batch(s * per_stream, per_stream, st)
    assert [ctx_w.stats(k)["needed"] for k in range(N_EVENTS)] == [st_["needed"] for st_ in stats], "the sizing hint changed the object counts"
    ctx_w.close()
    waves = {"what": "lst_config.launches_in_flight = 4: k_seg 16 blocks per event (the four launches of the stage all resident at once), "
                     "k_md / k_t3 27 (two waves); a k_seg launch then takes ~0.46 ms in step and ~0.29 ms alone instead of 0.33 / 0.19, so "
                     "the per-kernel roofline above is that of the default sizing",
             "events_per_s": whole_job_events_per_s(world, args.steps, waves_total_ms), "ms_per_step": waves_total_ms / args.steps,
             "events_per_s_default": value}

    # ---- the step before the path: module-map builder [B], built once per geometry ----
    from paper_2207_08207_b200 import synth as _synth
    mg = _synth.map_geometry(geom)
    margs = (mg["layer"], mg["phi"], mg["rho"], mg["gap"], mg["hw"], mg["zlo"], mg["zhi"])
    lst.build_module_map(*margs, device=local)
    b_offs, b_tg, b_ms = lst.build_module_map(*margs, device=local)
    map_builder = {"kernels_ms": {"count": b_ms[0], "fill": b_ms[1]}, "modules": int(geom.n_modules), "connections": int(len(b_tg)),
                   "pair_tests_per_s": 2 * geom.n_modules ** 2 / ((b_ms[0] + b_ms[1]) * 1e-3),
                   "equals_input_map": bool(np.array_equal(b_offs, mmap.row_offsets) and np.array_equal(b_tg, mmap.targets))}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
           "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic", "config": workload_config(), "clocks": clocks, "e2e": e2e,
           "gpu_launches": int(launches), "roofline": roof, "per_stage": per_stage,
           "us_per_event": 1e3 * total_ms / (args.steps * N_EVENTS), "wall_s_timed_region": wall,
           "objects_per_step": dict(hits=n_hits, md=needed[0], ls=needed[1], t3=needed[2], t5=needed[3]),
           "candidates_per_step": dict(md=cands[0], ls=cands[1], t3=cands[2], t5=cands[3]),
           "evaluated_per_step": dict(md=evals[0], ls=evals[1], t3=evals[2], t5=evals[3]),
           "roofline_path": path,
           "stage_overlap": {"sum_of_launch_ms_per_step": launches_per_step * sum(v["ms"] for v in per_stage.values()),
                             "sum_of_alone_ms_per_step": launches_per_step * sum(v["alone"]["ms"] for v in per_stage.values()),
                             "ms_per_step_4_streams": total_ms / args.steps,
                             "factor": launches_per_step * sum(v["ms"] for v in per_stage.values()) / (total_ms / args.steps),
                             "alone_factor": launches_per_step * sum(v["alone"]["ms"] for v in per_stage.values()) / (total_ms / args.steps),
                             "what": "launches per step x (sum of the kernels' durations) / the step. `factor` uses the durations inside the "
                                     "4-stream step (kernels of different streams run side by side and stretch one another), `alone_factor` "
                                     "the durations with the GPU otherwise idle: what the 4-stream pipeline gains over running the same "
                                     "launches back to back"},
           "csrc_digest": csrc_digest(),
           "duplicate_cleaning": clean, "pixel_linking": pixel, "reduced_precision_store": half, "wave_aligned_grids": waves, "module_map_builder": map_builder,
           "rewalks_per_step": dict(md=rewalks[0], ls=rewalks[1], t3=rewalks[2], t5=rewalks[3]),
           "arena_mib": arena_mib, "impl": "ours"}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_pass, t_cpu = 0, 0.0
        while t_cpu < 12.0 and n_pass < 8:          # a bounded sample: whole passes over the workload, >= 12 s of CPU work
            t_cpu += oracle_events_per_s(geom, mmap, events, check=e2e_tuples if n_pass == 0 else None)[1]
            n_pass += 1
        # [P]: the links of event 0 as the timed step left them, against the oracle's full product
        r0 = _oracle_with_seeds(geom, mmap, events[0], seeds[0])
        for kind in (0, 1):
            got = np.concatenate([pix_links0[kind][:, :1], pix_objs0[kind][pix_links0[kind][:, 1]].reshape(len(pix_links0[kind]), -1)], 1)
            assert set(map(tuple, got.tolist())) == set(map(tuple, r0.pix_tuples(kind).tolist())), "pixel links of event 0 differ from the oracle's"
        out["pixel_linking"]["verified"] = "pixel triplets and quintuplets of event 0 after the timed steps equal the oracle's (seed index + hit indices)"
        out["e2e"]["verified"] = f"the quintuplets of all {N_EVENTS} events as downloaded by the end-to-end arm equal the oracle's (sets of 10 hit indices)"
        out["cpu_baseline"] = {"value": n_pass * N_EVENTS / t_cpu, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "sample": f"all {N_EVENTS} events of the workload x {n_pass} passes, single thread, {t_cpu:.1f} s"}
        # the same oracle on every host core: events are independent (SURVEY 8(d) "all host cores" figure)
        from concurrent.futures import ThreadPoolExecutor
        from oracle import oracle as _oracle
        o = _oracle.load("f32")
        n_thr = os.cpu_count() or 1
        def _one(ev):
            o.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side)   # ctypes releases the GIL
        work = events * max(2, (64 * n_thr + N_EVENTS - 1) // N_EVENTS)       # ~64 events per thread: several seconds
        t0 = time.perf_counter()
        with ThreadPoolExecutor(n_thr) as pool:
            list(pool.map(_one, work))
        dt = time.perf_counter() - t0
        t0 = time.perf_counter()
        o.build_map(*margs)
        map_builder["oracle_s_one_thread"] = time.perf_counter() - t0
        out["cpu_baseline"]["all_cores"] = {"value": len(work) / dt, "unit": UNIT, "cores": n_thr,
                                            "sample": f"{len(work)} events on {n_thr} threads, {dt:.1f} s"}
    ctx.close()
    if rank == 0:
        print(json.dumps(out))
    if dist:
        dist.destroy_process_group()


def pcie_ceiling(torch, dev, np_in, out_bytes, S, reps=10):
    """Plain copies of the end-to-end arm's byte counts, both directions at once: per step the host->device transfers the
    library makes (np_in: per event the list of pinned host tensors that travel -- ONE block in the packed layout, five arrays
    otherwise) on one stream and 128 device->host transfers (hit tuples and values of every event) on another, from / to the
    same pinned buffers.  Returns the step time and what it would allow in events/s."""
    h_src = [[a if hasattr(a, "data_ptr") else torch.from_numpy(a) for a in ev] for ev in np_in]
    d_dst = [[torch.empty(t.numel(), dtype=t.dtype, device=dev) for t in ev] for ev in h_src]
    per = N_EVENTS // N_STREAMS
    h_out = [(torch.from_numpy(S["idx"][k // per][k % per]).view(torch.uint8).reshape(-1), torch.from_numpy(S["val"][k // per][k % per]).view(torch.uint8).reshape(-1))
             for k in range(N_EVENTS)]
    d_src = torch.empty(max(max(a, b) for a, b in out_bytes) + 16, dtype=torch.uint8, device=dev)
    up, down = torch.cuda.Stream(dev), torch.cuda.Stream(dev)

    def step(do_up=True, do_down=True):
        if do_up:
            with torch.cuda.stream(up):
                for hs, ds in zip(h_src, d_dst):
                    for h, d in zip(hs, ds):
                        d.copy_(h, non_blocking=True)
        if do_down:
            with torch.cuda.stream(down):
                for (hi, hv), (nb_i, nb_v) in zip(h_out, out_bytes):
                    hi[:nb_i].copy_(d_src[:nb_i], non_blocking=True)
                    hv[:nb_v].copy_(d_src[:nb_v], non_blocking=True)

    def timed(**kw):
        for _ in range(2):
            step(**kw)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        for _ in range(reps):
            step(**kw)
        torch.cuda.synchronize(dev)
        return (time.perf_counter() - t0) / reps

    both, only_up, only_down = timed(), timed(do_down=False), timed(do_up=False)
    h2d = sum(t.numel() * t.element_size() for ev in h_src for t in ev)
    d2h = sum(a + b for a, b in out_bytes)
    return {"ms_per_step_both_directions": 1e3 * both, "events_per_s": N_EVENTS / both, "h2d_alone_gbs": h2d / only_up / 1e9,
            "d2h_alone_gbs": d2h / only_down / 1e9, "h2d_gbs_duplex": h2d / both / 1e9, "d2h_gbs_duplex": d2h / both / 1e9,
            "h2d_transfers_per_step": sum(len(ev) for ev in h_src), "d2h_transfers_per_step": 2 * N_EVENTS,
            "what": "cudaMemcpyAsync (torch copy_) of the end-to-end arm's transfers only, two streams, same pinned buffers, same box; "
                    "no kernel running"}


def per_kernel_times(lst, geom, mmap, d_in, local, with_clean=False, reps=6, alone=False, store_half=False, d_seeds=None):
    """Average duration (ms) of ONE launch of every kernel, from CUDA events recorded by the library around every launch on
    the stream it is launched on (lst_config.timing), L2 flushed before every step.
    alone=False: the configuration the timed region uses -- 4 streams x 16-event launches running concurrently (concurrent
    kernels share the SMs, so the durations of one step add up to more than the step).
    alone=True: the same 16-event launches one batch at a time on one stream, the GPU otherwise idle.
    The optional cleaning stage [D] is timed the same way; with d_seeds the step also loads the seeds and runs LST_PIXEL and
    the three [P] kernels are returned instead."""
    import torch
    cfg = lst.default_config()
    cfg.device, cfg.n_slots, cfg.timing, cfg.store_half = local, N_EVENTS, 1, int(store_half)
    ctx = lst.Lst.from_synth(geom, mmap, cfg)
    streams = [torch.cuda.Stream() for _ in range(N_STREAMS)]
    per = N_EVENTS // N_STREAMS
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    rows = []

    def enqueue(s, st):
        ctx.load_events(s * per, d_in[s * per:(s + 1) * per], stream=st)
        ctx.run_batch(s * per, per, st)
        if with_clean:                                  # optional stage [D], reported beside the path, not in it
            ctx.run_stage(s * per, per, lst.CLEAN, st)
        if d_seeds is not None:                         # optional stage [P]
            ctx.load_seeds(s * per, d_seeds[s * per:(s + 1) * per], stream=st)
            ctx.run_stage(s * per, per, lst.PIXEL, st)

    def collect(s, st, keep):
        ctx.sync_batch(s * per, per, st)
        for k in range(s * per, (s + 1) * per, 16):    # one set of launches per 16 events; times kept on its first slot
            if keep:
                rows.append(ctx.stats(k)["pix_ms"] if d_seeds is not None else ctx.stats(k)["kernel_ms"][:11])

    for rep in range(reps + 2):
        if alone:
            for s in range(N_STREAMS):
                flush.zero_()
                torch.cuda.synchronize()
                enqueue(s, streams[0])
                collect(s, streams[0], rep >= 2)
        else:
            flush.zero_()
            torch.cuda.synchronize()
            for s, st in enumerate(streams):
                enqueue(s, st)
            for s, st in enumerate(streams):
                collect(s, st, rep >= 2)
    ctx.close()
    names = ("seed_bin", "pt3", "pt5") if d_seeds is not None else lst.KERNEL_NAMES
    return dict(zip(names, np.mean(np.asarray(rows), axis=0).tolist())), max(1, per // 16) * N_STREAMS


def csrc_digest() -> str:
    """sha256 over the CUDA sources and the header the library is built from: ties a committed ncu summary to the code it
    was taken on (there is no .git on the GPU box)."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2207_08207_b200", "csrc")
    for f in sorted(os.listdir(d)) + [os.path.join("..", "..", "include", "lst.h")]:
        if f.endswith((".cu", ".cuh", ".h")):
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


NCU_SUMMARY = os.path.join("profiles", "r2_ncu_full_summary.csv")      # r2_ncu_full_summary.digest.txt beside it: "csrc_digest=..." and "commit=..." of the capture


def ncu_traffic_bytes(kernel: str):
    """(bytes, note): dram__bytes_read.sum + dram__bytes_write.sum per 16-event launch of `kernel` from the committed
    `ncu --set full` summary -- a CITATION of that capture, not a measurement of this run; refused (None) when the CUDA
    sources have changed since the capture was taken."""
    import csv
    path = os.path.join(ROOT, NCU_SUMMARY)
    try:
        meta = dict(l.strip().split("=", 1) for l in open(path[:-4] + ".digest.txt") if "=" in l)
        if meta.get("csrc_digest") != csrc_digest():
            return None, f"{NCU_SUMMARY} is stale: taken at csrc digest {meta.get('csrc_digest')}, this run is {csrc_digest()}"
        rows = list(csv.reader(open(path)))
        h = rows[0]
        unit = {"Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "Gbyte": 1e9}
        def col(r, name):
            i = h.index(name)
            return float(r[i]) * unit[rows[1][i]]
        vals = [col(r, "dram__bytes_read.sum") + col(r, "dram__bytes_write.sum")
                for r in rows[2:] if r[h.index("Kernel Name")].startswith("k_" + kernel + "(")]
        if not vals:
            return None, f"{NCU_SUMMARY} has no row for k_{kernel}"
        return sum(vals) / len(vals), (f"cited from {NCU_SUMMARY} (ncu --set full of this code, csrc digest {meta['csrc_digest']}, "
                                      f"commit {meta.get('commit', '?')}; bytes per 16-event launch, kernel alone)")
    except Exception as e:                       # noqa: BLE001
        return None, f"no usable {NCU_SUMMARY}: {e}"


def roofline(kernel_ms, alone_ms, n_hits, needed, cands, peaks, events_per_launch):
    """Per-stage table and the `roofline` object (achieved HBM fraction) for the dominant kernel.
    kernel_ms: average duration of one launch inside the timed 4-stream configuration (kernels of other streams share the
    SMs); alone_ms: the same launch with nothing else on the GPU.  Both from CUDA events the library records around every
    launch on the stream it is launched on.  Bytes / flops are those of ONE launch (`events_per_launch` events).
    The ALU view (SPEC flops of the evaluated candidates / non-FMA fp32 peak = 148 SMs x 128 lanes x sm_max clock; the
    SPEC forbids FMA contraction) is kept beside the HBM view: this path is not bandwidth bound."""
    alu_peak_tflops = 148 * 128 * peaks["sm_max_mhz"] * 1e6 / 1e12
    groups = (("a0_bin", A0_KERNELS), ("a1_md", ("md",)), ("a2_ls", ("seg",)), ("a3_t3", ("t3",)), ("a4_t5", ("t5",)))

    def views(b, fl, ms):
        if not ms:
            return {"ms": ms}
        return {"ms": ms, "hbm_gbs": b / (ms * 1e-3) / 1e9, "hbm_frac": b / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                "hbm_frac_nominal": b / (ms * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
                "alu_tflops": fl / (ms * 1e-3) / 1e12, "alu_frac": fl / (ms * 1e-3) / 1e12 / alu_peak_tflops}

    per_stage = {}
    for i, (name, ks) in enumerate(groups):
        b = algorithmic_bytes(i, n_hits, needed)
        fl = cands[i - 1] * FLOPS_PER_CAND[i - 1] if i else 0
        per_stage[name] = {"algorithmic_bytes": int(b), "spec_flops": int(fl),
                           "kernels_ms_in_step": {k: kernel_ms[k] for k in ks}, "kernels_ms_alone": {k: alone_ms[k] for k in ks},
                           "in_step": views(b, fl, sum(kernel_ms[k] for k in ks)), "alone": views(b, fl, sum(alone_ms[k] for k in ks))}
        per_stage[name]["ms"] = per_stage[name]["in_step"]["ms"]
    top = max(kernel_ms, key=kernel_ms.get)
    si = next(i for i, (_, ks) in enumerate(groups) if top in ks)
    b = algorithmic_bytes(si, n_hits, needed)
    fl = cands[si - 1] * FLOPS_PER_CAND[si - 1] if si else 0
    ins, alo = views(b, fl, kernel_ms[top]), views(b, fl, alone_ms[top])
    traffic, note = ncu_traffic_bytes(top) if events_per_launch == 16 else (None, "launch is not 16 events")
    roof = {"bound": "hbm", "achieved": ins["hbm_gbs"], "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ins["hbm_frac"],
            "traffic": traffic, "traffic_source": note, "kernel": "k_" + top, "algorithmic_bytes": int(b),
            "kernel_ms": kernel_ms[top], "kernel_ms_alone": alone_ms[top], "peak_source": peaks["source"],
            "launch": f"one launch = {events_per_launch} events (grid.y = event); kernel_ms = average launch duration inside the timed "
                      "4-stream configuration (CUDA events on the launching stream), kernel_ms_alone = the same launch with the GPU "
                      "otherwise idle; achieved = algorithmic_bytes / kernel_ms",
            "alone": {"achieved": alo["hbm_gbs"], "frac": alo["hbm_frac"]},
            "nominal": {"peak": NOMINAL_HBM_GBS, "frac": ins["hbm_frac_nominal"], "frac_alone": alo["hbm_frac_nominal"],
                        "what": "the same against the nominal 8 TB/s BASELINE.json quotes (SURVEY 8(d) asks for both)"},
            "alu_view": {"what": "secondary bound: SPEC flops of the evaluated candidates / non-FMA fp32 peak", "spec_flops": int(fl),
                         "peak_tflops": alu_peak_tflops, "in_step": {"achieved_tflops": ins["alu_tflops"], "frac": ins["alu_frac"]},
                         "alone": {"achieved_tflops": alo["alu_tflops"], "frac": alo["alu_frac"]}},
            "why_low": "the path is latency / issue bound, not bandwidth bound: a 16-event batch is L2 resident (traffic < algorithmic "
                       "bytes) and the search is a gather; DESIGN.md section 7"}
    return roof, per_stage


# ------------------------------------------------------------------------------------------
# BASELINE.json configs[4]: occupancy sweep, a0 + mini-doublet + segment kernels only
# ------------------------------------------------------------------------------------------
def run_sweep(args):
    """One JSON line per size (1 k, 10 k, 100 k, 1 M hits on the configs[0] geometry, 50 % track hits): per-kernel
    ms (CUDA events around every launch, median of 5 after 2 warm-ups, L2 flushed), algorithmic HBM GB/s and its
    fraction of the measured peak, evaluated candidates per second.  Capacities are grown from the sizes the
    library reports as needed (LST_ERR_OVERFLOW -> lst_get_stats.needed), as a caller would."""
    import torch
    from paper_2207_08207_b200 import lst, synth
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    geom = synth.make_geometry()
    mmap = make_map(geom, device=0)
    peaks = measured_peaks()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    st = torch.cuda.Stream()
    for n in (1000, 10000, 100000, 1000000):
        ev = synth.generate_occupancy_event(geom, n, seed=4)
        d_in = [torch.from_numpy(a).cuda() for a in (ev.x, ev.y, ev.z, ev.module, ev.side)]
        caps = dict(cap_hits=max(ev.n, 1024), cap_md=max(2 * ev.n, 1024), cap_seg=max(4 * ev.n, 1024), cap_t3=1024, cap_t5=1024)
        for _ in range(4):                       # grow the capacities until MD and LS fit
            cfg = lst.default_config()
            cfg.n_slots, cfg.timing = 1, 1
            for k, v in caps.items():
                setattr(cfg, k, int(v))
            ctx = lst.Lst.from_synth(geom, mmap, cfg)
            ctx.load_events(0, [d_in], stream=st)
            ctx.run_stage(0, 1, lst.MD, st)
            ctx.run_stage(0, 1, lst.SEG, st)
            status = ctx.sync(0, st, check=False)
            need = ctx.stats(0)["needed"]
            if status == lst.OK:
                break
            ctx.close()
            caps["cap_md"] = max(caps["cap_md"], int(1.1 * need[0]) + 1024)
            caps["cap_seg"] = max(caps["cap_seg"], int(1.1 * need[1]) + 1024, 4 * caps["cap_md"])
        assert status == lst.OK, (n, status, need)
        rows = []
        for _ in range(7):
            with torch.cuda.stream(st):
                flush.zero_()
            ctx.load_events(0, [d_in], stream=st)
            ctx.run_stage(0, 1, lst.MD, st)
            ctx.run_stage(0, 1, lst.SEG, st)
            ctx.sync(0, st)
            rows.append(ctx.stats(0)["kernel_ms"][:5])
        stt = ctx.stats(0)
        k_ms = dict(zip(lst.KERNEL_NAMES[:5], np.median(np.asarray(rows[2:]), axis=0).tolist()))
        need, evl, cand = stt["needed"], stt["evaluated"], stt["candidates"]
        per = {}
        for name, ks, stage in (("a0_bin", A0_KERNELS, 0), ("a1_md", ("md",), 1), ("a2_ls", ("seg",), 2)):
            ms = sum(k_ms[k] for k in ks)
            b = algorithmic_bytes(stage, stt["n_hits"], need)
            per[name] = {"ms": ms, "algorithmic_bytes": int(b), "hbm_gbs": b / (ms * 1e-3) / 1e9,
                         "hbm_frac": b / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                         "hbm_frac_nominal": b / (ms * 1e-3) / 1e9 / NOMINAL_HBM_GBS}
            if stage:
                per[name].update(candidates=cand[stage - 1], evaluated=evl[stage - 1], passed=need[stage - 1],
                                 evaluated_per_s=evl[stage - 1] / (ms * 1e-3))
        print(json.dumps({"sweep": "BASELINE.json configs[4]", "hits": ev.n, "kernels_ms": k_ms, "per_stage": per,
                          "rewalks": stt["rewalks"][:2], "capacities": caps, "peak_hbm_gbs": peaks["hbm_gbs"],
                          "peak_source": peaks["source"], "arena_mib": ctx.arena_bytes()[0] / 2 ** 20}))
        ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--profile", action="store_true",
                    help="device-resident steps only (no e2e, per-kernel timing or CPU baseline): the command ncu wraps")
    ap.add_argument("--with-optional", action="store_true", help="with --profile: two more steps that also run LST_CLEAN and LST_PIXEL")
    ap.add_argument("--sweep", action="store_true", help="BASELINE.json configs[4]: occupancy sweep of the a0 / MD / LS kernels")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
