#!/usr/bin/env python
"""bench.py -- throughput of the CDC seed-scan hot path on B200 (BASELINE.json metric: seed-propagations/s).

A "step" is one pass of the whole hot path over one batch of synthetic events: A1 event binning, A2 Hough
pre-vote, A3-A7 RKN propagate-and-score with fused argmax, A8 fp64 re-score of the near-best seeds, A9 labels
(DESIGN.md section 2).  Default workload = BASELINE.json configs[3], the largest fixed single-GPU configuration:
256 events (2/3 single-turn, 1/3 multi-turn, 20 % noise) in the tabulated field, 16^5 = 1,048,576 seeds each,
<= 4500 steps of 2 mm.  One JSON line on stdout (rank 0); configs[1] (the small uniform-field case) is measured
briefly as well and reported under the key "cfg1".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg0|cfg1|cfg2|cfg3] [--events E] [--grid-n G]
    python bench.py --impl reference ...     # the CPU oracle on this box's host cores, same metric
"""
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

from paper_1908_01949_b200 import synth  # noqa: E402

METRIC = "seed_propagations_per_s"
UNIT = "seeds/s"
# Algorithmic FP32 flops (FMA = 2) of the scan kernel's arithmetic, DESIGN.md section 7
FLOPS_STEP = {0: 78.0, 1: 237.0}        # per RKN step, uniform / tabulated field (compensated state included)
# what the kernel executes for the same step: the closed-form map in the uniform field; in the tabulated field two table
# look-ups per step instead of three (the start vertex's B is carried from the previous 4th stage: scan.cu, field reuse)
FLOPS_STEP_EXECUTED = {0: 56.0, 1: 212.0}
FLOPS_LOOKUP, FLOPS_G, FLOPS_APPROACH = 43.0, 22.0, 35.0
PEAK_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # 74.4: 148 SMs x 128 FP32 lanes x 2 x 1965 MHz (B200_PROFILING.md)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=["cfg0", "cfg1", "cfg2", "cfg3"])
    ap.add_argument("--events", type=int, default=0, help="events per GPU (0 = the config's own: 256 for cfg3, else 1)")
    ap.add_argument("--kernel-variant", type=int, default=0, choices=[0, 1, 2, 3],
                    help="0 = production scan kernel, 1 = the two-seeds-per-thread comparison variant, 2 = the lane-refill "
                         "comparison variant, 3 = the production kernel with the field reuse off (A / B)")
    ap.add_argument("--no-secondary", action="store_true", help="skip the short configs[1] measurement")
    ap.add_argument("--shard", default="auto", choices=["auto", "events", "theta"],
                    help="with N GPUs: 'events' = every rank scans its own events (weak scaling, no collective); 'theta' = "
                         "all ranks scan the SAME events, each a slab of the theta axis, exact winners merged by one "
                         "all_gather + one all_reduce (strong scaling); auto = events if the workload has >= N events")
    ap.add_argument("--grid-n", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE.json configs[4]: throughput of the scan over grid size, batch size and step size "
                         "(one JSON line per point; not the driver's bench line)")
    ap.add_argument("--paper-mapping", action="store_true",
                    help="measure the re-created thread mapping of the paper (one block per seed, one thread per fired "
                         "wire) against the product kernel on a sample of the workload's seeds (comparison point)")
    ap.add_argument("--issue-probe", action="store_true",
                    help="issue rates of FFMA / FFMA2 / FADD2 / FMUL2 alone and mixed with integer work (the measurement "
                         "behind the packed pairs of the scan kernel)")
    ap.add_argument("--adaptive", action="store_true",
                    help="SURVEY 8(f) #4: the adaptive-step scan against the fixed step on the workload: steps per seed, "
                         "seeds/s, position difference (one JSON line per tolerance)")
    ap.add_argument("--peel", action="store_true",
                    help="measure the turn-partition peeling loop (cdc_peel_turns, SURVEY 8(f) #3) on the workload's "
                         "events: events/s, partitions found, efficiency / purity against the synthetic truth")
    return ap.parse_args()


def make_workload(args, rank, workload=None):
    cfg_id = int((workload or args.workload)[3:])
    cfg = synth.CONFIGS[cfg_id]
    geom = synth.make_geometry()
    field = synth.make_uniform_field() if cfg.field_kind == 0 else synth.make_table_field()
    n_events = (args.events if workload is None else 0) or cfg.n_events
    events = synth.generate_events_parallel(cfg_id, n_events, rank * n_events)
    n = (args.grid_n if workload is None else 0) or cfg.grid_n
    grids = [synth.truth_anchored_grid(ev.seed, n)[0] for ev in events]
    return cfg_id, cfg, geom, field, events, grids


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe).  The sampler
    runs from before the warm-up; only the samples stamped inside [mark_start, mark_stop] are reported (if the region
    is shorter than the sampling period, the sample nearest to it, flagged with "samples": 0)."""
    Q = "timestamp,clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.proc, self.index, self.t0, self.t1 = [], None, index, None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def mark_start(self):
        self.t0 = time.time()

    def mark_stop(self):
        self.t1 = time.time()

    def stop(self):
        if self.proc:
            time.sleep(0.12)                       # let the sample that covers the end of the region arrive
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                pass
        ok = [(t, r) for t, r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        inside = [r for t, r in ok if self.t0 is not None and self.t0 <= t <= self.t1 + 0.06]
        n_inside = len(inside)
        if not inside and ok:
            mid = 0.5 * ((self.t0 or 0) + (self.t1 or 0))
            inside = [min(ok, key=lambda tr: abs(tr[0] - mid))[1]]
        sm = [float(r[1]) for r in inside]
        mx = [float(r[2]) for r in inside]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in inside for i in range(4) if r[3 + i].lower() == "active"})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": n_inside}


def oracle_sample_time(cfg, geom, field, ev, grid, n_sample, key, fast_build=False):
    """Time the oracle, as it stands, single-threaded, on a stratified sample of the workload's seeds.  fast_build:
    the same source compiled -O3 -march=native with contraction allowed (a second, reported number; never the parity
    build)."""
    import oracle
    if fast_build:
        return oracle.timed_with_fast_build(lambda: oracle_sample_time(cfg, geom, field, ev, grid, n_sample, key))
    sel = synth.stratified_seed_sample(grid.n_seeds, n_sample, key)
    b = oracle.Bound(geom, field, dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm,
                                       eloss=cfg.eloss_MeV_per_mm))
    t0 = time.perf_counter()
    out = oracle.scan(b, ev.wire_id, ev.drift_mm, grid, index_list=sel)
    dt = time.perf_counter() - t0
    return sel.size, int(out["n_steps"].sum()), dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    args.events = args.events or 1                  # the oracle is timed on a sample of event 0's seeds
    cfg_id, cfg, geom, field, events, grids = make_workload(args, 0)
    per_step = 4096
    times, seeds, steps = [], 0, 0
    for i in range(args.warmup + args.steps):
        n, st, dt = oracle_sample_time(cfg, geom, field, events[0], grids[0], per_step, key=1000 + i)
        if i >= args.warmup:
            times.append(dt); seeds += n; steps += st
    total = sum(times)
    val = seeds / total
    sample = f"{per_step} stratified seeds of event 0 per step ({steps / max(seeds, 1):.0f} RKN steps/seed)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            # the workload is the main arm's (same keys, same values); what the oracle was timed on is in `sample`
            "config": {"workload": args.workload, "events_per_gpu": synth.CONFIGS[cfg_id].n_events,
                       "seeds_per_event": grids[0].n_seeds, "max_steps": cfg.max_steps, "h_mm": cfg.h_mm,
                       "field": "table" if cfg.field_kind else "uniform", "hits_event0": len(events[0].wire_id),
                       "sample": sample},
            "rkn_steps_per_s": steps / total,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def measured_traffic(workload):
    """dram bytes per launch of the scan kernel from the committed ncu capture (profiles/), and where it came from."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "scan_kernel_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row["dram_bytes_read"]:
                    return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"] or 0), \
                        f"profiles/scan_kernel_traffic.csv ({row.get('capture', 'ncu --set full')}); not re-measured in this run"
    except OSError:
        pass
    return None, None


def measure(args, workload, steps, warmup, rank, world, local, dist, with_cpu_baseline):
    """One workload through the whole hot path: device-timed arm, end-to-end arm, roofline of the scan kernel."""
    import torch
    from paper_1908_01949_b200 import api, binding as B
    cfg0 = synth.CONFIGS[int(workload[3:])]
    n_ev = (args.events if workload == args.workload else 0) or cfg0.n_events
    theta = args.shard == "theta" or (args.shard == "auto" and world > 1 and n_ev < world)
    cfg_id, cfg, geom, field, events, grids = make_workload(args, 0 if theta else rank,
                                                            None if workload == args.workload else workload)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    E = len(events)
    P = B.scan_params(cfg.h_mm, cfg.max_steps, cfg.window_mm, cfg.eloss_MeV_per_mm, kernel_variant=args.kernel_variant)
    hp = B.hough_params()
    zref = np.array([ev.seed[1] for ev in events], dtype=np.float32)
    if cfg.hough_axes:
        # BJ configs[2]: "Hough pre-vote narrows the ranges": (theta, px, py) axes span the GPU's own Hough ranges, the
        # (z, pz) axes stay truth-anchored; the end-to-end arm does the same inside cdc_find_tracks_host
        Ev0 = sc.upload(off, w, d)
        rg = sc.hough(Ev0, zref)["ranges"]
        Ev0.close()
        for e, g in enumerate(grids):
            lo = g.lo.copy(); hi = g.lo + g.step * (g.n - 1)
            lo[[0, 2, 3]] = rg[e][:, 0]; hi[[0, 2, 3]] = rg[e][:, 1]
            grids[e] = synth.ranges_grid(lo, hi, g.n)
    full_grids = grids
    slab_off = None
    if theta:                                          # this rank's slab of every grid (node values bit-identical to the full grid's)
        grids, slab_off = sc.slabs(full_grids, rank, world)
    n_seeds = sum(g.n_seeds for g, o in zip(grids, slab_off or [0] * len(grids)) if o >= 0)
    specs = B.grid_specs(grids)
    # device-resident inputs and outputs of the device-timed arm
    d_w = torch.tensor(w, device="cuda"); d_d = torch.tensor(d, device="cuda"); d_zref = torch.tensor(zref, device="cuda")
    d_ranges = torch.zeros((E, 3, 2), dtype=torch.float64, device="cuda")
    d_peak = torch.zeros((E, 4), dtype=torch.int32, device="cuda")
    d_key = torch.zeros(E, dtype=torch.int64, device="cuda"); d_seed = torch.zeros(E, dtype=torch.int64, device="cuda")
    d_nm = torch.zeros(E, dtype=torch.int32, device="cuda"); d_c2 = torch.zeros(E, dtype=torch.float64, device="cuda")
    d_lab = torch.zeros(max(int(off[-1]), 1), dtype=torch.int32, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")       # > 126 MB L2

    def step():
        ev = B.Events(sc.geometry, off, d_w, d_d)                                   # A1
        B.cdc_hough_seed_ranges(sc.geometry, ev, hp, -1, d_zref, d_ranges, d_peak)  # A2
        B.cdc_seed_scan(sc.geometry, ev, specs, P, d_key)                           # A3-A7
        B.cdc_best_track(sc.geometry, ev, specs, P, d_key, d_seed, d_nm, d_c2, d_lab)   # A8-A9
        if theta:                                      # exact winners of the slabs -> the event's best seed and labels
            from paper_1908_01949_b200 import dist as D
            torch.cuda.synchronize()
            res = dict(best_seed=d_seed.cpu().numpy(), best_n_match=d_nm.cpu().numpy().astype(np.uint32),
                       best_chi2=d_c2.cpu().numpy(), labels=d_lab.cpu().numpy()[:int(off[-1])])
            merged[0] = D.merge_slab_results_collective(res, slab_off, cfg.window_mm, off, device=torch.device("cuda", local))
        return ev

    merged = [None]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local); sampler.start()
    for _ in range(warmup):
        flush.fill_(1); step().close()
    barrier()
    sampler.mark_start()
    l0 = B.cdc_kernel_launch_count()
    ms, kernel_ms, acc = [], [], {}
    for _ in range(steps):
        flush.fill_(1)
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(); ev = step(); e1.record(); e1.synchronize()
        ms.append(e0.elapsed_time(e1))
        st = B.cdc_scan_get_stats(ev)
        kernel_ms.append(st["kernel_ms"])
        for k, v in st.items():
            acc[k] = acc.get(k, 0) + v
        ev.close()
    barrier()
    sampler.mark_stop()
    launches = B.cdc_kernel_launch_count() - l0
    clocks = sampler.stop()
    best = (d_seed.cpu().numpy().tolist(), d_nm.cpu().numpy().tolist())
    if theta:
        best = (merged[0]["best_seed"].tolist(), merged[0]["best_n_match"].tolist())

    # end to end: host buffers through the C ABI (cdc_find_tracks_host: A1, A2, A3-A9), H2D + D2H inside the timed
    # region, wall clock around the call.  The same steps as the device-timed arm: the Hough vote runs; its ranges
    # replace the (theta, px, py) axes only where the config says so (configs[2])
    pin = lambda a: torch.from_numpy(a).pin_memory().numpy()   # noqa: E731
    h_off, h_w, h_d = off, pin(w), pin(d)
    e2e_grids = grids
    if cfg.hough_axes:
        e2e_grids = [synth.truth_anchored_grid(evn.seed, g.n)[0] for evn, g in zip(events, grids)]   # (z, pz) axes; the rest is replaced
    e2e_steps = max(1, min(steps, 5)) if E >= 64 else steps
    if theta:
        e2e_grids = full_grids                         # the end-to-end call is the one-GPU call: every rank runs the whole event
    sc.find_tracks_host(h_off, h_w, h_d, e2e_grids, P, hp=hp, zref=zref, hough_sets_axes=bool(cfg.hough_axes))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        out = sc.find_tracks_host(h_off, h_w, h_d, e2e_grids, P, hp=hp, zref=zref, hough_sets_axes=bool(cfg.hough_axes))
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    assert out["best_seed"].tolist() == best[0], "end-to-end call and staged calls disagree on the best seeds"
    h2d = int(w.nbytes + d.nbytes + off.nbytes + zref.nbytes + E * 6 * max(int(g.n.max()) for g in grids) * 8)
    d2h = int(E * (8 + 4 + 8 + 8 + 48) + 4 * int(off[-1]))

    total_ms = float(sum(ms))
    t = torch.tensor([total_ms, e2e_s, float(sum(kernel_ms))], dtype=torch.float64, device="cuda")
    cnt = torch.tensor([float(n_seeds), float(acc["n_steps"]), float(E)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX); dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    total_ms, e2e_s, ksum_ms = t.tolist()
    seeds_all, steps_all, events_all = cnt.tolist()
    if theta:
        events_all = float(E)                          # the same events on every rank
        e2e_seeds = float(sum(g.n_seeds for g in full_grids))
    else:
        e2e_seeds = seeds_all
    if rank != 0:
        return None
    K = steps
    flops = FLOPS_STEP[cfg.field_kind] * acc["n_steps"] + FLOPS_LOOKUP * acc["n_lookups"] + \
        FLOPS_G * (acc["n_approach_tests"] + acc["n_g1"]) + FLOPS_APPROACH * acc["n_approaches"]
    k_s = sum(kernel_ms) * 1e-3
    achieved = flops / k_s / 1e12
    traffic, traffic_source = measured_traffic(workload)
    line = {"metric": METRIC, "value": seeds_all * K / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": warmup, "ms_per_step": total_ms / K, "ms_per_step_median": float(np.median(ms)),
            "ms_per_step_max": float(np.max(ms)), "higher_is_better": True, "scaling": "strong" if theta else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload, "events_per_gpu": E, "seeds_per_event": grids[0].n_seeds,
                       "max_steps": cfg.max_steps, "h_mm": cfg.h_mm, "field": "table" if cfg.field_kind else "uniform",
                       "hits_per_event": int(off[-1]) // E, "l2": "flushed between steps (256 MB write)",
                       "seed_axes": "theta, px, py from the Hough ranges; z, pz truth-anchored" if cfg.hough_axes
                       else "truth-anchored (the Hough vote runs, its ranges are not used for the grid)",
                       "kernel_variant": args.kernel_variant,
                       "parallelism": (f"theta{world} (every rank scans a theta slab of the same events; exact winners merged "
                                       f"by one all_gather + one all_reduce(MAX), a few bytes per event)") if theta
                       else f"dp{world} (events sharded over ranks, no data-path collective)"},
            "rkn_steps_per_s": steps_all * 1.0 / (total_ms * 1e-3), "events_per_s": events_all * K / (total_ms * 1e-3),
            "scan_kernel_ms": sum(kernel_ms) / K, "scan_kernel_share": ksum_ms / total_ms,
            "rkn_steps_per_s_kernel": acc["n_steps"] / k_s,
            "candidate_pool": {"entries_per_step": acc["n_pool"] / K, "capacity": int(st["pool_cap"])},
            "clocks": clocks,
            "e2e": {"value": e2e_seeds / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "call": "cdc_find_tracks_host (A1, A2 Hough vote, A3-A9)"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": PEAK_FP32_TFLOPS, "unit": "TFLOP/s",
                         "frac": achieved / PEAK_FP32_TFLOPS, "traffic": traffic, "traffic_source": traffic_source,
                         "kernel": "seed_scan_kernel",
                         "flops_per_rkn_step": flops / max(acc["n_steps"], 1),
                         "note": "flops = the step as the method defines it (DESIGN.md section 7)" +
                                 ("; the tabulated-field kernel carries B at a step's start vertex over from the previous "
                                  "step's 4th-stage point (within half an ulp32 of B): it executes 212 instead of 237 "
                                  "flops per step" if cfg.field_kind else
                                  "; the uniform-field kernel executes its closed form, 56 instead of 78 flops per step"),
                         "frac_executed": (achieved - (FLOPS_STEP[cfg.field_kind] - FLOPS_STEP_EXECUTED[cfg.field_kind]) *
                                           acc["n_steps"] / k_s / 1e12) / PEAK_FP32_TFLOPS,
                         "peak_source": "148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (nominal, B200_PROFILING.md; "
                                        "MEASURED_PEAKS.json has no FP32 figure)"}}
    f, _ = B.cdc_fp32_peak_probe(4096)
    line["roofline"]["ffma_probe_tflops"] = f / 1e12
    line["roofline"]["frac_of_probe"] = achieved / (f / 1e12)
    if with_cpu_baseline:
        n, st_, dt = oracle_sample_time(cfg, geom, field, events[0], grids[0], 32768 if cfg_id < 3 else 65536, key=77)
        line["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{n} stratified seeds of event 0 ({st_} RKN steps, {dt:.1f} s)",
                                "rkn_steps_per_s": st_ / dt}
        # the same oracle as N independent single-threaded processes over disjoint seed ranges
        import oracle
        ncore = os.cpu_count() or 1
        sel = synth.stratified_seed_sample(grids[0].n_seeds, 4 * n, 78)
        t0 = time.perf_counter()
        o = oracle.scan_parallel(geom, field, dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm,
                                                   eloss=cfg.eloss_MeV_per_mm), events[0].wire_id, events[0].drift_mm,
                                 grids[0], index_list=sel, n_proc=ncore)
        dtn = time.perf_counter() - t0
        line["cpu_baseline"]["all_cores"] = {"value": sel.size / dtn, "unit": UNIT, "cores": ncore,
                                             "rkn_steps_per_s": int(o["n_steps"].sum()) / dtn,
                                             "sample": f"{sel.size} stratified seeds over {ncore} processes ({dtn:.1f} s)"}
        # the parity build (-O2, no contraction) is a slow denominator; the same source built for speed
        try:
            n2, st2, dt2 = oracle_sample_time(cfg, geom, field, events[0], grids[0], n, key=77, fast_build=True)
            line["cpu_baseline"]["o3_native_build"] = {"value": n2 / dt2, "unit": UNIT, "cores": 1,
                                                       "flags": "-O3 -march=native -ffp-contract=fast",
                                                       "rkn_steps_per_s": st2 / dt2}
        except Exception as exc:                          # noqa: BLE001 -- a reported extra, never fatal
            line["cpu_baseline"]["o3_native_build"] = {"unavailable": str(exc)[:120]}
    sc.close()
    return line


def run_ours(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "WARN")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    line = measure(args, args.workload, args.steps, args.warmup, rank, world, local, dist, not args.no_cpu_baseline)
    if args.workload != "cfg1" and not args.no_secondary:
        # the small uniform-field case (BASELINE.json configs[1]), briefly: a second object, not the headline
        sec = measure(args, "cfg1", max(3, min(args.steps, 10)), 3, rank, world, local, dist, False)
        if rank == 0:
            line["cfg1"] = {k: sec[k] for k in ("value", "unit", "ms_per_step", "scan_kernel_ms", "rkn_steps_per_s_kernel",
                                                "config", "roofline", "e2e", "steps", "warmup")}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """configs[4] as a star: grid n in {8,12,16,24,32} at batch 1; batch in {1,...,1024} at 16^5;
    h in {1,2,4} mm at 16^5 x 16 events (max_steps = 9000 mm / h).  Field, hits and noise of configs[3].  Beyond 64 events the
    batch repeats the 64 generated ones (their hit tables are still uploaded and scanned separately)."""
    import dataclasses
    import torch
    from paper_1908_01949_b200 import api, binding as B
    torch.cuda.set_device(0)
    cfg = synth.CONFIGS[4]
    geom = synth.make_geometry(); field = synth.make_table_field()
    base = synth.generate_events(cfg, geom, field, 64)
    sc = api.SeedScanner(geom, field)
    points = [("grid", n, 1, 2.0) for n in (8, 12, 16, 24, 32)] + \
             [("batch", 16, b, 2.0) for b in (1, 4, 16, 64, 256, 1024)] + [("step", 16, 16, h) for h in (1.0, 2.0, 4.0)]
    for axis, n, batch, h in points:
        events = [base[i % len(base)] for i in range(batch)]
        grids = [synth.truth_anchored_grid(ev.seed, n)[0] for ev in events]
        off, w, d = synth.pack_hits(events)
        specs = B.grid_specs(grids)
        P = B.scan_params(h, int(round(9000.0 / h)), cfg.window_mm)
        ev = B.Events(sc.geometry, off, w, d)
        d_key = torch.zeros(batch, dtype=torch.int64, device="cuda")
        ms = []
        for it in range(3):
            B.cdc_seed_scan(sc.geometry, ev, specs, P, d_key)
            st = B.cdc_scan_get_stats(ev)
            if it:
                ms.append(st["kernel_ms"])
        t = float(np.mean(ms)) * 1e-3
        flops = FLOPS_STEP[1] * st["n_steps"] + FLOPS_LOOKUP * st["n_lookups"] + \
            FLOPS_G * (st["n_approach_tests"] + st["n_g1"]) + FLOPS_APPROACH * st["n_approaches"]
        print(json.dumps({"sweep_axis": axis, "grid_n": n, "events": batch, "h_mm": h, "seeds": st["n_seeds"],
                          "rkn_steps": st["n_steps"], "kernel_ms": t * 1e3, "seeds_per_s": st["n_seeds"] / t,
                          "rkn_steps_per_s": st["n_steps"] / t, "events_per_s": batch / t,
                          "tflops": flops / t / 1e12, "frac_fp32_peak": flops / t / 1e12 / PEAK_FP32_TFLOPS}), flush=True)
        ev.close()


def run_paper_mapping(args):
    """seeds/s of the paper's v1 mapping on this GPU, same event, same grid, a stratified
    sample of the seeds; the product kernel is timed on the whole grid."""
    import torch
    from paper_1908_01949_b200 import api, binding as B
    torch.cuda.set_device(0)
    cfg_id, cfg, geom, field, events, grids = make_workload(args, 0)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    ev = B.Events(sc.geometry, off, w, d)
    P = B.scan_params(cfg.h_mm, cfg.max_steps, cfg.window_mm)
    n = 8192
    sel = synth.stratified_seed_sample(grids[0].n_seeds, n, key=4)
    d_sel = torch.tensor(sel, dtype=torch.int64, device="cuda")
    d_nm = torch.zeros(n, dtype=torch.int32, device="cuda"); d_c2 = torch.zeros(n, dtype=torch.float32, device="cuda")
    ms = []
    for it in range(3):
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); e0.record()
        B.cdc_seed_scan_paper_mapping(sc.geometry, ev, 0, grids[0], P, d_sel, d_nm, d_c2)
        e1.record(); e1.synchronize()
        if it:
            ms.append(e0.elapsed_time(e1))
    ms2 = []
    for it in range(3):                      # the two-kernel mapping: record, then DCA per wire
        k = B.cdc_seed_scan_paper_mapping_v2(sc.geometry, ev, 0, grids[0], P, d_sel, d_nm, d_c2, timed=True)
        if it:
            ms2.append(k)
    d_key = torch.zeros(len(events), dtype=torch.int64, device="cuda")
    for it in range(3):
        B.cdc_seed_scan(sc.geometry, ev, B.grid_specs(grids), P, d_key)
        st = B.cdc_scan_get_stats(ev)
    t_v1 = float(np.mean(ms)) * 1e-3
    k1, k2 = (float(v) * 1e-3 for v in np.mean(ms2, axis=0))
    ours = st["n_seeds"] / (st["kernel_ms"] * 1e-3)
    print(json.dumps({"comparison": "paper_v1_mapping", "workload": args.workload, "hits": int(off[1]), "sample_seeds": n,
                      "paper_mapping_ms": t_v1 * 1e3, "paper_mapping_seeds_per_s": n / t_v1,
                      "product_kernel_seeds_per_s": ours, "ratio": ours / (n / t_v1)}))
    print(json.dumps({"comparison": "paper_v2_mapping", "workload": args.workload, "hits": int(off[1]), "sample_seeds": n,
                      "record_kernel_ms": k1 * 1e3, "dca_kernel_ms": k2 * 1e3, "record_bytes": 32 * n * (cfg.max_steps + 1),
                      "paper_mapping_seeds_per_s": n / (k1 + k2), "product_kernel_seeds_per_s": ours,
                      "ratio": ours / (n / (k1 + k2))}))


def run_peel(args):
    """the event reconstruction loop without the fit.  Partition 0's grid is the workload's own;
    the following partitions use 8^5 nodes centred on the extrapolated seed with the paper's quoted resolutions as
    half-widths.  One partition's track is at most max_steps / n_turns steps long."""
    import torch
    from paper_1908_01949_b200 import api, binding as B
    torch.cuda.set_device(0)
    cfg_id, cfg, geom, field, events, grids = make_workload(args, 0)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    ev = B.Events(sc.geometry, off, w, d)
    steps = 1500
    P = B.scan_params(cfg.h_mm, steps, cfg.window_mm, cfg.eloss_MeV_per_mm)
    hw = [0.01, 26.0, 2.5, 2.5, 1.7]
    ms, ms_ad = [], []
    n0 = B.cdc_kernel_launch_count()
    for it in range(args.warmup + args.steps):
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); e0.record()
        out = B.cdc_peel_turns(sc.geometry, ev, B.grid_specs(grids), P, [8] * 5, hw, max_partitions=4)
        e1.record(); e1.synchronize()
        if it == args.warmup - 1:
            n0 = B.cdc_kernel_launch_count()
        if it >= args.warmup:
            ms.append(e0.elapsed_time(e1))
    n1 = B.cdc_kernel_launch_count()
    for it in range(args.warmup + args.steps):       # the same with the adaptive extrapolation between partitions
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); e0.record()
        out_ad = B.cdc_peel_turns(sc.geometry, ev, B.grid_specs(grids), P, [8] * 5, hw, max_partitions=4,
                                  extrap_tol=1e-4, extrap_h_max=16.0)
        e1.record(); e1.synchronize()
        if it >= args.warmup:
            ms_ad.append(e0.elapsed_time(e1))
    launches = (n1 - n0) // max(args.steps, 1)
    # Eq. (2), (3) against the generator's truth turns, by the library's own kernel (not part of the timed region)
    truth = torch.tensor(np.concatenate([e.truth_turn for e in events]).astype(np.int32), device="cuda")
    q = B.cdc_classification_quality(ev, 3, out["d_partition"], truth)
    eff, pur, found = [], [], 0
    for e, evt in enumerate(events):
        eff += [float(v) for v in q["efficiency"][e][:evt.n_turns] if v >= 0]
        pur += [float(v) for v in q["purity"][e][:evt.n_turns] if v >= 0]
        found += int(out["n_partitions"][e] >= evt.n_turns)
    t = float(np.mean(ms)) * 1e-3
    print(json.dumps({"measurement": "turn_peeling", "workload": args.workload, "events": len(events),
                      "seeds_partition0": int(grids[0].n_seeds), "seeds_next": 8 ** 5, "max_steps": steps,
                      "ms_per_call": t * 1e3, "events_per_s": len(events) / t, "kernel_launches_per_call": int(launches),
                      "ms_per_call_adaptive_extrapolation": float(np.mean(ms_ad)),
                      "adaptive_same_partitions": bool(np.array_equal(out["partition"], out_ad["partition"])),
                      "partitions_found": [int(v) for v in out["n_partitions"]], "true_turns": [e.n_turns for e in events],
                      "status": [int(v) for v in out["status"]], "events_with_all_turns": found,
                      "mean_efficiency": float(np.mean(eff)) if eff else None,
                      "mean_purity": float(np.mean(pur)) if pur else None}))


def run_issue_probe(args):
    import torch
    from paper_1908_01949_b200 import binding as B
    torch.cuda.set_device(0)
    names = ["FFMA", "FFMA2", "FADD", "FADD2", "FMUL2", "FFMA2 + LOP3", "FFMA + LOP3", "FFMA2 + FFMA"]
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    for mode, name in enumerate(names):
        ms, wi, fl = B.cdc_fp32_issue_probe(mode, 4096)
        print(json.dumps({"probe": name, "ms": ms, "tflops": fl / ms * 1e-9,
                          "warp_inst_per_clk_per_smsp_at_1965MHz": wi / (ms * 1e-3) / (sm * 4 * 1.965e9)}))


def run_adaptive(args):
    """Adaptive step against the fixed step on the same events and grids: kernel time, accepted steps per seed, and how
    far the adaptive track ends from the fixed-step one (different path lengths by up to one long step are excluded:
    only seeds that ended by the path cap at equal units are compared)."""
    import torch
    from paper_1908_01949_b200 import api, binding as B
    torch.cuda.set_device(0)
    args.events = args.events or (4 if args.workload == "cfg3" else 1)
    cfg_id, cfg, geom, field, events, grids = make_workload(args, 0)
    sc = api.SeedScanner(geom, field)
    off, w, d = synth.pack_hits(events)
    P = B.scan_params(cfg.h_mm, cfg.max_steps, cfg.window_mm, cfg.eloss_MeV_per_mm)
    E = sc.upload(off, w, d)
    fx = sc.scan(E, grids, P, per_seed=True, debug=True, best=False)
    fx = sc.scan(E, grids, P, per_seed=True, debug=True, best=False)
    n_seeds = fx["stats"]["n_seeds"]
    print(json.dumps({"propagator": "fixed", "workload": args.workload, "events": len(events), "h_mm": cfg.h_mm,
                      "kernel_ms": fx["stats"]["kernel_ms"], "seeds_per_s": n_seeds / (fx["stats"]["kernel_ms"] * 1e-3),
                      "steps_per_seed": fx["stats"]["n_steps"] / n_seeds, "note": "TRACK variant (debug records on)"}))
    for tol, h_max in ((1e-6, 8.0), (1e-5, 8.0), (1e-4, 8.0)):
        ad = sc.scan_adaptive(E, grids, P, tol, h_max)
        ad = sc.scan_adaptive(E, grids, P, tol, h_max)
        same = ad["debug"]["pad"] == fx["debug"]["n_steps"]
        dpos = np.sqrt(sum((ad["debug"][k] - fx["debug"][k]) ** 2 for k in ("x", "y", "z")))
        dn = ad["n_match"].astype(np.int64) - fx["n_match"].astype(np.int64)
        print(json.dumps({"propagator": "adaptive", "tol_mm": tol, "h_max_mm": h_max, "kernel_ms": ad["stats"]["kernel_ms"],
                          "seeds_per_s": n_seeds / (ad["stats"]["kernel_ms"] * 1e-3),
                          "steps_per_seed": ad["stats"]["n_steps"] / n_seeds,
                          "path_units_per_seed": ad["stats"]["n_gas_steps"] / n_seeds,
                          "steps_per_level": ad["n_level"].sum(axis=0).tolist(),
                          "seeds_ending_at_equal_path": float(same.mean()),
                          "max_position_difference_mm_at_equal_path": float(dpos[same].max()) if same.any() else None,
                          "n_match_differs_on_fraction": float((dn != 0).mean()),
                          "best_seed_same": bool(np.array_equal(ad["S32_argmax"], fx["S32_argmax"]))}))


if __name__ == "__main__":
    a = parse()
    if a.issue_probe:
        run_issue_probe(a)
    elif a.adaptive:
        run_adaptive(a)
    elif a.peel:
        run_peel(a)
    elif a.paper_mapping:
        run_paper_mapping(a)
    elif a.sweep:
        run_sweep(a)
    else:
        run_reference(a) if a.impl == "reference" else run_ours(a)
