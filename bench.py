#!/usr/bin/env python
"""bench.py -- particle-bounces/s of the TPMC hot path (seed -> trace -> reflect -> accumulate -> reduce).

Headline (default, `--config C5`): synthetic config C5 of BASELINE.json, the ~1.0e6-facet procedural body, 70 % O /
30 % He, T_inf = 900 K, |V| = 7700 m/s, N = 1e9 particles per attitude of the 64-attitude sweep.  `--config C1..C4`
times the other four configs at the sizes of SURVEY 8(d) (their bench lines are recorded in DESIGN.md section 7).

One "step" = one tpmc_run of N particles at one point of the config's sweep (the whole hot path over one batch).
  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl tpmc|reference] [--config C5] [--particles N]
N > 1: launched by torchrun, one rank per GPU; rank r runs sweep points r, r+N, ... (weak scaling, no data-path
collective: sweep points are independent problems); value = all ranks' bounces / max time.
`--split slices` is the other split of SURVEY 8(e): every rank runs its particle range of the SAME sweep point and the
outputs are all-reduced (NCCL, SUM) inside the timed region (strong scaling).
Prints ONE JSON line on rank 0 (contract in DESIGN.md "Measurement").
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import tpmc_inputs as ti

METRIC = "particle_bounces_per_s"
UNIT = "bounces/s"
WORKLOADS = {
    "C1": "C1: flat plate, 2 two-sided facets, normal 30 deg to the stream, O, 1000 K, 7500 m/s, N = 1e5",
    "C2": "C2: geodesic sphere, 20480 facets, O, 7500 m/s, S in {2, 5, 8}, N = 1e7 per run",
    "C3": "C3: capped cylinder, 2048 facets, Maxwell sigma = 0.8, axis at 0/45/90 deg, N = 1e8 per run",
    "C4": "C4: concave satellite (bus + pocket + 2 canted panels), 50160 facets, 16 pitch angles, N = 1e8 per run",
    "C5": "C5: ~1.0e6-facet noise-displaced geodesic body + 6 panels, O/He 70/30, 900 K, 7700 m/s",
}


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json, copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(config: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one steady-state k_trace_wf launch, from the tracked summary of
    the latest `ncu --set full` capture in this launch configuration (profiles/trace_traffic.json names the capture)."""
    p = os.path.join(ROOT, "profiles", "trace_traffic.json")
    if os.path.exists(p):
        d = json.load(open(p))
        if config in d:
            return d[config]["dram_bytes_per_launch"], d[config]["source"]
    return None, None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region."""

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) >= 6 and r[2 + k] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def attitude_index(step: int, rank: int, world: int, n_attitudes: int) -> int:
    """Which point of the sweep a rank runs at a step: ranks take disjoint points (weak scaling)."""
    return (step * world + rank) % n_attitudes


def reduce_over_ranks(times, totals, world: int, device=None):
    """MAX of the per-rank times and SUM of the per-rank totals (the only collective, after the timed region)."""
    import torch
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    tot = torch.tensor(list(totals), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return t.tolist(), tot.tolist()


def sum_slices(parts, world: int, device=None):
    """The other split of SURVEY 8(e): ranks run disjoint (first, count) slices of ONE run and the outputs (force,
    torque, per-facet momentum: slices are additive) are summed across ranks.  parts: list of tensors."""
    import torch
    out = [torch.as_tensor(p, dtype=torch.float64, device=device).clone() for p in parts]
    if world > 1:
        import torch.distributed as dist
        for t in out:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return out


def slice_of(rank: int, world: int, N: int):
    """Contiguous particle range of a rank: (first, count), covering [0, N) without overlap."""
    per = N // world
    first = rank * per
    return first, (N - first if rank == world - 1 else per)


def split_plan(split: str, step: int, rank: int, world: int, n_attitudes: int, N: int):
    """What a rank runs at a step: (sweep point, first particle, particle count).
    "attitudes": ranks take disjoint sweep points, each the whole stream (independent problems, no exchange).
    "slices": every rank runs its contiguous range of the SAME point's stream (particles are independent);
    the outputs are then summed across ranks (allreduce_outputs) -- the split of SURVEY 8(e)."""
    if split == "slices":
        first, count = slice_of(rank, world, N)
        return step % n_attitudes, first, count
    return attitude_index(step, rank, world, n_attitudes), 0, N


def allreduce_outputs(tensors, world: int):
    """The one exchange step of the "slices" split: in-place SUM over ranks of a slice's force, torque and per-facet
    momentum (3 + 3 + 3 nt doubles; NCCL on the device under torchrun, gloo on CPU tensors in the tests)."""
    if world > 1:
        import torch.distributed as dist
        for t in tensors:
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return tensors


def oracle_sample(cfgs, count_per_thread, threads):
    """The oracle, as it stands, on a bounded slice of the same workload, one slice per host thread."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    m = cfgs[0].mesh()
    om = oracle.OracleMesh(m.vertices, m.indices, m.flags)
    cfg = cfgs[0]
    count_per_thread = max(1, min(count_per_thread, cfg.N // threads))

    def work(k):
        return om.run(cfg, first=k * count_per_thread, count=count_per_thread, debug=False, facets=False)

    t0 = time.perf_counter()
    with ThreadPoolExecutor(threads) as ex:
        res = list(ex.map(work, range(threads)))
    dt = time.perf_counter() - t0
    hits = sum(r.hits for r in res)
    return hits, dt, count_per_thread * threads


def run_reference(args, cfgs, rank):
    """--impl reference: the CPU oracle (there is no third-party implementation of this paper)."""
    if rank != 0:
        return
    threads = os.cpu_count() or 1
    per = max(1000, int(args.ref_particles // threads))
    oracle_sample(cfgs, 2000, threads)                       # builds the oracle mesh, warms caches
    for _ in range(max(args.warmup, 0)):
        oracle_sample(cfgs, max(per // 10, 1000), threads)
    tot_hits, tot_t, n = 0, 0.0, 0
    for _ in range(args.steps):
        h, dt, n = oracle_sample(cfgs, per, threads)
        tot_hits += h
        tot_t += dt
    val = tot_hits / tot_t
    sample = f"{n} particles per step ({threads} slices) of the N={cfgs[0].N:.0e} stream, sweep point 0"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "particles_per_step": n, "facets": cfgs[0].mesh().nt},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tpmc", choices=["tpmc", "reference"])
    ap.add_argument("--config", default="C5", choices=sorted(WORKLOADS))
    ap.add_argument("--particles", type=float, default=None, help="override N per step (default: the config's)")
    ap.add_argument("--ref-particles", type=float, default=4_000_000, help="oracle particles per reference step")
    ap.add_argument("--cpu-baseline-particles", type=float, default=80_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-peaks", action="store_true")
    ap.add_argument("--split", default="attitudes", choices=["attitudes", "slices"],
                    help="N > 1: ranks take disjoint sweep points (default, weak scaling, no exchange), or disjoint particle "
                         "ranges of the same point with an all-reduce of the outputs inside the timed region (strong scaling)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    cfgs = ti.config(args.config)
    if args.particles:
        cfgs = [c.with_(N=int(args.particles)) for c in cfgs]

    if args.impl == "reference":
        run_reference(args, cfgs, rank)
        return

    import torch
    import torch.distributed as dist

    import paper_1312_3691_b200 as tpmc

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the TPMC hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    m = cfgs[0].mesh()
    mesh = tpmc.Mesh(m.vertices, m.indices, m.flags)
    info = mesh.info()
    N = cfgs[0].N
    stream = torch.cuda.current_stream()
    force = torch.empty(3, dtype=torch.float64, device=dev)
    torque = torch.empty(3, dtype=torch.float64, device=dev)
    facets = torch.empty((mesh.nt, 3), dtype=torch.float64, device=dev)
    L = tpmc.lib()
    import ctypes as C

    # C5's structure (149 MB) and its per-wave lists exceed the 126 MB L2; the small configs fit, so their L2 is flushed
    # between steps by writing a 512 MB buffer (outside the per-step event pairs).
    flush = None if args.config == "C5" else torch.empty(512 << 20, dtype=torch.uint8, device=dev)

    slices = args.split == "slices"
    my_count = split_plan(args.split, 0, rank, world, len(cfgs), N)[2]

    def step(k, stats=None, flags=0):
        att, first, count = split_plan(args.split, k, rank, world, len(cfgs), N)
        p, keep = tpmc.make_params(cfgs[att], first=first, count=count, flags=flags)
        rc = L.tpmc_run(mesh._h, C.byref(p), stream.cuda_stream or None, force.data_ptr(), torque.data_ptr(),
                        facets.data_ptr(), None if stats is None else C.byref(stats), None)
        if rc != 0:
            raise SystemExit(f"tpmc_run failed: {rc} {L.tpmc_last_cuda_error().decode()}")
        if slices:      # the exchange step, inside the timed region: every rank ends the step with the whole run's outputs
            allreduce_outputs([force, torque, facets], world)

    # ---- warm-up (untimed)
    for k in range(args.warmup):
        step(k)
    barrier()

    # ---- timed: exactly K steps, device-resident, CUDA events on the launching stream
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    if flush is None:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for k in range(args.steps):
            step(args.warmup + k)
        e1.record(stream)
        barrier()
        ms_total = e0.elapsed_time(e1)
    else:
        evs = []
        for k in range(args.steps):
            flush.fill_(k & 0xFF)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            step(args.warmup + k)
            b.record(stream)
            evs.append((a, b))
        barrier()
        ms_total = sum(a.elapsed_time(b) for a, b in evs)
    clocks = sampler.stop()

    # ---- one more pass per timed sweep point with stats on: hits (the metric's numerator) and the
    #      per-kernel event times for the roofline.  Same work, same stream; not part of `value`'s clock.
    tot = {}
    keys = ["hits", "segments", "kernel_launches", "ms_seed", "ms_trace", "ms_reflect", "ms_finish", "ms_sort", "ms",
            "timed_waves", "node_visits", "tri_tests", "culled", "trace_launches", "traced_rays", "overflow_rays"]
    for k in range(args.steps):
        st = tpmc.tpmc_stats()
        step(args.warmup + k, st)
        for f in keys:
            tot[f] = tot.get(f, 0) + getattr(st, f)
    barrier()
    # ---- and once more with the seed kernels of the next wave BEHIND trace/reflect instead of beside them
    #      (TPMC_FLAG_SERIAL_SEED; same kernels, same grids, same arguments): the event pair around a launch then
    #      brackets that kernel alone, not the kernel plus whatever share of the SMs the other stream took meanwhile.
    #      The roofline's launch duration is taken from this pass; the overlapped one is reported beside it.
    ser = {}
    for k in range(args.steps):
        st = tpmc.tpmc_stats()
        step(args.warmup + k, st, flags=tpmc.TPMC_FLAG_SERIAL_SEED)
        for f in ("ms", "ms_seed", "ms_trace", "ms_reflect", "ms_finish", "ms_sort", "trace_launches", "traced_rays"):
            ser[f] = ser.get(f, 0) + getattr(st, f)
    barrier()
    hits, segs, launches = tot["hits"], tot["segments"], tot["kernel_launches"]

    # ---- end to end: host buffers through tpmc_run_host (params H2D, results D2H inside the region)
    e2e = None
    if not args.no_e2e:
        hF, hT = np.empty(3), np.empty(3)
        hP_t = torch.empty((mesh.nt, 3), dtype=torch.float64).pin_memory()
        hP = hP_t.numpy()
        att0, first0, count0 = split_plan(args.split, args.warmup, rank, world, len(cfgs), N)
        p0, keep0 = tpmc.make_params(cfgs[att0], first=first0, count=count0)
        L.tpmc_run_host(mesh._h, C.byref(p0), stream.cuda_stream or None, hF.ctypes.data, hT.ctypes.data, hP.ctypes.data, None)
        barrier()
        e2e_s = 0.0
        t0 = time.perf_counter()
        for k in range(args.steps):
            if flush is not None:            # same rule as the device-timed loop: L2 flushed between steps, outside the clock
                flush.fill_(k & 0xFF)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
            if slices and world > 1:
                # host buffers at the end of the step need the exchange first: device run, all-reduce, then the D2H copies
                step(args.warmup + k)
                hP_t.copy_(facets, non_blocking=True)
                hFT = torch.cat([force, torque]).cpu()
                torch.cuda.synchronize()
            else:
                att, first, count = split_plan(args.split, args.warmup + k, rank, world, len(cfgs), N)
                p, keep = tpmc.make_params(cfgs[att], first=first, count=count)
                rc = L.tpmc_run_host(mesh._h, C.byref(p), stream.cuda_stream or None, hF.ctypes.data, hT.ctypes.data,
                                     hP.ctypes.data, None)           # returns after its own stream synchronisation
                if rc != 0:
                    raise SystemExit(f"tpmc_run_host failed: {rc}")
            if flush is not None:
                e2e_s += time.perf_counter() - t0
        barrier()
        if flush is None:
            e2e_s = time.perf_counter() - t0
        e2e = {"hits": hits, "s": e2e_s}

    peaks = None
    if rank == 0 and not args.no_peaks:
        peaks = tpmc.tpmc_measure_peaks()

    # ---- max over ranks, totals over ranks
    (ms_total_max, e2e_s_max), (hits_all, segs_all, parts_all) = reduce_over_ranks(
        [ms_total, e2e["s"] if e2e else 0.0], [hits, segs, my_count * args.steps], world, dev)

    if rank == 0:
        value = hits_all / (ms_total_max * 1e-3)
        hbm, hbm_src = hbm_peak()
        traced, nodes, tris = tot["traced_rays"], tot["node_visits"], tot["tri_tests"]
        launches_trace = max(tot["trace_launches"], 1)         # k_trace_wf launches, rays they processed
        avg_ms_overlapped = tot["ms_trace"] / launches_trace   # seed kernels of the next wave share the SMs meanwhile
        avg_ms = ser["ms_trace"] / max(ser["trace_launches"], 1)   # the kernel alone (serialised pass)
        depth = int(np.ceil(np.log2(max(mesh.nt, 2))))
        # Algorithmic work per segment: ceil(log2 T) nodes x 64 B + one triangle of
        # 48 B + 32 B ray in + 8 B result out; ceil(log2 T) node visits x 2 slab tests x 18 ops + one facet test of 60 ops.
        per_seg_bytes = depth * 64 + 48 + 32 + 8
        per_seg_ops = depth * 2 * 18 + 60
        rays_per_launch = traced / launches_trace
        t = avg_ms * 1e-3
        alg_bw = rays_per_launch * per_seg_bytes / t / 1e9 if t > 0 else 0.0                  # GB/s
        alg_ops = rays_per_launch * per_seg_ops / t / 1e12 if t > 0 else 0.0                  # T lane-op/s
        fetched_bw = (nodes * 64 + tris * 48) / launches_trace / t / 1e9 if t > 0 else 0.0    # what the kernel really gathers (64-byte wide nodes)
        ms_stat = tot["ms"]
        traffic, traffic_src = ncu_traffic(args.config)
        roof = {"kernel": "k_trace_wf", "segments_per_launch": rays_per_launch, "avg_launch_ms": avg_ms,
                "avg_launch_ms_overlapped": avg_ms_overlapped,
                "timing": "CUDA events around every k_trace_wf launch on its stream, in a pass with the seed kernels of the next "
                          "wave enqueued behind trace/reflect (TPMC_FLAG_SERIAL_SEED) so that the bracket holds this kernel alone; "
                          "avg_launch_ms_overlapped is the same bracket in the normal, overlapped schedule",
                "ms_per_step_serialised": ser["ms"] / args.steps,
                "share_of_step_serialised": {k: (ser[f] / ser["ms"] if ser.get("ms") else None) for k, f in
                                             (("seed+precull", "ms_seed"), ("k_trace_wf", "ms_trace"), ("k_reflect", "ms_reflect"),
                                              ("k_finish_final", "ms_finish"))},
                "launches_timed": int(launches_trace), "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes_per_segment": per_seg_bytes, "algorithmic_ops_per_segment": per_seg_ops,
                "nodes_per_traced_segment": nodes / max(traced, 1), "tri_tests_per_traced_segment": tris / max(traced, 1),
                "share_of_step": {k: (tot[f] / ms_stat if ms_stat else None) for k, f in
                                  (("seed+precull", "ms_seed"), ("sort", "ms_sort"), ("k_trace_wf", "ms_trace"),
                                   ("k_reflect", "ms_reflect"), ("k_finish_final", "ms_finish"))}}
        if peaks:
            # ncu (profiles/) shows the L1TEX data pipe as the busiest unit of k_trace_wf (scattered 32-byte gathers that
            # hit L2), then instruction issue; DRAM is a few per cent.  Binding roofline: the gather path, against the
            # measured rate of independent 32-byte gathers over an array of the structure's size at this kernel's
            # residency.  The fp32-issue and HBM views are reported beside it.
            gpk = peaks["gather64_bytes_per_s"] / 1e9
            t_ov = avg_ms_overlapped * 1e-3
            roof.update({"bound": "l2-gather", "achieved": alg_bw, "peak": gpk, "unit": "GB/s", "frac": alg_bw / gpk,
                         # `value` is timed in the overlapped schedule (the next wave's seed kernels share the SMs), `frac` on
                         # the kernel alone; the same ratio with the overlapped launch duration:
                         "frac_as_scheduled": (rays_per_launch * per_seg_bytes / t_ov / 1e9 / gpk) if t_ov > 0 else None,
                         "peak_source": "measured in this run (tpmc_measure_peaks.gather64_bytes_per_s): 64-byte records over 83 MB "
                                        "read as two 32-byte ld.global.nc of one line, two records in flight per lane, 7 x 128 "
                                        "threads per SM = k_trace_wf's access shape and residency; the one-load-in-flight figure "
                                        "of earlier rounds is peaks.gather32_bytes_per_s",
                         "fetched_view": {"achieved": fetched_bw, "peak": gpk, "unit": "GB/s", "frac": fetched_bw / gpk,
                                          "what": "wide nodes x 64 B + facets x 48 B the kernel really fetched"},
                         "alu_view": {"achieved": alg_ops, "peak": peaks["fp32_lane_ops_per_s"] / 1e12, "unit": "T lane-op/s",
                                      "frac": alg_ops / (peaks["fp32_lane_ops_per_s"] / 1e12),
                                      "peak_source": "measured in this run: FFMA lane-instructions/s at full occupancy"}})
        else:
            roof.update({"bound": "hbm", "achieved": alg_bw, "peak": hbm, "unit": "GB/s", "frac": alg_bw / hbm, "peak_source": hbm_src})
        roof["hbm_view"] = {"achieved": alg_bw, "peak": hbm, "unit": "GB/s", "frac": alg_bw / hbm, "peak_source": hbm_src}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total_max / args.steps, "higher_is_better": True,
            "scaling": "strong" if slices and world > 1 else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "particles_per_step": N, "facets": mesh.nt, "bvh_nodes": info["n_nodes"],
                       "sweep": (f"{len(cfgs)} points, point step mod {len(cfgs)} on every rank; rank r runs particles "
                                 f"[r N/{world}, (r+1) N/{world}) and the outputs (force, torque, {mesh.nt} x 3 per-facet momentum, "
                                 f"{24 * mesh.nt + 48} B) are all-reduced (NCCL, SUM) inside the timed region" if slices else
                                 f"{len(cfgs)} points, point (step*world+rank) mod {len(cfgs)}"),
                       "split": args.split, "cv_radius_factor": cfgs[0].cv_radius_factor,
                       "l2": ("inputs larger than L2: hierarchy + facets 149 MB, per-facet momentum 25 MB, ~2 GB of lists and ray "
                              "queues rewritten every wave" if flush is None else
                              "L2 flushed between steps (512 MB written); each step timed by its own event pair"),
                       "mesh_build_ms": info["build_ms"], "horizon_build_ms": info["horizon_ms"],
                       "wave_particles": min(1 << 26, max(N, 256))},
            "clocks": clocks,
            "rates": {"segments_per_s": segs_all / (ms_total_max * 1e-3), "particles_per_s": parts_all / (ms_total_max * 1e-3),
                      "hits_per_particle": hits_all / parts_all},
            "roofline": roof,
            "gpu_launches": int(launches),
        }
        if peaks:
            line["peaks"] = peaks
        if e2e:
            line["e2e"] = {"value": hits_all / e2e_s_max, "unit": UNIT,
                           "h2d_bytes_per_step": int(C.sizeof(tpmc.tpmc_params) + 16 * len(cfgs[0].m)),
                           "d2h_bytes_per_step": int(mesh.nt * 24 + 48),
                           "api": "tpmc_run + all-reduce + D2H copies" if slices and world > 1 else "tpmc_run_host"}
        if world == 1 and not args.no_cpu_baseline:
            threads = os.cpu_count() or 1
            per = max(1000, int(args.cpu_baseline_particles // threads))
            oracle_sample(cfgs, 1000, threads)
            h, dt, n = oracle_sample(cfgs, per, threads)
            h1, dt1, n1 = oracle_sample(cfgs, max(1000, int(args.cpu_baseline_particles // 40)), 1)   # one thread
            line["cpu_baseline"] = {"value": h / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
                                    "sample": f"{n} particles ({threads} slices) of the same N={N:.0e} stream, sweep point 0, {dt:.1f} s",
                                    "per_core": {"value": h1 / dt1, "unit": UNIT, "cores": 1,
                                                 "sample": f"{n1} particles, one thread, {dt1:.1f} s"}}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
