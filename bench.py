#!/usr/bin/env python
"""bench.py -- particle-bounces/s of the TPMC hot path (seed -> trace -> reflect -> accumulate ->
reduce) on synthetic config C5 of BASELINE.json: the ~1.0e6-facet procedural body, 70 % O / 30 % He,
T_inf = 900 K, |V| = 7700 m/s, N = 1e9 particles per attitude of the 64-attitude sweep.

One "step" = one tpmc_run of N particles at one attitude (the whole hot path over one batch).
  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl tpmc|reference] [--particles N]
N > 1: launched by torchrun, one rank per GPU; rank r runs attitudes r, r+N, ... (weak scaling, no
data-path collective: attitudes are independent problems); value = all ranks' bounces / max time.
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

# dram__bytes_read.sum + dram__bytes_write.sum of one steady-state k_trace_wf launch in this launch configuration
# (wave of 2^26 particles, ~1.3e7 rays per launch), from the `ncu --set full` capture summarised in
# profiles/r1_ncu_full_pipeline_v6.md
NCU_TRAFFIC_BYTES_PER_LAUNCH = 2_793_646_504
METRIC = "particle_bounces_per_s"
UNIT = "bounces/s"
WORKLOAD = "C5: ~1.0e6-facet noise-displaced geodesic body + 6 panels, O/He 70/30, 900 K, 7700 m/s"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json, copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region."""

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "200"], stdout=subprocess.PIPE, text=True)
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
    """Which attitude of the sweep a rank runs at a step: ranks take disjoint attitudes (weak scaling)."""
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


def oracle_sample(cfgs, count_per_thread, threads):
    """The oracle, as it stands, on a bounded slice of the same workload, one slice per host thread."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    m = cfgs[0].mesh()
    om = oracle.OracleMesh(m.vertices, m.indices, m.flags)
    cfg = cfgs[0]

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
    tot_hits, tot_t = 0, 0.0
    for _ in range(args.steps):
        h, dt, n = oracle_sample(cfgs, per, threads)
        tot_hits += h
        tot_t += dt
    val = tot_hits / tot_t
    sample = f"{per * threads} particles per step ({threads} slices of {per}) of the N={cfgs[0].N:.0e} stream, attitude 0"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "particles_per_step": per * threads, "facets": cfgs[0].mesh().nt},
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
    ap.add_argument("--particles", type=float, default=None, help="override N per step (default: the config's 1e9)")
    ap.add_argument("--ref-particles", type=float, default=4_000_000, help="oracle particles per reference step")
    ap.add_argument("--cpu-baseline-particles", type=float, default=80_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    cfgs = ti.config("C5")
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

    def step(k, stats=None):
        cfg = cfgs[attitude_index(k, rank, world, len(cfgs))]
        p, keep = tpmc.make_params(cfg)
        rc = L.tpmc_run(mesh._h, C.byref(p), stream.cuda_stream or None, force.data_ptr(), torque.data_ptr(),
                        facets.data_ptr(), None if stats is None else C.byref(stats), None)
        if rc != 0:
            raise SystemExit(f"tpmc_run failed: {rc} {L.tpmc_last_cuda_error().decode()}")

    # ---- warm-up (untimed)
    for k in range(args.warmup):
        step(k)
    barrier()

    # ---- timed: exactly K steps, device-resident, CUDA events on the launching stream
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for k in range(args.steps):
        step(args.warmup + k)
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_total = e0.elapsed_time(e1)

    # ---- one more pass per timed attitude with stats on: hits (the metric's numerator) and the
    #      per-kernel event times for the roofline.  Same work, same stream; not part of `value`'s clock.
    hits = segs = launches = 0
    ms_seed = ms_trace = ms_reflect = ms_finish = ms_stat = 0.0
    waves = nodes = tris = culled = tr_launches = traced = 0
    for k in range(args.steps):
        st = tpmc.tpmc_stats()
        step(args.warmup + k, st)
        hits += st.hits; segs += st.segments; launches += st.kernel_launches
        ms_seed += st.ms_seed; ms_trace += st.ms_trace; ms_stat += st.ms
        ms_reflect += st.ms_reflect; ms_finish += st.ms_finish
        waves += st.timed_waves; nodes += st.node_visits; tris += st.tri_tests; culled += st.culled
        tr_launches += st.trace_launches; traced += st.traced_rays
    barrier()

    # ---- end to end: host buffers through tpmc_run_host (params H2D, results D2H inside the region)
    e2e = None
    if not args.no_e2e:
        hF, hT = np.empty(3), np.empty(3)
        hP = torch.empty((mesh.nt, 3), dtype=torch.float64).pin_memory().numpy()
        barrier()
        t0 = time.perf_counter()
        for k in range(args.steps):
            cfg = cfgs[attitude_index(args.warmup + k, rank, world, len(cfgs))]
            p, keep = tpmc.make_params(cfg)
            rc = L.tpmc_run_host(mesh._h, C.byref(p), stream.cuda_stream or None, hF.ctypes.data, hT.ctypes.data,
                                 hP.ctypes.data, None)
            if rc != 0:
                raise SystemExit(f"tpmc_run_host failed: {rc}")
        barrier()
        e2e_s = time.perf_counter() - t0
        e2e = {"hits": hits, "s": e2e_s}

    # ---- max over ranks, totals over ranks
    (ms_total_max, e2e_s_max), (hits_all, segs_all, parts_all) = reduce_over_ranks(
        [ms_total, e2e["s"] if e2e else 0.0], [hits, segs, N * args.steps], world, dev)

    if rank == 0:
        value = hits_all / (ms_total_max * 1e-3)
        peak, peak_src = peaks()
        # dominant kernel = trace/reflect.  Algorithmic bytes per segment:
        # ceil(log2 T) nodes * 64 B + 1 triangle * 48 B + 32 B ray in + 8 B result out.
        per_seg = int(np.ceil(np.log2(mesh.nt))) * 64 + 48 + 32 + 8
        launches_trace = max(tr_launches, 1)         # k_trace_wf launches (rounds x waves), rays they processed
        bytes_per_launch = traced * per_seg / launches_trace
        avg_ms = ms_trace / launches_trace
        achieved = bytes_per_launch / (avg_ms * 1e-3) / 1e9 if avg_ms > 0 else 0.0
        # ncu shows the kernel bound by instruction issue (DRAM 1-4 %, L2 < 20 %, issue slots ~72 % busy; profiles/),
        # so the binding roofline is the fp32 lane-instruction rate: SMs x 128 lanes x SM clock under this load.
        # Algorithmic fp32 work per segment: ceil(log2 T) node visits x 2 slab tests x 18 ops + one
        # watertight facet test of 60 ops; none of it pairs into FMAs, so one op = one lane-instruction.
        ops_per_seg = int(np.ceil(np.log2(mesh.nt))) * 2 * 18 + 60
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        clk_mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965.0
        alu_peak = sms * 128 * clk_mhz * 1e6 / 1e12                      # T lane-op/s
        alu_ach = (traced * ops_per_seg / launches_trace) / (avg_ms * 1e-3) / 1e12 if avg_ms > 0 else 0.0
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "particles_per_step": N, "facets": mesh.nt, "bvh_nodes": info["n_nodes"],
                       "attitudes": "fibonacci(64)[step*world+rank]", "cv_radius_factor": cfgs[0].cv_radius_factor,
                       "l2": "inputs larger than L2: hierarchy + facets 149 MB (33 MB compact nodes, 66 MB fp32 nodes, 50 MB facets), per-facet momentum 25 MB, ~2 GB of lists and ray queues rewritten every wave",
                       "mesh_build_ms": info["build_ms"], "horizon_build_ms": info["horizon_ms"],
                       "wave_particles": 1 << 26},
            "clocks": clocks,
            "rates": {"segments_per_s": segs_all / (ms_total_max * 1e-3), "particles_per_s": parts_all / (ms_total_max * 1e-3),
                      "hits_per_particle": hits_all / parts_all},
            "roofline": {"kernel": "k_trace_wf", "bound": "alu", "achieved": alu_ach, "peak": alu_peak, "unit": "TFLOP/s",
                         "frac": alu_ach / alu_peak, "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH,
                         "peak_source": f"derived: {sms} SMs x 128 fp32 lanes x {clk_mhz:.0f} MHz sampled under this load "
                                        "(one lane-instruction = 1 op; DESIGN.md section 7)",
                         "algorithmic_ops_per_segment": ops_per_seg,
                         "hbm_view": {"achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                                      "peak_source": peak_src, "algorithmic_bytes_per_segment": per_seg},
                         "segments_per_launch": traced / launches_trace,
                         "avg_launch_ms": avg_ms, "launches_timed": int(launches_trace),
                         "share_of_step": {"k_seed": ms_seed / ms_stat if ms_stat else None,
                                           "k_trace_wf": ms_trace / ms_stat if ms_stat else None,
                                           "k_reflect": ms_reflect / ms_stat if ms_stat else None,
                                           "k_finish": ms_finish / ms_stat if ms_stat else None},
                         "nodes_per_traced_segment": nodes / max(traced, 1), "tri_tests_per_traced_segment": tris / max(traced, 1)},
            "gpu_launches": int(launches),
        }
        if e2e:
            line["e2e"] = {"value": hits_all / e2e_s_max, "unit": UNIT, "h2d_bytes_per_step": int(C.sizeof(tpmc.tpmc_params) + 16 * len(cfgs[0].m)),
                           "d2h_bytes_per_step": int(mesh.nt * 24 + 48), "api": "tpmc_run_host"}
        if world == 1 and not args.no_cpu_baseline:
            threads = os.cpu_count() or 1
            per = max(1000, int(args.cpu_baseline_particles // threads))
            oracle_sample(cfgs, 1000, threads)
            h, dt, n = oracle_sample(cfgs, per, threads)
            line["cpu_baseline"] = {"value": h / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
                                    "sample": f"{n} particles ({threads} slices of {per}) of the same N={N:.0e} stream, attitude 0, {dt:.1f} s"}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
