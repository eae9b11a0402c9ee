#!/usr/bin/env python
"""bench.py -- vehicle-updates/s of the MANTA hot path on B200 (BASELINE.json metric), one JSON line.

Workload: BASELINE.json configs[2], the Bay-Area-shaped synthetic morning: ~224 k nodes,
~556 k directed edges, 3.2 M routed trips, dt = 0.5 s.  A bench "step" is ONE simulation timestep = one pass of
the whole hot path (admission, look-ahead, IDM, lane change, integration, edge transfer, atlas write, compaction)
over all active vehicles.  The simulation is first advanced (untimed: initialisation) to --start-step (default
18,000 = 07:30, the start of the peak hour), then W warm-up steps, then exactly K timed steps (default 7,200 =
07:30-08:30).  Inputs are resident in HBM when the timed region starts; the working set (0.7 GB of atlas planes,
3-6 GB of route records, 50-100 MB of vehicle state) exceeds the 126 MB L2, so no explicit L2 flush is needed.

  value      whole-job vehicle-updates/s (sum over ranks / max-over-ranks device time; ranks run independent
             replicas -- "replicas only")
  e2e        same metric through the C ABI with HOST buffers: manta_load_trips (H2D of routes and departures) +
             manta_step from 05:00 to the end of the timed window + manta_readback (D2H), wall clock
  roofline   update-phase kernel: algorithmic bytes per launch / its CUDA-event duration, vs measured HBM peak
  cpu_baseline  the oracle (oracle/manta_oracle.c, single thread) on a bounded sample of the same workload

--impl reference times the oracle itself (there is no other reference implementation: the paper ships no code).
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

METRIC = "vehicle_updates_per_s"
UNIT = "vehicle-updates/s"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


CONFIGS = {2: ("configs[2] Bay-Area-shaped synthetic morning", 50400),
           3: ("configs[3] congestion stress (lane-reduced configs[2] network, 2 x demand in 06:00-09:00)", 43200),
           4: ("configs[4] 2 x 2 tiled configs[2] network, 4 x demand", 50400)}


def make_workload(scale, n_threads=None, cache=True, config=2):
    from paper_2007_03614_b200 import workloads as wl
    tag = "/tmp/manta_cfg%d_%g_v3.npz" % (config, scale)
    if cache and os.path.exists(tag):
        try:
            z = np.load(tag, allow_pickle=False)
            net = {k[4:]: z[k] for k in z.files if k.startswith("net_")}
            net["n_nodes"], net["n_edges"] = int(net["n_nodes"]), int(net["n_edges"])
            trips = {k[5:]: z[k] for k in z.files if k.startswith("trip_")}
            trips["init_pos_m"] = trips["init_speed"] = None
            return net, trips, dict(lookahead_cells=256), CONFIGS[config][1]
        except Exception:
            pass
    gen = {2: wl.config2, 3: wl.config3, 4: wl.config4}[config]
    net, trips, params, n_steps = gen(scale=scale, n_threads=n_threads)
    if cache:
        try:
            keep = ("n_nodes", "n_edges", "row_ptr", "head", "length_m", "lanes", "speed_limit", "node_ctrl")
            np.savez(tag, **{"net_" + k: np.asarray(net[k]) for k in keep},
                     **{"trip_" + k: trips[k] for k in ("route_ptr", "route_edges", "depart_time_s")})
        except Exception:
            pass
    net = {k: net[k] for k in ("n_nodes", "n_edges", "row_ptr", "head", "length_m", "lanes", "speed_limit", "node_ctrl")}
    return net, trips, params, n_steps


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu):
        self.rows, self.proc, self.gpu = [], None, gpu

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip().split(", "))

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if val.strip().lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def algorithmic_bytes(hbar, flc, lookback):
    """Algorithmic bytes per vehicle-update, 1-bit occupancy plane + 8-byte payload plane +
    64-byte in-place vehicle state.  Update phase: state read 64 (position / speed, edge geometry, cached rows and
    lengths of the next four route edges) + rewritten position word 16, own-lane occupancy bits hbar / 8, leader
    payload 8, new mark (8-byte word) 8 + own payload 8, toggling the old mark off 8; a deferred adjacent-lane
    evaluation adds its list entry (16 written + 16 read), the target row's bits ahead and behind and two payloads.
    The whole step adds the cross-list entry and claim of the ~2 % of vehicles at an edge end and the amortised
    re-sort (128 B per vehicle every MANTA_SORT_EVERY = 64 steps), folded in as 6 B."""
    upd = 64.0 + 16.0 + hbar / 8.0 + 8.0 + 8.0 + 8.0 + 8.0 + flc * (32.0 + (hbar + lookback) / 8.0 + 16.0)
    return upd, upd + 6.0


# DRAM bytes k_update actually moved, from the committed ncu --set full capture (profiles/r01e_two_stage.md):
# dram__bytes_read.sum + dram__bytes_write.sum = 72.7 MB + 6.7 MB for a launch of 383,948 vehicle-updates with the
# L2 flushed before the launch (ncu's default cache control), i.e. 207 B per update (live, application replay:
# 135-165 B).  bench.py reports it scaled to the updates per launch of its own timed window.
NCU_TRAFFIC_BYTES_PER_UPDATE = (72.678656e6 + 6.671360e6) / 383948.0


def oracle_sample(net, trips, params, start_step, n_sample_trips, n_steps, dt=0.5):
    """Bounded sample of the same workload for the CPU oracle: the first n_sample_trips trips departing at or
    after start_step, their departures shifted so the earliest leaves at t = 0; run n_steps timesteps."""
    from oracle import manta_oracle
    dep = trips["depart_time_s"]
    rp = trips["route_ptr"].astype(np.int64)
    cand = np.nonzero(dep >= start_step * dt)[0]
    cand = cand[np.argsort(dep[cand], kind="stable")][:n_sample_trips]
    cand = np.sort(cand)
    lens = rp[cand + 1] - rp[cand]
    new_rp = np.zeros(len(cand) + 1, np.uint64)
    new_rp[1:] = np.cumsum(lens)
    idx = np.concatenate([np.arange(rp[i], rp[i + 1]) for i in cand]) if len(cand) else np.zeros(0, np.int64)
    sub = dict(route_ptr=new_rp, route_edges=trips["route_edges"][idx], depart_time_s=dep[cand] - dep[cand].min(),
               init_pos_m=None, init_speed=None)
    t0 = time.perf_counter()
    o = manta_oracle.Oracle(net, params, sub)
    t_setup = time.perf_counter() - t0
    t0 = time.perf_counter()
    o.step(n_steps)
    wall = time.perf_counter() - t0
    s = o.summary()
    o.close()
    return s["vehicle_updates"], wall, len(cand), t_setup


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same config / metric / unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    net, trips, params, _ = make_workload(args.scale, config=args.config)
    K, W = args.steps, args.warmup
    # sample sized so that W + K oracle steps end within ~2 minutes (about 1.5 us per update on one core)
    n_sample = int(min(200000, max(2000, 100.0 / ((K + W) * 1.5e-6))))
    from oracle import manta_oracle
    manta_oracle.build()
    upd_w, wall_w, n_tr, _ = oracle_sample(net, trips, params, args.start_step, n_sample, W + K)
    # time K steps = total minus a separately timed W-step warm-up run of the same sample
    upd_0, wall_0, _, _ = oracle_sample(net, trips, params, args.start_step, n_sample, W) if W else (0, 0.0, 0, 0)
    upd, wall = upd_w - upd_0, max(wall_w - wall_0, 1e-9)
    val = upd / wall
    sample = ("first %d trips departing from step %d of configs[%d] (scale %g), run %d timesteps from their first "
              "departure" % (n_tr, args.start_step, args.config, args.scale, K))
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
           "warmup": W, "ms_per_step": wall / K * 1e3, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": "%s, scale %g" % (CONFIGS[args.config][0], args.scale),
                      "sample": sample, "l2": "n/a (CPU)"},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def aggregate(ms, updates, world, device="cpu"):
    """Whole-job figures of N independent replicas: MAX over ranks of the device time of the
    timed region, SUM over ranks of the vehicle-updates processed in it; value = SUM / MAX.  These two reductions
    (and the barriers around the timed region) are the only collectives of a multi-GPU run."""
    import torch
    import torch.distributed as dist
    t_ms = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    t_upd = torch.tensor([float(updates)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
        dist.all_reduce(t_upd, op=dist.ReduceOp.SUM)
    ms_max, upd_all = float(t_ms.item()), float(t_upd.item())
    return ms_max, upd_all, upd_all / (ms_max * 1e-3)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=7200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scale", type=float, default=1.0, help="configs[2] size factor (1.0 = the named workload)")
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4],
                    help="BASELINE.json config: 2 = the workload the metric is quoted on (default); 3, 4 = the larger cases")
    ap.add_argument("--start-step", type=int, default=None,
                    help="timestep at which the timed window starts (default: 07:30 = step 18000; configs[3]: 07:00 = step 7200)")
    ap.add_argument("--flags", type=int, default=0, help="manta_params.flags (A/B switches)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.start_step is None:
        args.start_step = 7200 if args.config == 3 else 18000
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2007_03614_b200 import binding
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.load_library()
    K, W = args.steps, max(args.warmup, 3)
    t0 = time.time()
    net, trips, params, n_total = make_workload(args.scale, config=args.config)
    params = dict(params, flags=args.flags)
    n_trips = len(trips["depart_time_s"])
    log("[bench] workload ready in %.1f s: %d nodes %d edges %d trips %d route entries" % (
        time.time() - t0, net["n_nodes"], net["n_edges"], n_trips, len(trips["route_edges"])))

    stream = torch.cuda.Stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident measurement -------------------------------------------------------------------
    sim = binding.Sim(net, params, trips, device=local, stream=stream)
    dev_bytes = sim.device_bytes
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    ev[0].record(stream)
    sim.set_multi_kernel(False)                           # the untimed fast-forward always runs in the persistent kernel
    sim.step_async(args.start_step)                       # initialisation: advance to the peak (untimed region)
    sim.set_multi_kernel(bool(args.flags & 2))
    ev[1].record(stream)
    sim.step(W)                                           # warm-up steps
    s0 = sim.readback(state=False, edge_entries=False, trips=False)["summary"]
    launches0 = sim.launch_count
    clocks = ClockSampler(local)
    clocks.start()
    barrier()
    ev[2].record(stream)
    sim.step_async(K)
    ev[3].record(stream)
    barrier()
    clk = clocks.stop()
    ms = ev[2].elapsed_time(ev[3])
    ms_pre = ev[0].elapsed_time(ev[1])
    s1 = sim.readback(state=False, edge_entries=False, trips=False)["summary"]
    launches = sim.launch_count - launches0
    upd = s1["vehicle_updates"] - s0["vehicle_updates"]
    ms_max, upd_all, value = aggregate(ms, upd, world, "cuda")
    sim.close()

    # ---- roofline of the update-phase kernel: per-phase CUDA events on the launching stream ---------------
    sim = binding.Sim(net, params, trips, device=local, stream=stream)
    sim.set_multi_kernel(False)
    sim.step(args.start_step + W)
    # up to 1,200 of the K timesteps, in 12 slices spread evenly over the timed window (the active-vehicle count
    # changes several-fold across it); the steps between the slices run untimed in the persistent kernel
    Kp = min(K, 1200)
    n_sl = 12 if K >= 2400 else 1
    per, gap = Kp // n_sl, (K - Kp) // n_sl
    Kp = per * n_sl
    ph, d = [0.0, 0.0, 0.0], None
    for _ in range(n_sl):
        r0 = sim.readback(state=False, edge_entries=False, trips=False)["summary"]
        p_sl = sim.step_timed(per)
        r1 = sim.readback(state=False, edge_entries=False, trips=False)["summary"]
        ph = [a + b for a, b in zip(ph, p_sl)]
        d = {k: (d[k] if d else 0) + r1[k] - r0[k] for k in r0}
        if gap:
            sim.step(gap)
    sim.close()
    hbar = d["cells_examined"] / max(1, d["vehicle_updates"])
    flc = d["lc_evals"] / max(1, d["vehicle_updates"])
    # algorithmic bytes per vehicle-update: whole step, and the update phase alone
    bytes_update, bytes_step = algorithmic_bytes(hbar, flc, params.get("lookback_cells", 64))
    peak, peak_src = measured_peak()
    upd_per_launch = d["vehicle_updates"] / Kp
    t_update = ph[1] / Kp * 1e-3
    achieved = bytes_update * upd_per_launch / t_update / 1e9
    roofline = {"bound": "hbm", "kernel": "k_update", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES_PER_UPDATE * upd_per_launch,
                "traffic_source": "ncu --set full (profiles/r01e_two_stage.md): %.0f B per update, L2 flushed; "
                                  "scaled to this run's updates per launch" % NCU_TRAFFIC_BYTES_PER_UPDATE,
                "peak_source": peak_src,
                "bytes_per_update": bytes_update, "updates_per_launch": upd_per_launch,
                "avg_launch_us": t_update * 1e6, "hbar_cells": hbar, "f_lc": flc,
                "phase_ms_per_step": {"admit": ph[0] / Kp, "update": ph[1] / Kp, "second": ph[2] / Kp},
                "step_bytes_per_update": bytes_step,
                "step_frac": bytes_step * value / world / 1e9 / peak}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
           "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": "%s, scale %g: %d nodes, %d directed edges, %d trips, dt 0.5 s" % (
                          CONFIGS[args.config][0], args.scale, net["n_nodes"], net["n_edges"], n_trips),
                      "timed_window": "timesteps %d..%d (%d steps of 0.5 s)" % (args.start_step + W, args.start_step + W + K, K),
                      "parallelism": "replicas x%d" % world, "flags": args.flags,
                      "l2": "inputs larger than L2 (%.1f GB device-resident), no flush" % (dev_bytes / 1e9)},
           "clocks": clk, "gpu_launches": launches, "roofline": roofline,
           "active_vehicles": {"start": s0["n_active"], "end": s1["n_active"]},
           "sim_hours_per_wall_s": K * 0.5 / 3600.0 / (ms_max * 1e-3),
           "fast_forward_ms": ms_pre}

    # ---- end to end through the C ABI with host buffers -------------------------------------------------
    if not args.no_e2e:
        n_e2e = n_total if (args.start_step + W + K) <= n_total and K >= 7200 else args.start_step + W + K
        barrier()
        t0 = time.perf_counter()
        sim = binding.Sim(net, params, None, device=local, stream=stream)   # network upload = initialisation
        t1 = time.perf_counter()
        sim.load_trips(trips)                                                 # H2D: routes, departures
        t2 = time.perf_counter()
        sim.step(n_e2e)
        t3 = time.perf_counter()
        res = sim.readback()                                                  # D2H: state, per-edge counts, trip results
        t4 = time.perf_counter()
        sim.close()
        wall = t4 - t1
        h2d = trips["route_ptr"].nbytes + trips["route_edges"].nbytes + trips["depart_time_s"].nbytes
        d2h = n_trips * (1 + 4 + 1 + 1 + 4 + 4 + 4 + 8) + net["n_edges"] * 4
        e_upd = res["summary"]["vehicle_updates"]
        out["e2e"] = {"value": e_upd * world / wall, "unit": UNIT, "h2d_bytes_per_step": h2d / n_e2e,
                      "d2h_bytes_per_step": d2h / n_e2e, "timesteps": n_e2e, "wall_s": wall,
                      "load_trips_s": t2 - t1, "step_s": t3 - t2, "readback_s": t4 - t3, "create_s": t1 - t0,
                      "done_trips": res["summary"]["n_done"], "vehicle_updates": e_upd,
                      "sim_hours_per_wall_s": n_e2e * 0.5 / 3600.0 / (t3 - t2)}
    # ---- the oracle beside it (rank 0, N = 1 only) -------------------------------------------------------
    if not args.no_cpu and rank == 0 and world == 1:
        from oracle import manta_oracle
        manta_oracle.build()
        n_s, k_s = 12000, 1800
        c_upd, c_wall, n_tr, _ = oracle_sample(net, trips, params, args.start_step, n_s, k_s)
        out["cpu_baseline"] = {"value": c_upd / c_wall, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "sample": "first %d trips departing from step %d of the same workload, %d timesteps "
                                         "(%.2e updates in %.1f s)" % (n_tr, args.start_step, k_s, c_upd, c_wall)}
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
