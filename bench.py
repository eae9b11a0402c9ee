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
  e2e        ... always the WHOLE morning (05:00-12:00), whatever --steps is; its stepping is three manta_step calls
             (to the timed window's start, the 7,200 steps of the peak hour, the rest) so that
  peak_hour  carries BASELINE.json's "wall-clock for simulated morning peak": device time of those 7,200 steps
  roofline   the kernel the headline runs in, k_persistent (one launch = the K timed steps): SURVEY 8(d) useful
             bytes of a whole step x updates / its CUDA-event duration, vs the measured HBM peak (frac); the
             per-phase figures of k_update (kernel-per-phase mode), the layout's own byte model and the committed ncu
             traffic of the persistent kernel beside it
  cpu_baseline  the oracle (oracle/manta_oracle.c, single thread) started from the library's snapshot at the first
             timed step (Oracle.set_state) and run over the same timesteps, capped at ORACLE_MAX_STEPS

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


def contract_bytes(hbar, flc):
    """SURVEY.md section 8(d), "Algorithmic bytes per vehicle-update", useful-byte column, evaluated at the measured
    mean look-ahead hbar (cells) and lane-change evaluation fraction flc: active index 4, hot state read + write
    16 + 16, route entries 16, edge attributes 16, forward occupancy scan 2 hbar (the contract counts the paper's
    2-byte cells), leader speed 4, lane-change rows flc (2 hbar + 128 + 8), new occupancy + speed + old clear 8.
    Returns (bytes of the update pass = everything but the lane-change rows, bytes of the whole step).  The pass
    kernel (k_update) does not touch the lane-change rows: those vehicles are finished in the second phase."""
    base = 4.0 + 32.0 + 16.0 + 16.0 + 2.0 * hbar + 4.0 + 8.0
    return base, base + flc * (2.0 * hbar + 136.0)


def layout_bytes(hbar, flc, lookback):
    """Bytes the method must move with THIS layout: 1-bit occupancy plane, 8-byte payload entry
    per four cells, 64-byte in-place vehicle state.  Pass: state read 64 + rewritten position word 16, own-lane
    occupancy bits hbar / 8, leader payload 8, new mark (8-byte word) 8 + own payload 8, old mark off 8.  Whole step:
    + the deferred adjacent-lane evaluations (list entry 32, target row bits ahead and behind, two payloads) and 6 B
    for the cross list, claims and the amortised re-sort."""
    upd = 64.0 + 16.0 + hbar / 8.0 + 8.0 + 8.0 + 8.0 + 8.0
    return upd, upd + flc * (32.0 + (hbar + lookback) / 8.0 + 16.0) + 6.0


def source_hash():
    """sha256 over the DEVICE sources (kernels, device functions, launch geometry constants) the library is built
    from: keys the ncu traffic captures under profiles/.  The host side (manta_api.cu) does not change what a launch
    of k_update moves with the L2 flushed before it."""
    import hashlib
    h = hashlib.sha256()
    base = os.path.join(ROOT, "paper_2007_03614_b200", "csrc")
    for name in ("manta_kernels.cuh", "manta_device.cuh"):
        with open(os.path.join(base, name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic(config, start_step, name="k_update_traffic.csv"):
    """DRAM bytes a kernel moved per vehicle-update (dram__bytes_read.sum + dram__bytes_write.sum of one
    `ncu --set full` capture), from profiles/<name> -- k_update_traffic.csv: one k_update launch, L2 flushed before
    it; k_persistent_traffic.csv: one k_persistent launch of 20 timesteps, caches left as they are -- only a line
    captured on THIS build of the sources (source_hash) and this workload window counts; None if there is none."""
    path = os.path.join(ROOT, "profiles", name)
    if not os.path.exists(path):
        return None
    sh = source_hash()
    best = None
    with open(path) as f:
        for line in f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7 or c[0].startswith("#") or c[0] == "source_hash":
                continue
            if c[0] == sh and int(c[1]) == config and int(c[2]) == start_step:
                best = {"bytes_per_update": (float(c[4]) + float(c[5])) / float(c[3]), "capture": c[6], "source_hash": sh}
    return best


def host_cpu():
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return model, os.cpu_count() or 1


ORACLE_SAMPLE_TRIPS, ORACLE_SAMPLE_STEPS = 12000, 1800


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


ORACLE_MAX_STEPS = 100      # ~229 k active vehicles x 100 steps = 2.3e7 updates: ~20 s of one host core


def oracle_at_load(net, trips, params, t, snap, n_steps):
    """The oracle at the load that is timed: started from the LIBRARY's snapshot at step t (manta_readback ->
    Oracle.set_state: state transfer, no arithmetic of the method), run over n_steps timesteps on one host core.
    Returns (vehicle-updates, wall seconds of the steps, set-up seconds)."""
    from oracle import manta_oracle
    t0 = time.perf_counter()
    o = manta_oracle.Oracle(net, params, trips)
    o.set_state(t, snap, snap["edge_entries"])
    t_setup = time.perf_counter() - t0
    u0 = o.summary()["vehicle_updates"]
    t0 = time.perf_counter()
    o.step(n_steps)
    wall = time.perf_counter() - t0
    upd = o.summary()["vehicle_updates"] - u0
    o.close()
    return upd, wall, t_setup


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same config / metric / unit.  Its timed sample is
    the one the cpu_baseline leg of the default run uses (ORACLE_SAMPLE_TRIPS trips departing from the start of the
    timed window, ORACLE_SAMPLE_STEPS timesteps), so the two oracle figures agree; it does not depend on --steps:
    20 timesteps of a 12,000-trip sample would be a nearly empty network."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    net, trips, params, _ = make_workload(args.scale, config=args.config)
    K, W = args.steps, args.warmup
    from oracle import manta_oracle
    manta_oracle.build()
    if W:   # warm-up: page the library and the workload in
        oracle_sample(net, trips, params, args.start_step, 2000, min(200, 10 * W))
    upd, wall, n_tr, _ = oracle_sample(net, trips, params, args.start_step, ORACLE_SAMPLE_TRIPS, ORACLE_SAMPLE_STEPS)
    val = upd / wall
    model, cores = host_cpu()
    sample = ("first %d trips departing from step %d of configs[%d] (scale %g), %d timesteps from their first "
              "departure (%.2e updates in %.1f s); the sample does not scale with --steps"
              % (n_tr, args.start_step, args.config, args.scale, ORACLE_SAMPLE_STEPS, upd, wall))
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
           "warmup": W, "ms_per_step": wall / ORACLE_SAMPLE_STEPS * 1e3, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": "%s, scale %g" % (CONFIGS[args.config][0], args.scale),
                      "sample": sample, "l2": "n/a (CPU)"},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                            "cpu_model": model, "host_cores": cores},
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
    want_cpu = not args.no_cpu and rank == 0 and world == 1
    snap0 = sim.readback() if want_cpu else None          # state at the first timed step: where the oracle starts too
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
    sim.step_timed(3)                                     # the kernel-per-phase variants load on first use: not timed
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
    # Algorithmic bytes per vehicle-update.  Contract figure: SURVEY.md section 8(d)'s useful-byte table at the
    # measured hbar / f_lc (roofline.frac).  Beside it the bytes this layout must move (frac_layout), and the DRAM
    # bytes ncu saw k_update move on this build, if a capture of this build is committed (frac_traffic).
    c_update, c_step = contract_bytes(hbar, flc)
    l_update, l_step = layout_bytes(hbar, flc, params.get("lookback_cells", 64))
    peak, peak_src = measured_peak()
    upd_per_launch = d["vehicle_updates"] / Kp
    t_update = ph[1] / Kp * 1e-3
    achieved = c_update * upd_per_launch / t_update / 1e9
    tr = ncu_traffic(args.config, args.start_step)
    trp = ncu_traffic(args.config, args.start_step, "k_persistent_traffic.csv")
    # The dominant kernel of the headline is k_persistent: ONE launch runs the K timed steps (all phases of every
    # step), so "bytes per launch / launch duration" = step bytes x updates of the timed region / its device time.
    persist = not (args.flags & 2)
    n_launch = max(1, launches)
    step_achieved = c_step * (upd / (ms * 1e-3)) / 1e9
    roofline = {"bound": "hbm", "kernel": "k_persistent" if persist else "k_admit + k_update + k_second",
                "achieved": step_achieved, "peak": peak, "unit": "GB/s", "frac": step_achieved / peak,
                "bytes_model": "SURVEY.md 8(d) useful bytes of a WHOLE step at the measured hbar, f_lc.  Note: 2 hbar of "
                               "them (%.0f of %.0f B) are the survey's 2-byte cells over the look-ahead; this layout "
                               "reads 1 bit per cell (hbar / 8 B), so frac says how fast the survey's layout would "
                               "have had to move data to keep up, and frac_layout / frac_traffic say what this one moves"
                               % (2.0 * hbar, c_step),
                "bytes_per_update": c_step, "bytes_per_launch": c_step * upd / n_launch,
                "avg_launch_us": ms * 1e3 / n_launch, "launches": launches, "updates_per_launch": upd / n_launch,
                "frac_layout": l_step * (upd / (ms * 1e-3)) / 1e9 / peak, "bytes_per_update_layout": l_step,
                "traffic": trp["bytes_per_update"] * upd / n_launch if trp else None,
                "frac_traffic": trp["bytes_per_update"] * (upd / (ms * 1e-3)) / 1e9 / peak if trp else None,
                "traffic_source": ("profiles/k_persistent_traffic.csv, capture %s on this build (sources %s): %.0f B of DRAM "
                                   "traffic per update (one 20-step launch at this window, caches left warm); scaled to "
                                   "this run's updates per launch" % (trp["capture"], trp["source_hash"], trp["bytes_per_update"]))
                                  if trp else "no ncu capture of k_persistent on this build (sources %s) at this window is committed" % source_hash(),
                "target_frac": 0.5, "peak_source": peak_src, "hbar_cells": hbar, "f_lc": flc,
                # the update pass alone, timed in kernel-per-phase mode (manta_step_timed) -- a mode the headline does
                # not run in (its three launches per step cost 1.5 x the persistent kernel's step)
                "k_update": {"achieved": achieved, "frac": achieved / peak, "bytes_per_update": c_update,
                             "frac_layout": l_update * upd_per_launch / t_update / 1e9 / peak,
                             "bytes_per_update_layout": l_update,
                             "traffic": tr["bytes_per_update"] * upd_per_launch if tr else None,
                             "frac_traffic": tr["bytes_per_update"] * upd_per_launch / t_update / 1e9 / peak if tr else None,
                             "traffic_source": ("profiles/k_update_traffic.csv, capture %s (sources %s): %.0f B per update, L2 "
                                                "flushed before the launch" % (tr["capture"], tr["source_hash"], tr["bytes_per_update"]))
                                               if tr else "no ncu capture of k_update on this build is committed",
                             "updates_per_launch": upd_per_launch, "avg_launch_us": t_update * 1e6,
                             "phase_ms_per_step": {"admit": ph[0] / Kp, "update": ph[1] / Kp, "second": ph[2] / Kp}}}

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
        # the whole simulated run, whatever --steps is; inside it the peak hour (7,200 steps from --start-step) between
        # two CUDA events and two summary readbacks (their cost stays inside the end-to-end wall time)
        n_e2e = max(n_total, args.start_step + 7200)
        pk = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        barrier()
        t0 = time.perf_counter()
        sim = binding.Sim(net, params, None, device=local, stream=stream)   # network upload = initialisation
        t1 = time.perf_counter()
        sim.load_trips(trips)                                                 # H2D: routes, departures
        t2 = time.perf_counter()
        sim.step(args.start_step)
        p0 = sim.readback(state=False, edge_entries=False, trips=False)["summary"]
        tp0 = time.perf_counter()
        pk[0].record(stream)
        sim.step_async(7200)
        pk[1].record(stream)
        sim.sync()
        tp1 = time.perf_counter()
        p1 = sim.readback(state=False, edge_entries=False, trips=False)["summary"]
        sim.step(n_e2e - args.start_step - 7200)
        t3 = time.perf_counter()
        res = sim.readback()                                                  # D2H: state, per-edge counts, trip results
        t4 = time.perf_counter()
        sim.close()
        wall = t4 - t1
        pk_ms = pk[0].elapsed_time(pk[1])
        pk_upd = p1["vehicle_updates"] - p0["vehicle_updates"]
        # the step bytes of the HOUR: SURVEY 8(d) at the hour's own mean look-ahead and lane-change fraction (denser
        # traffic finds its leaders sooner: fewer contract bytes per update than in the first seconds of the hour)
        pk_hbar = (p1["cells_examined"] - p0["cells_examined"]) / max(1, pk_upd)
        pk_flc = (p1["lc_evals"] - p0["lc_evals"]) / max(1, pk_upd)
        pk_c_step = contract_bytes(pk_hbar, pk_flc)[1]
        pk_l_step = layout_bytes(pk_hbar, pk_flc, params.get("lookback_cells", 64))[1]
        out["peak_hour"] = {"start_step": args.start_step, "steps": 7200, "simulated_s": 3600.0,
                            "device_s": pk_ms * 1e-3, "wall_s": tp1 - tp0, "us_per_step": pk_ms * 1e3 / 7200,
                            "vehicle_updates": pk_upd, "value": pk_upd / (pk_ms * 1e-3), "unit": UNIT,
                            "sim_hours_per_wall_s": 1.0 / (pk_ms * 1e-3),
                            "active_vehicles": {"start": p0["n_active"], "end": p1["n_active"]},
                            "hbar_cells": pk_hbar, "f_lc": pk_flc, "bytes_per_update": pk_c_step,
                            "roofline_frac": pk_c_step * pk_upd / (pk_ms * 1e-3) / 1e9 / peak,
                            "roofline_frac_layout": pk_l_step * pk_upd / (pk_ms * 1e-3) / 1e9 / peak,
                            "note": "device time (CUDA events on the simulation's stream) of manta_step(7200) inside the "
                                    "end-to-end run; roofline_frac = SURVEY 8(d) step bytes at THIS hour's hbar and f_lc "
                                    "x updates / device time / peak (the formula of roofline.frac)"}
        h2d = trips["route_ptr"].nbytes + trips["route_edges"].nbytes + trips["depart_time_s"].nbytes
        d2h = n_trips * (1 + 4 + 1 + 1 + 4 + 4 + 4 + 8) + net["n_edges"] * 4
        e_upd = res["summary"]["vehicle_updates"]
        out["e2e"] = {"value": e_upd * world / wall, "unit": UNIT, "h2d_bytes_per_step": h2d / n_e2e,
                      "d2h_bytes_per_step": d2h / n_e2e, "timesteps": n_e2e, "wall_s": wall,
                      "load_trips_s": t2 - t1, "step_s": t3 - t2, "readback_s": t4 - t3, "create_s": t1 - t0,
                      "done_trips": res["summary"]["n_done"], "vehicle_updates": e_upd,
                      "sim_hours_per_wall_s": n_e2e * 0.5 / 3600.0 / (t3 - t2),
                      "what": "manta_load_trips + manta_step over the whole simulated run (three calls, two summary "
                              "readbacks between them) + manta_readback, host buffers, wall clock"}
    # ---- the oracle beside it (rank 0, N = 1 only) -------------------------------------------------------
    if want_cpu:
        from oracle import manta_oracle
        manta_oracle.build()
        k_s = min(K, ORACLE_MAX_STEPS)
        c_upd, c_wall, c_setup = oracle_at_load(net, trips, params, args.start_step + W, snap0, k_s)
        model, cores = host_cpu()
        out["cpu_baseline"] = {"value": c_upd / c_wall, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "cpu_model": model, "host_cores": cores, "same_load": True,
                               "sample": "the same workload at the same load: all %d trips, started from the library's "
                                         "snapshot at timestep %d (%d active vehicles), the first %d of the %d timed "
                                         "timesteps (%.2e updates in %.1f s; oracle set-up %.1f s not counted)"
                                         % (n_trips, args.start_step + W, s0["n_active"], k_s, K, c_upd, c_wall, c_setup)}
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
