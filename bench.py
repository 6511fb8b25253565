#!/usr/bin/env python
"""bench.py -- throughput of the geometric-network hot path on B200 (contract in the task prompt).

  python bench.py [--gpus N] [--steps K] [--warmup W]            # our arm (CUDA library via the C ABI)
  python bench.py --impl reference [--steps K] [--warmup W]      # the CPU oracle on the host cores

Workload (config.workload): BASELINE.json configs[3] -- the 1M-vertex / ~200M-edge 3D random geometric
graph the real-time-factor target is quoted on.  One bench "step" is
`sim_steps_per_step` (default 100 = 10 ms simulated) consecutive passes of the whole hot path
(a1 ring read-and-clear + drive, a2 vertex update, a3 detect/compact/raster, a4 event delivery;
a5 observation when the config has it), so the default K=100 is the config's full 10,000-step run.
`value` = simulated vertex-steps per second with every input resident in HBM.  L2 is not flushed
between steps: the working set (512 MB ring + 1.8 GB edges + 16 MB state) is >> the 126 MB L2.

One JSON line on stdout (rank 0).  Everything else goes to stderr.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC, UNIT = "vertex-steps/s", "vertex-steps/s"
UPDATE_BYTES_PER_VERTEX = 35.125       # V,W,r r+w 24, ring slot r+clear 8, refr 2, class 1, raster bit 1/8
UPDATE_BYTES_PER_VERTEX_OBS = 12.0     # + c r+w 8, frame accumulator amortised / trace row 4 per frame (counted per step as 4)
HH_BYTES_PER_VERTEX = 51.125           # Hodgkin-Huxley class: V, n, r, m, h r+w 40, ring slot r+clear 8, refr 2, class 1, raster bit 1/8
HH_FP32_PER_VERTEX = 141.0             # fp32 operations of the contract per Hodgkin-Huxley vertex-step (6 exp32 x 14,
                                       # rate arguments and shapes 25, currents 16, gates 12, V, PSC, input 4; a division counts 1)
FP32_LANES_PER_SM, SM_COUNT, SM_HZ = 128, 148, 1.965e9   # B200_PROFILING.md: 148 SMs, 1965 MHz; 4 x 32 fp32 lanes per SM
IZH_OPS_PER_VERTEX = 46.0              # lane-instructions of the contract per Izhikevich vertex-step, counted from the kernel source:
                                       # vertex_step 12 fp32 (W line 3, V line 6, PSC 1, calcium 2) + detection / hold / raster 2 +
                                       # a quarter of a Philox4x32-10 block (10 rounds x 2 mul.lo, 2 mul.hi, 4 xor + 2 key adds = 102
                                       # + counter set-up ~26 = ~128 per block of 4 vertices: 32)
EVENT_BYTES = 17.0                     # edge record 9 (target 4, weight 4, delay 1) + ring word read-modify-write 8
SOURCE_BYTES = 12.0                    # two row offsets + active-list entry per fired source
SECTOR_EVENT_BYTES = 73.0              # 9 + one 32 B sector fetched + one written back (ring >> L2)


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception as e:   # no nvidia-smi: report that, do not invent clocks
            log("clock sampler unavailable:", e)
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                smax.append(float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm)}


def measured_traffic():
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of each kernel from the committed `ncu --set full` captures:
    profiles/traffic.csv, whose first line names the capture and its step range.  {kernel: (per launch, per event or None)}."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        lines = [l.strip() for l in open(path).read().splitlines() if l.strip()]
        src = lines[0].lstrip("# ") if lines[0].startswith("#") else "profiles/traffic.csv"
        rows = [l.split(",") for l in lines if not l.startswith("#")][1:]
        return {r[0]: (float(r[1]), float(r[2]) if len(r) > 2 and r[2] else None) for r in rows}, src
    except Exception:
        return {}, None


def rank_seed(config, rank):
    """Replicas only: rank r steps its own independent network of the same recipe."""
    from gn_inputs import MASTER_SEED
    return MASTER_SEED + config + 1000 * rank


def reduce_over_ranks(dist, device, ms, spikes, events):
    """Whole-job figures: time = MAX over ranks, spikes / events = SUM over ranks (no data-path collective)."""
    import torch
    if dist is None:
        return ms, spikes, events
    tms = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(tms, op=dist.ReduceOp.MAX)
    tot = torch.tensor([spikes, events], device=device, dtype=torch.float64)
    dist.all_reduce(tot)
    return float(tms.item()), float(tot[0]), float(tot[1])


def workload_name(net_in, cfg, args):
    return (f"BASELINE configs[{args.config - 1}] {cfg['name']}: N={net_in.n_vertices}, E={net_in.n_edges}, "
            f"D={cfg['ring_slots']}, dt={cfg['dt_ms']} ms")


# ---------------------------------------------------------------------------------------------------
def run_reference(args):
    """The oracle, as it stands, on the host cores: same config / metric / unit; each bench step is a
    bounded sample (a few simulated steps of the full-size network) so the run ends in minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from gn_inputs import make_config
    from oracle import Oracle
    cores = len(os.sched_getaffinity(0))
    t0 = time.time()
    net_in, cfg = make_config(args.config, n=args.n)
    cfg = dict(cfg, obs_stride=0 if args.config == 4 else cfg["obs_stride"])
    if args.model == "hh":
        from gn_inputs import as_hodgkin_huxley
        cfg = as_hodgkin_huxley(cfg)
    if args.psc_alpha:
        cfg = dict(cfg, classes=[dict(c, psc_alpha=1.0) for c in cfg["classes"]], name=cfg["name"] + "+alpha_psc")
    log(f"[reference] inputs in {time.time() - t0:.1f} s: N={net_in.n_vertices} E={net_in.n_edges}")
    o = Oracle(net_in, cfg, "fp32", threads=cores)
    t0 = time.time()
    o.step(1)
    t1 = max(time.time() - t0, 1e-6)
    budget = 90.0
    s_ref = int(max(1, min(args.sim_steps, budget / (args.steps + args.warmup) / t1)))
    for _ in range(args.warmup):
        o.step(s_ref)
    c0 = o.counters()
    t0 = time.time()
    for _ in range(args.steps):
        o.step(s_ref)
    dt = time.time() - t0
    c1 = o.counters()
    n = net_in.n_vertices
    value = n * s_ref * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(net_in, cfg, args), "sim_steps_per_step": s_ref,
                   "note": "oracle/gn_oracle.c fp32-faithful mode, OpenMP over vertices / fired sources, from rest"},
        "events_per_s": (c1["delivered"] - c0["delivered"]) / dt,
        "real_time_factor": s_ref * args.steps * cfg["dt_ms"] * 1e-3 / dt,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{(args.steps + args.warmup) * s_ref + 1} simulated steps of the full network from rest; "
                                   f"timed {args.steps * s_ref}"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
def cpu_baseline(net_in, cfg, budget_s=20.0):
    from oracle import Oracle
    cores = len(os.sched_getaffinity(0))
    o = Oracle(net_in, cfg, "fp32", threads=cores)
    t0 = time.time()
    o.step(2)
    per = max((time.time() - t0) / 2, 1e-6)
    n_steps = int(max(5, min(2000, budget_s / per)))
    c0 = o.counters()
    t0 = time.time()
    o.step(n_steps)
    dt = time.time() - t0
    c1 = o.counters()
    # one thread as well (the paper's own CPU baseline was a single thread): a shorter sample
    o1 = Oracle(net_in, cfg, "fp32", threads=1)
    t1 = time.time()
    o1.step(2)
    per1 = max((time.time() - t1) / 2, 1e-6)
    n1 = int(max(3, min(500, 6.0 / per1)))
    t1 = time.time()
    o1.step(n1)
    dt1 = time.time() - t1
    one = {"value": net_in.n_vertices * n1 / dt1, "unit": UNIT, "cores": 1,
           "sample": f"{n1} simulated steps of the same network from rest, one thread"}
    return {"value": net_in.n_vertices * n_steps / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "one_thread": one,
            "sample": f"{n_steps} simulated steps of the same full-size network from rest (fp32-faithful mode, OpenMP), "
                      f"{c1['delivered'] - c0['delivered']} events delivered",
            "events_per_s": (c1["delivered"] - c0["delivered"]) / dt,
            "real_time_factor": n_steps * cfg["dt_ms"] * 1e-3 / dt}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--n", type=int, default=None, help="override the vertex count (debugging only)")
    ap.add_argument("--sim-steps", type=int, default=100, help="simulated steps per bench step")
    ap.add_argument("--delivery", default="auto", choices=["auto", "ring", "queue"], help="gn_config.delivery_mode")
    ap.add_argument("--queue-group", type=int, default=0, help="gn_config.queue_group (0 = library default)")
    ap.add_argument("--psc-alpha", action="store_true", help="every class uses the alpha-function PSC (DESIGN.md f-1) "
                                                              "instead of the config's exponential one: a different workload")
    ap.add_argument("--model", default="izhikevich", choices=["izhikevich", "hh"],
                    help="hh: every class a Hodgkin-Huxley vertex at dt = 0.03 ms (the paper's second benchmarked model, "
                         "PAPER.md:382): a different workload, reported with an fp32-ALU roofline beside the HBM one")
    ap.add_argument("--stdp", action="store_true", help="plastic weights (gn_config.stdp_alpha = 0.5 / ms, stdp_beta = 0.05 / ms; "
                                                       "DESIGN.md 6.7): delivery at arrival time, eq. 32-33 every step -- a different "
                                                       "workload; the CPU baseline (static oracle) is skipped")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this library has no CPU fallback)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    import paper_0908_3934_b200 as gn
    from gn_inputs import make_config

    K, W, S = args.steps, max(args.warmup, 3), args.sim_steps
    t0 = time.time()
    # replicas only: rank r steps its own independent network of the same recipe
    net_in, cfg = make_config(args.config, n=args.n, seed=rank_seed(args.config, rank))
    if args.model == "hh":
        from gn_inputs import as_hodgkin_huxley
        cfg = as_hodgkin_huxley(cfg)
    if args.psc_alpha:
        cfg = dict(cfg, classes=[dict(c, psc_alpha=1.0) for c in cfg["classes"]], name=cfg["name"] + "+alpha_psc")
    if args.stdp:
        cfg = dict(cfg, name=cfg["name"] + "+stdp")
    N, E = net_in.n_vertices, net_in.n_edges
    log(f"[rank {rank}] inputs in {time.time() - t0:.1f} s: N={N} E={E} mean out-degree {E / N:.1f}")
    obs = int(cfg["obs_stride"])
    frames_per_step = S // obs if obs else 0

    def create(arrays=None):
        a = arrays or dict(pos=net_in.positions, row=net_in.row_offsets, tgt=net_in.targets, w=net_in.weights,
                           cls=net_in.vertex_class, net=net_in.net_offsets)
        c = gn.make_config(N, net_in.dim, E, cfg["ring_slots"], cfg["dt_ms"], cfg["speed"], len(cfg["classes"]),
                           n_networks=net_in.n_networks, tau_ca_ms=cfg["tau_ca_ms"], ca_jump=cfg["ca_jump"],
                           obs_gain=cfg["obs_gain"], obs_offset=cfg["obs_offset"], obs_sigma=cfg["obs_sigma"],
                           obs_stride=obs, raster_capacity_steps=S, trace_capacity_frames=max(frames_per_step, 1) if obs else 0,
                           seed=cfg["seed"], delivery_mode={"auto": 0, "ring": 1, "queue": 2}[args.delivery],
                           queue_group=args.queue_group, stdp_alpha=0.5 if args.stdp else 0.0, stdp_beta=0.05 if args.stdp else 0.0)
        return gn.gn_create(c, cfg["classes"], a["pos"], a["row"], a["tgt"], a["w"], None, a["cls"], None, a["net"],
                            device=dev)

    def counters(g):
        c = gn.gn_read_state(g, gn.GN_COUNTERS)
        return int(c[0]), int(c[1]), int(c[2])

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident arm ------------------------------------------------------------------------
    g = create()
    for _ in range(W):
        gn.gn_step(g, S)
    barrier()
    c0 = counters(g)
    _, l0 = gn.gn_profile_read(g)
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(K):
        gn.gn_step(g, S)
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    c1 = counters(g)
    _, l1 = gn.gn_profile_read(g)
    launches = int(l1[4] - l0[4])
    ms, spikes, events = reduce_over_ranks(dist, dev, ms, c1[1] - c0[1], c1[2] - c0[2])
    sec = ms * 1e-3
    sim_steps = K * S
    value = world * N * sim_steps / sec

    # ---- per-kernel pass: EXACTLY the timed steps again (the run is deterministic and starts from rest, so a
    # fresh handle stepped through the same W warm-up steps is in the state the timed pass started from), this
    # time with a CUDA event wherever the kind of kernel changes (gn_profile: everything serialised on one stream)
    del g
    g = create()
    for _ in range(W):
        gn.gn_step(g, S)
    cp0 = counters(g)
    gn.gn_profile(g, True)
    gn.gn_step(g, sim_steps)
    kms, kn = gn.gn_profile_read(g)
    gn.gn_profile(g, False)
    cp1 = counters(g)
    assert cp0 == c0 and cp1 == c1, "the per-kernel pass did not replay the timed steps"
    peak, peak_src = peaks()
    driver = int(gn.gn_read_state(g, gn.GN_DRIVER)[0])      # which step driver gn_create chose: read back, not guessed
    queue_mode = driver == gn.GN_DRIVER_QUEUE       # delivers once per slot group; ring mode (and plastic mode) every step
    persist = driver == gn.GN_DRIVER_PERSISTENT
    resident = persist or driver == gn.GN_DRIVER_RESIDENT
    names = ["gn_persist_kernel (a1-a5, one cooperative launch per call)" if persist else
             "gn_resident_kernel (a1-a5, one CTA or cluster per network)" if resident else
             "gn_update_kernel (a1-a3 + a4 fused)" if kn[1] == 0 else "gn_update_kernel (a1-a3)",
             "gn_log_kernel (a3 compaction + a4: spikes into the log)" if queue_mode else
             "gn_arrive_kernel (a4 at arrival time: plastic weights)" if args.stdp else "gn_deliver_kernel (a4)",
             "gn_observe_kernel (a5)",
             "gn_spikes_kernel + gn_plast_kernel (eq. 32, eq. 33)" if args.stdp else
             "gn_fold_kernel (a4: expansion of the log + ring reductions)"]
    p_events, p_spikes = cp1[2] - cp0[2], cp1[1] - cp0[1]
    # algorithmic bytes per launch: 17 B per event (+12 B per fired source) for the
    # delivery of either mode (queue mode, per slot group: the logging kernel takes the 12 B per fired source, the fold
    # kernel the 17 B per event of the group it expands)
    delivery_bytes = p_events * EVENT_BYTES + p_spikes * SOURCE_BYTES
    per_vertex = HH_BYTES_PER_VERTEX if args.model == "hh" else UPDATE_BYTES_PER_VERTEX
    if args.stdp:
        # plastic mode, per step: arrivals re-read the raster of the last D - 1 steps (N/8 bytes each) and move 8 B edge + 4 B
        # weight + 8 B ring word per event; eq. 33 moves 8 B edge + 8 B weight per arrival (weakening), 8 B in-edge entry + 8 B
        # edge + 8 B weight per in-edge of a fired vertex (strengthening; as many as events in the long run), and eq. 32 8 B per vertex
        ring_d = cfg["ring_slots"]
        arrive_b = (p_events * 20.0 + sim_steps * (ring_d - 1) * N / 8.0)
        plast_b = (p_events * (16.0 + 24.0) + sim_steps * ((ring_d - 1) * N / 8.0 + N * 8.0))
    kbytes = [N * (per_vertex + (UPDATE_BYTES_PER_VERTEX_OBS if obs else 0.0)) * (sim_steps / max(int(kn[0]), 1))
              + (delivery_bytes / max(int(kn[0]), 1) if kn[1] == 0 else 0.0),
              (arrive_b if args.stdp else p_spikes * SOURCE_BYTES if queue_mode else delivery_bytes) / max(int(kn[1]), 1),
              N * 8.0,
              (plast_b if args.stdp else p_events * EVENT_BYTES) / max(int(kn[3]), 1)]
    traffic_tab, traffic_src = measured_traffic()
    l2_bw, hbm_rmw = gn.gn_debug_stream_ceilings(device=dev)       # streaming read-modify-write, from L2 and from HBM: measured here
    kernels = []
    for k in range(4):
        if kn[k] == 0:
            continue
        avg_s = kms[k] * 1e-3 / kn[k]
        row = {"kernel": names[k], "launches": int(kn[k]), "avg_us": avg_s * 1e6, "share": float(kms[k] / kms.sum()),
               "bytes_per_launch": kbytes[k], "achieved": kbytes[k] / avg_s / 1e9, "frac": kbytes[k] / avg_s / 1e9 / peak}
        tr = traffic_tab.get(names[k].split()[0] + ("_hh" if args.model == "hh" and k == 0 else ""))
        if tr is not None and not resident:
            # what DRAM moved for this kernel in the committed ncu capture named in traffic_source (NOT measured in this run;
            # per event where the kernel's work is per event, scaled by this run's event count) over the live time
            row["traffic"] = tr[1] * p_events / kn[k] if tr[1] is not None else tr[0]
            row["dram_frac"] = row["traffic"] / avg_s / 1e9 / peak
        # what binds the kernel: "hbm" only when DRAM really carries at least half of the algorithmic bytes AND one of the two
        # fractions is past one half; a working set served by L2 is rated against the L2 ceiling measured in this run
        if k == 0 and resident:
            row["bound"] = "alu"             # state in registers, ring in shared memory: the algorithmic bytes are not moved at all
            row["frac"] = row["achieved"] = None
            row["bytes_not_moved"] = row.pop("bytes_per_launch")
        elif k == 3 and queue_mode or k == 1 and not queue_mode and not args.stdp:
            row["bound"] = "l2-atomics"      # one int32 reduction per event in the L2 (a4_delivery.atomic_path has the ceiling)
        elif args.stdp and k in (1, 3):
            row["bound"] = "latency"
        else:
            df = row.get("dram_frac")
            if k == 0:
                row["l2_frac"] = kbytes[k] / avg_s / l2_bw
            row["bound"] = ("hbm" if df is not None and df >= 0.5 * row["frac"] and max(df, row["frac"]) >= 0.5 else
                            "l2" if df is not None and df < 0.5 * row["frac"] else "latency")
        kernels.append(row)
    a4_s = (kms[1] + kms[3]) * 1e-3
    a4 = {"what": "a4 delivery as a whole (routing + folding), 17 B per event + 12 B per fired source",
          "bytes": p_events * EVENT_BYTES + p_spikes * SOURCE_BYTES, "ms": a4_s * 1e3,
          "achieved": (p_events * EVENT_BYTES + p_spikes * SOURCE_BYTES) / max(a4_s, 1e-12) / 1e9}
    a4["frac"] = a4["achieved"] / peak if a4_s > 0 else None      # (no separate delivery kernel: a4 is inside the update / persistent kernel)
    if a4_s <= 0:
        a4["achieved"] = None
    if queue_mode and a4_s > 0:
        # what bounds event delivery is not HBM but the L2's atomic path: one int32 reduction per event is the
        # least any atomic delivery does, and the fold gathers each event's 8-byte edge in short random segments on top.  Both
        # ceilings are MEASURED here, on this device, with the bare access pattern (gn_debug_ceilings).
        group = args.queue_group or 8
        seg = max(1, int(round(E / N * group / cfg["ring_slots"])))
        red_only, gather_red = gn.gn_debug_ceilings(seg, device=dev)
        fold_s = kms[3] * 1e-3
        a4["atomic_path"] = {"bound": "l2-atomics", "unit": "events/s", "achieved": p_events / max(fold_s, 1e-12),
                             "peak": red_only, "frac": p_events / max(fold_s, 1e-12) / red_only,
                             "achieved_incl_logging": p_events / a4_s, "frac_incl_logging": p_events / a4_s / red_only,
                             "gather_plus_red_reference": gather_red, "segment_edges": seg,
                             "peak_source": "measured in this run by gn_debug_ceilings: scattered int32 RED.ADD into a 16 MB "
                                            "L2-resident region, one per event -- the least any atomic delivery does "
                                            "(gather_plus_red_reference: the same loop with each event's 8-byte edge gathered "
                                            f"first, in random {seg}-edge segments of a 2 GB array: a reference point, not a "
                                            "ceiling -- the fold kernel keeps more loads in flight); achieved = delivered "
                                            "events / summed gn_fold_kernel time"}
    dom = max(kernels, key=lambda r: r["share"])
    roofline = {"bound": dom["bound"], "kernel": dom["kernel"], "achieved": dom["achieved"], "peak": peak, "unit": "GB/s",
                "frac": dom["frac"], "traffic": dom.get("traffic"), "traffic_source": traffic_src if "traffic" in dom else None,
                "dram_frac": dom.get("dram_frac"), "peak_source": peak_src,
                "stream_ceilings": {"l2_gbs": l2_bw / 1e9, "hbm_read_modify_write_gbs": hbm_rmw / 1e9,
                                    "source": "gn_debug_stream_ceilings, measured in this run: 128-bit read-modify-write over a "
                                              "32 MB (L2-resident) and a 2 GB buffer, bytes read + written per second"},
                "note": "achieved / frac = ALGORITHMIC bytes over the live CUDA-event time against the HBM peak (the contract's "
                        "definition), whatever `bound` says; `bound` names what really limits the kernel (rule in bench.py: hbm only "
                        "when DRAM carries at least half of the algorithmic bytes) and the matching rating sits beside it: "
                        "l2-atomics -> a4_delivery.atomic_path (measured RED ceiling), l2 / hbm -> kernels[].l2_frac and "
                        "dram_frac (traffic from the committed ncu capture in traffic_source, not from this run), alu -> alu "
                        "(DESIGN.md 6.3, 6.5, 7)",
                "timing": "the SAME K steps as the timed pass, replayed from rest on a fresh handle with a CUDA event at every "
                          "kernel boundary (gn_profile; serialised on one stream)",
                "kernels": kernels, "a4_delivery": a4, "profile_pass_events_per_sim_step": p_events / sim_steps,
                "timed_pass_events_per_sim_step": (c1[2] - c0[2]) / sim_steps}
    if resident:                # nothing moves through HBM: lane-instructions of the contract against the SMs' issue rate
        upd = kernels[0]
        ops = HH_FP32_PER_VERTEX + 34.0 if args.model == "hh" else IZH_OPS_PER_VERTEX
        alu_peak = FP32_LANES_PER_SM * SM_COUNT * SM_HZ
        ach = N * ops * sim_steps / (kms[0] * 1e-3)
        roofline.update({"achieved": ach / 1e12, "peak": alu_peak / 1e12, "unit": "T lane-instr/s", "frac": ach / alu_peak,
                         "traffic": None, "dram_frac": None,
                         "peak_source": "148 SMs x 128 lanes x 1.965 GHz (B200_PROFILING.md unit counts and clock)",
                         "ops_per_vertex_step": ops,
                         "ops_source": "counted from the arithmetic contract (bench.py IZH_OPS_PER_VERTEX / HH_FP32_PER_VERTEX + "
                                       "generator and detection), an FMA counts once; the kernel is below this ceiling because "
                                       "one barrier per step serialises it (DESIGN.md 6.5)"})
    if args.model == "hh" and not resident:      # the update kernel against the fp32 pipe as well: which of the two bounds it depends on the measurement
        upd = kernels[0]
        fp32_peak = FP32_LANES_PER_SM * SM_COUNT * SM_HZ
        ach = N * HH_FP32_PER_VERTEX * (sim_steps / max(int(kn[0]), 1)) / (upd["avg_us"] * 1e-6)
        roofline["alu"] = {"bound": "alu", "kernel": upd["kernel"], "achieved": ach / 1e12, "peak": fp32_peak / 1e12,
                           "unit": "T fp32 instr/s", "frac": ach / fp32_peak,
                           "peak_source": "148 SMs x 128 fp32 lanes x 1.965 GHz (B200_PROFILING.md unit counts and clock; an FMA "
                                          "counts once); 141 fp32 operations of the contract per vertex-step"}
    if dom["kernel"].startswith("gn_deliver"):   # ring mode only: what DRAM moves when every event misses L2
        sect = (p_events * SECTOR_EVENT_BYTES + p_spikes * SOURCE_BYTES) / max(int(kn[1]), 1)
        roofline["sector_granular"] = {"bytes_per_launch": sect, "achieved": sect / (dom["avg_us"] * 1e-6) / 1e9,
                                       "frac": sect / (dom["avg_us"] * 1e-6) / 1e9 / peak}
    del g

    # ---- end to end through the C ABI with HOST buffers ----------------------------------------------
    e2e = None
    if not args.no_e2e:
        pin = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        host = dict(pos=pin(net_in.positions), row=pin(net_in.row_offsets.view(np.int64)), tgt=pin(net_in.targets.view(np.int32)),
                    w=pin(net_in.weights), cls=pin(net_in.vertex_class),
                    net=None if net_in.net_offsets is None else pin(net_in.net_offsets.view(np.int32)))
        words = (N + 31) // 32
        # the step's result (the raster of its S simulated steps) leaves through a device staging buffer and a copy stream,
        # so that its device -> host copy runs beside the next step's kernels (two of each: a buffer is reused two steps on)
        rast_host = [torch.empty((S, words), dtype=torch.int32).pin_memory() for _ in range(2)]
        rast_dev = [torch.empty((S, words), dtype=torch.int32, device=dev) for _ in range(2)]
        copied = [torch.cuda.Event() for _ in range(2)]
        copy_stream = torch.cuda.Stream(device=dev)
        v_host = torch.empty(N, dtype=torch.float32).pin_memory()
        z_host = torch.empty((max(frames_per_step, 1), N), dtype=torch.float32).pin_memory() if obs else None
        h2d = sum(t.numel() * t.element_size() for t in host.values() if t is not None)
        d2h = rast_host[0].numel() * 4 + (z_host.numel() * 4 if obs else 0) + v_host.numel() * 4 / K
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g2 = create(host)                                    # host -> device of every input, validation, quantisation, delays
        main = torch.cuda.current_stream(dev)
        for k in range(K):
            gn.gn_step(g2, S)
            b = k & 1
            if k >= 2:
                main.wait_event(copied[b])                   # the buffer's previous copy has left
            gn.gn_read_raster(g2, k * S, S, rast_dev[b])     # device destination: asynchronous on the handle's stream
            ready = torch.cuda.Event()
            ready.record(main)
            copy_stream.wait_event(ready)
            with torch.cuda.stream(copy_stream):
                rast_host[b].copy_(rast_dev[b], non_blocking=True)      # device -> host of the step's result
                copied[b].record(copy_stream)
            if obs:
                gn.gn_observe(g2, k * frames_per_step, frames_per_step, z_host.numpy())
        gn.gn_read_state(g2, gn.GN_V, v_host.numpy())
        main.wait_stream(copy_stream)
        e1.record()
        barrier()
        ems = e0.elapsed_time(e1)
        ems, _, _ = reduce_over_ranks(dist, dev, ems, 0, 0)
        e2e = {"value": world * N * sim_steps / (ems * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d / K,
               "d2h_bytes_per_step": d2h, "ms_total": ems,
               "what": "gn_create from pinned host arrays (upload + validation + quantisation + eq. 25 delays) + K x "
                       "[gn_step(S) + gn_read_raster of the S steps, through a device staging buffer and a copy stream, to pinned "
                       "host memory] + final V to host"}
        del g2

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": workload_name(net_in, cfg, args), "sim_steps_per_step": S,
                   "l2": "no flush: working set (ring + edges + state) >> 126 MB L2",
                   "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (no collective)"},
        "events_per_s": events / sec, "real_time_factor": sim_steps * cfg["dt_ms"] * 1e-3 / sec,
        "us_per_sim_step": ms * 1e3 / sim_steps,
        "mean_rate_hz": spikes / (world * N * sim_steps * cfg["dt_ms"] * 1e-3),
        "events_per_sim_step": events / world / sim_steps,
        "roofline": roofline, "clocks": clocks, "gpu_launches": launches, "e2e": e2e,
    }
    if args.stdp:
        line["config"]["workload"] += " + STDP (alpha 0.5 / ms, beta 0.05 / ms)"
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.stdp:
        line["cpu_baseline"] = cpu_baseline(net_in, cfg)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
