#!/usr/bin/env python
"""bench.py -- throughput of the hot path (transport + imaging) in photon packets/s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2] [--batch B] [--impl reference]

A "step" is one pass of the whole hot path over one batch of B new packets of the workload:
krp_transport(B) (emit, flights, scatterings, event records) followed by krp_image (every event toward
every observer, attenuated to the grid edge, summed into the fp64 I,Q,U,V maps).  Packet ids continue
from step to step, so K steps are K*B distinct packets of the job.  Inputs are seeded and synthetic
(paper_2512_01283_b200.inputs, recipe in DESIGN.md).  BASELINE.json's metric names no config, so the default
workload is the largest single-GPU one, configs[4] (C5: turbulent cloud, 512^3 cells, 8 observers at 512x512);
--workload c1..c4 time the others.

One JSON line goes to stdout (rank 0).  `value` is device-resident throughput; `e2e` is the same metric
through the C ABI with HOST buffers (grid upload, transport, imaging, image download inside the timed
region); `roofline` is the dominant kernel against its binding ceiling; `cpu_baseline` is the fp64 oracle
on this box's host cores.  `--impl reference` times the oracle alone (rank 0 only).
"""
import argparse
import json
import math
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "photon packets/sec (transport+imaging)"
UNIT = "packets/s"

# Algorithmic work per unit: bytes that must move and thread-instructions that must issue
# per cell step of the two hot loops, for the two cell layouts, and per ray / flight outside the loop.  The loop bodies
# as ptxas emits them, with the counts marked, are in profiles/r2_sass_hot_loops.md (executed: 18.5 / 52 imaging,
# 31 / ~230 flight); the algorithmic count is what the written-out algorithm needs:
#   image_inst   scalar: min3, sub, 3 setp, 3 predicated fadd + 3 iadd, address, gather, fma, sentinel test, branch
#                general (per-observer coefficient array): march 13, gather 3, sincos of 2 eta and rotation in 7, series
#                of sinh/cosh-1/sin/cos-1 and the update as 16 chained FFMAs 22, loop test 3
#   flight_inst  scalar: re-based march (13) + optical-depth product, fp64 compare and subtract, gather, tests
#                general: fp64 re-based march, fp64 mu and table segment, eta, App. A series, rotation, depth bookkeeping
ALGO = {
    "scalar":  dict(cell_bytes=4,  image_inst=16, flight_inst=23, ray_inst=250, flight_fixed_inst=200),
    "general": dict(cell_bytes=16, image_inst=48, flight_inst=110, ray_inst=250, flight_fixed_inst=300),
}
EVENT_BYTES, CONTRIB_BYTES = 48, 32
N_SM, LANES_PER_SM = 148, 128          # B200: 148 SMs x 4 schedulers x 32 lanes, one warp-instruction per scheduler and clock
# Which ceiling binds a kernel, its DRAM traffic and the instructions it executes are NOT constants of this file: they are
# parsed from the committed ncu captures of this same command that profiles/roofline_sources.json names per workload and
# kernel class (read_capture below).


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=6)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="krp", choices=["krp", "reference"])
    ap.add_argument("--workload", default="c5", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--batch", type=int, default=0, help="packets per step and GPU (0 = workload default)")
    ap.add_argument("--n", type=int, default=0, help="override the grid size (testing only; marks the line reduced)")
    ap.add_argument("--form", default="events", choices=["events", "twostep"],
                    help="events: the north_star's form (per-event imaging, the contract's metric); twostep: the paper's own form "
                         "(every segment deposited into S(Omega_cam, x), one ray per pixel at the end of the timed steps)")
    ap.add_argument("--tune", default="", help="measurement only: transport_block,image_block,blocks_per_sm,flight_burst for krp_tune (0 keeps)")
    ap.add_argument("--fused", type=int, default=-1, help="measurement only: krp_tune_fused(max_packets); -1 keeps the library's default")
    ap.add_argument("--schedule", default="", help="measurement only: dir_sort,obs_cells,order_policy for krp_tune_schedule (-1 keeps)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    return ap.parse_args()


DEFAULT_BATCH = {"c1": 100000, "c2": 1 << 25, "c3": 1 << 22, "c4": 1 << 23, "c5": 1 << 22}


def make_workload(args):
    from paper_2512_01283_b200 import inputs
    kw = {}
    if args.n:
        kw["n"] = args.n
    cfg = inputs.make(args.workload, **kw)
    batch = args.batch or DEFAULT_BATCH[args.workload]
    return cfg, batch


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms while the timed region runs."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline and --impl reference): oracle/ as it stands, one host thread
# ------------------------------------------------------------------------------------------
def oracle_setup(cfg):
    from oracle import OracleModel, Observer as OraObserver
    m = OracleModel(cfg["nx"], cfg["ny"], cfg["nz"], cfg["bounds"], cfg["density"], cfg["bfield"], cfg["mueller"],
                    cfg["opacity"], w_min=cfg["w_min"], max_scatter=cfg["max_scatter"])
    s = cfg["source"]
    m.source_set(s["kind"], s["pos"], s["dir"], s.get("cell_weight"), s.get("emit_records", 0))
    obs = [OraObserver.make(o["theta"], o["phi"], o["center"], o["half_w"], o["half_h"]) for o in cfg["observers"]]
    return m, obs


def oracle_step(m, obs, cfg, id0, n):
    """Transport + image packets [id0, id0+n) with the oracle; returns (seconds, events)."""
    from oracle import OracleEvents, OracleStats
    ev = OracleEvents(max(1024, 64 * n))
    st = OracleStats()
    t0 = time.perf_counter()
    m.transport(id0, n, cfg["seed"], ev, st)
    m.image(ev, obs, cfg["npix"], cfg["npix"], stats=st, second_moment=False)
    return time.perf_counter() - t0, st.as_dict()


def oracle_timed(cfg, seconds, chunk=500):
    """Time the oracle on packets [0, n) of the workload, n grown in chunks until `seconds` have passed."""
    m, obs = oracle_setup(cfg)
    oracle_step(m, obs, cfg, 0, 50)                     # touch the arrays once
    t = 0.0
    n = 0
    events = 0
    while t < seconds:
        dt, st = oracle_step(m, obs, cfg, n, chunk)
        t += dt
        n += chunk
        events += st["events"]
    return dict(value=n / t, unit=UNIT, cores=1, kind="oracle", scatterings_per_s=events / t,
                sample="packet ids [0,%d) of the workload, transport+imaging, single thread fp64, %.1f s" % (n, t))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg, _ = make_workload(args)
    m, obs = oracle_setup(cfg)
    # each step is a bounded sample of the workload: `chunk` packets sized from a pilot so that the whole
    # run (warm-up + steps) takes about two minutes at most
    dt, _ = oracle_step(m, obs, cfg, 0, 200)
    per_packet = dt / 200
    total = max(args.steps + args.warmup, 1)
    chunk = int(max(100, min(200000, 100.0 / total / per_packet)))
    nid = 1000
    for _ in range(args.warmup):
        oracle_step(m, obs, cfg, nid, chunk); nid += chunk
    t = 0.0
    events = 0
    for _ in range(args.steps):
        dt, st = oracle_step(m, obs, cfg, nid, chunk); nid += chunk
        t += dt
        events += st["events"]
    value = args.steps * chunk / t
    sample = "%d packets per step of the workload's id stream, single thread fp64" % chunk
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "packets_per_step": chunk, "observers": len(cfg["observers"]),
                   "npix": cfg["npix"], "note": "oracle (oracle/krp_oracle.c) on host cores, bounded sample per step"},
        "scatterings_per_s": events / t,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------
# the CUDA leg
# ------------------------------------------------------------------------------------------
def read_capture(workload, cls):
    """Counters of one launch of kernel class `cls` ("flight" / "image") of `workload`, from the committed ncu captures
    that profiles/roofline_sources.json names: {"details": text of `ncu --page details`, "raw": csv of `ncu --page raw --csv`}.
    Returns None when no capture is committed for it."""
    idx = os.path.join(ROOT, "profiles", "roofline_sources.json")
    if not os.path.exists(idx):
        return None
    with open(idx) as f:
        src = json.load(f).get(workload, {}).get(cls)
    if not src:
        return None
    out = {"files": src}
    det = os.path.join(ROOT, src["details"])
    if os.path.exists(det):
        want = {"DRAM Throughput": "dram_pct", "Issue Slots Busy": "issue_pct", "L2 Cache Throughput": "l2_pct",
                "L1/TEX Cache Throughput": "l1_pct", "Duration": "duration", "Achieved Occupancy": "occupancy_pct",
                "Avg. Active Threads Per Warp": "active_threads", "Registers Per Thread": "registers"}
        with open(det) as f:
            for line in f:
                t = line.split()
                for key, name in want.items():
                    if line.strip().startswith(key + " ") and name not in out:
                        try:
                            val = float(t[-1].replace(",", ""))
                        except ValueError:
                            continue
                        if name == "duration":
                            unit = t[-2]
                            val *= {"us": 1e-3, "ms": 1.0, "s": 1e3, "ns": 1e-6}.get(unit, 1.0)
                            name = "duration_ms"
                        out[name] = val
                    if line.strip().startswith(key) and "krp_k_" in line:
                        pass
                if "krp_k_" in line and "kernel" not in out:
                    out["kernel"] = line.strip().split("(")[0].replace("void ", "")
    raw = os.path.join(ROOT, src.get("raw", ""))
    if src.get("raw") and os.path.exists(raw):
        import csv
        with open(raw) as f:
            rows = [r for r in csv.reader(f) if r]
        hdr = next((r for r in rows if "Kernel Name" in r), None)
        if hdr:
            data = rows[rows.index(hdr) + 2] if len(rows) > rows.index(hdr) + 2 else None      # header, units, first kernel
            units = rows[rows.index(hdr) + 1]
            def col(name):
                if data is None or name not in hdr:
                    return None
                k = hdr.index(name)
                try:
                    v = float(data[k].replace(",", ""))
                except ValueError:
                    return None
                return v * {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "byte": 1.0}.get(units[k], 1.0)
            r, w = col("dram__bytes_read.sum"), col("dram__bytes_write.sum")
            if r is not None and w is not None:
                out["dram_bytes"] = r + w
            ti = col("smsp__thread_inst_executed.sum")
            if ti is not None:
                out["thread_inst_executed"] = ti
            wi = col("smsp__inst_executed.sum")
            if wi is not None:
                out["warp_inst_executed"] = wi
    return out


def make_grid(krp, cfg, dens, bf, weight):
    g = krp.Grid(cfg["nx"], cfg["ny"], cfg["nz"], cfg["bounds"], dens, bf, cfg["mueller"], cfg["opacity"],
                 w_min=cfg["w_min"], max_scatter=cfg["max_scatter"])
    s = cfg["source"]
    g.source_set(s["kind"], s["pos"], s["dir"], weight, s.get("emit_records", 0))
    return g


def run_krp(args):
    import torch
    import torch.distributed as dist
    from paper_2512_01283_b200 import krp, shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg, batch = make_workload(args)
    n_obs, npix, seed = len(cfg["observers"]), cfg["npix"], cfg["seed"]
    dens = torch.from_numpy(cfg["density"]).to(dev)
    bf = None if cfg["bfield"] is None else torch.from_numpy(cfg["bfield"]).to(dev)
    w_host = cfg["source"].get("cell_weight")
    weight = None if w_host is None else torch.from_numpy(np.ascontiguousarray(w_host, np.float32).ravel()).to(dev)
    obs = [krp.make_observer(o["theta"], o["phi"], o["center"], o["half_w"], o["half_h"]) for o in cfg["observers"]]
    g = make_grid(krp, cfg, dens, bf, weight)
    if args.tune:
        g.tune(*[int(x) for x in args.tune.split(",")])
    if args.fused >= 0:
        g.tune_fused(args.fused)
    if args.schedule:
        g.tune_schedule(*[int(x) for x in args.schedule.split(",")])

    # pilot (untimed): events per packet of this workload, to size the event buffer once
    pilot = min(batch, 1 << 16)
    g.packet_id_set(1 << 40)
    g.transport(pilot, seed)
    st = g.stats_get()
    epp = st["events"] / max(st["packets"], 1)
    g.events_clear()
    torch.cuda.synchronize()
    ev_cap = int(batch * (1.25 * epp + 0.05)) + (1 << 16)
    g.events_reserve(ev_cap)

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    total_steps = args.warmup + args.steps
    E = lambda: torch.cuda.Event(enable_timing=True)
    marks = [(E(), E(), E()) for _ in range(args.steps)]

    twostep = args.form == "twostep"
    if twostep:
        g.sgrid_begin(obs)

    def step(i, mark=None):
        first, cnt = shard.step_id_range(i, rank, world, batch)
        g.packet_id_set(first)
        flush.zero_()
        if mark:
            mark[0].record()
        g.transport(cnt, seed)
        if mark:
            mark[1].record()
        if twostep:
            g.events_clear()               # the paper's form does not use the event buffer
        else:
            g.image(obs, npix, npix)
        if mark:
            mark[2].record()

    for i in range(args.warmup):
        step(i)
    g.stats_reset()
    g.timing_enable(True)
    g.timing_get()
    img = torch.zeros((n_obs, 4, npix, npix), dtype=torch.float64, device=dev)
    launches0 = g.launch_count()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    t_start, t_end = E(), E()
    t_start.record()
    for i in range(args.steps):
        step(args.warmup + i, marks[i])
    if twostep:
        g.image_rays(obs, npix, npix)      # step 2 of the paper's form, once for all packets of the timed steps
    t_end.record()
    barrier()
    clocks = sampler.stop() if sampler else None
    ms_total = t_start.elapsed_time(t_end)
    ms_own = ms_total                      # this rank's own time over the K steps (the max over ranks replaces ms_total below)
    timing = g.timing_get()
    g.timing_enable(False)
    launches = g.launch_count() - launches0
    # end of job: the one exchange of the path, sum of the per-rank maps (outside the per-step timing)
    g.image_get(out=img)
    shard.reduce_images(img)
    torch.cuda.synchronize()
    t_tr = float(np.mean([m[0].elapsed_time(m[1]) for m in marks]))
    t_im = float(np.mean([m[1].elapsed_time(m[2]) for m in marks]))
    st = g.stats_get()
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
        cnt = torch.tensor([st["packets"], st["events"], st["steps_transport"], st["steps_image"], st["contributions"]],
                           dtype=torch.float64, device=dev)
        dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
        tot = dict(zip(["packets", "events", "steps_transport", "steps_image", "contributions"], cnt.tolist()))
    else:
        tot = st
    sec = ms_total * 1e-3
    value = tot["packets"] / sec
    assert tot["packets"] == args.steps * batch * world, (tot["packets"], args.steps, batch, world)

    # roofline of the dominant kernel (this rank's launches), from the library's own per-launch CUDA events
    # on the launching stream (krp_timing_*): flight kernels (one launch per scattering order) or imaging
    # kernels (one launch per observer), whichever took more of the step
    pk = peaks()
    mode = "scalar" if (cfg["bfield"] is None and cfg["opacity"].shape[0] == 1) else "general"
    A = ALGO[mode]
    K = args.steps
    alu_peak = N_SM * LANES_PER_SM * pk["sm_max_mhz"] * 1e6          # thread-instructions/s at the maximum SM clock
    rays = st["events"] * n_obs
    flights = st["packets"] + st["events"]                             # an upper bound: every event but the last starts one
    work = {
        "image": dict(kernel="krp_k_image<true,false>" if mode == "scalar" else "krp_k_image<false,true>", steps=st["steps_image"],
                      bytes=st["steps_image"] * A["cell_bytes"] + rays * EVENT_BYTES + st["contributions"] * CONTRIB_BYTES,
                      inst=st["steps_image"] * A["image_inst"] + rays * A["ray_inst"]),
        # scalar mode: one launch per step = the one-kernel form of small batches (krp_tune_fused), else one per scattering order
        "flight": dict(kernel=("krp_k_packets_scalar" if timing["flight"][1] <= args.steps else "krp_k_flight_scalar_static")
                       if mode == "scalar" else "krp_k_flight_general", steps=st["steps_transport"],
                       bytes=st["steps_transport"] * A["cell_bytes"] + flights * 64 + st["events"] * 56,
                       inst=st["steps_transport"] * A["flight_inst"] + flights * A["flight_fixed_inst"]),
    }
    kernels = {}
    for cls, (ms, n_l) in timing.items():
        kernels[cls] = {"ms_per_step": ms / K, "launches_per_step": n_l / K, "share_of_step": ms / ms_own}
    if twostep:
        work["image"] = dict(kernel="krp_k_deposit", steps=st["segments"], bytes=st["segments"] * (A["cell_bytes"] + 32 * n_obs),
                             inst=st["segments"] * 150)
        timing = dict(timing, image=timing["deposit"])
    dom = max(("image", "flight"), key=lambda c: timing[c][0])
    per_class = {}
    for cls in ("image", "flight"):
        Wc = work[cls]
        t_c = timing[cls][0] * 1e-3                                     # seconds over the K timed steps, CUDA events per launch
        n_l = max(timing[cls][1], 1)
        if t_c <= 0:
            continue
        cap = read_capture(args.workload, cls)
        f_hbm = Wc["bytes"] / t_c / (pk["hbm_gbs"] * 1e9)
        f_alu = Wc["inst"] / t_c / alu_peak
        rec = {"kernel": (cap or {}).get("kernel", Wc["kernel"]), "launches_per_step": n_l / K, "avg_launch_ms": 1e3 * t_c / n_l,
               "kernel_ms_per_step": 1e3 * t_c / K, "share_of_step": timing[cls][0] / ms_own,
               "cell_steps_per_step": Wc["steps"] / K, "cell_steps_per_s": Wc["steps"] / t_c,
               "algorithmic_bytes_per_step": Wc["bytes"] / K, "algorithmic_inst_per_step": Wc["inst"] / K,
               "frac_hbm": f_hbm, "frac_alu": f_alu, "traffic": None, "capture": None}
        # which ceiling binds: read from the committed capture of this kernel -- issue slots busy against DRAM throughput;
        # when neither reaches 60 % the kernel is bound by latency / divergence, not by a throughput ceiling
        bound = "alu" if f_alu >= f_hbm else "hbm"
        if cap:
            issue, dram = cap.get("issue_pct"), cap.get("dram_pct")
            if issue is not None and dram is not None:
                bound = "latency" if max(issue, dram) < 60.0 else ("alu" if issue >= dram else "hbm")
            rec["traffic"] = cap.get("dram_bytes")
            rec["capture"] = {k: cap.get(k) for k in ("files", "issue_pct", "dram_pct", "l2_pct", "l1_pct", "duration_ms",
                                                       "active_threads", "occupancy_pct", "registers")}
            if cap.get("warp_inst_executed") and cap.get("active_threads") and cap.get("duration_ms"):
                # executed (not algorithmic) thread-instructions of the captured launch against the same issue ceiling, at the
                # capture's own duration: what the SASS really issues, idle lanes excluded
                rec["frac_alu_executed_in_capture"] = (cap["warp_inst_executed"] * cap["active_threads"] /
                                                       (cap["duration_ms"] * 1e-3) / alu_peak)
        rec["bound"] = bound
        per_class[cls] = rec
    D = per_class[dom]
    use_hbm = D["bound"] == "hbm" or (D["bound"] == "latency" and D["frac_hbm"] > D["frac_alu"])
    t_dom = timing[dom][0] * 1e-3
    if use_hbm:
        roof = {"bound": D["bound"], "achieved": work[dom]["bytes"] / t_dom / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": D["frac_hbm"]}
    else:
        roof = {"bound": D["bound"], "achieved": work[dom]["inst"] / t_dom / 1e12, "peak": alu_peak / 1e12, "unit": "Tinst/s", "frac": D["frac_alu"]}
    roof.update({k: v for k, v in D.items() if k != "bound"})
    roof.update({"peak_source": pk["source"], "peak_alu": "%d SMs x 4 schedulers x 32 lanes x %.0f MHz" % (N_SM, pk["sm_max_mhz"]),
                 "algorithmic_unit": "per cell step %d B and %d (image) / %d (flight) thread-instructions; per ray 48 B + 32 B and %d; "
                                     "per flight 64 B + 56 B and %d (DESIGN.md section 8, SASS excerpts in profiles/)"
                                     % (A["cell_bytes"], A["image_inst"], A["flight_inst"], A["ray_inst"], A["flight_fixed_inst"]),
                 "other": {c: v for c, v in per_class.items() if c != dom}, "kernels": kernels})
    return dict(world=world, rank=rank, cfg=cfg, batch=batch, value=value, ms_total=ms_total, clocks=clocks, roof=roof,
                t_tr=t_tr, t_im=t_im, tot=tot, launches=launches, epp=epp, mode=mode, krp=krp, obs=obs, dev=dev,
                ev_cap=ev_cap, grid=g, version=g.version())


def run_e2e(args, r):
    """The same metric through the C ABI with HOST buffers.  The model is created once; every timed step hands the
    library a density (and field) snapshot in pinned host memory -- krp_grid_stage / krp_grid_update_staged, the
    pipelined form of krp_grid_update(KRP_MEM_HOST): one full host-to-device copy per step inside the timed region,
    overlapped with the kernels of the step before the one that uses it -- transports and images one batch, and reads
    the maps back to pinned host memory (krp_image_get with KRP_MEM_HOST), whose total the host then takes."""
    import torch
    krp, cfg, batch, obs, dev = r["krp"], r["cfg"], r["batch"], r["obs"], r["dev"]
    rank, world = r["rank"], r["world"]
    from paper_2512_01283_b200 import shard
    n_obs, npix, seed = len(obs), cfg["npix"], cfg["seed"]
    pin = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a, np.float32)).pin_memory()
    h_dens, h_bf = pin(cfg["density"]), pin(cfg["bfield"])
    w_host = cfg["source"].get("cell_weight")
    weight = None if w_host is None else torch.from_numpy(np.ascontiguousarray(w_host, np.float32).ravel()).to(dev)
    h_img = torch.zeros((n_obs, 4, npix, npix), dtype=torch.float64).pin_memory()
    h2d = h_dens.numel() * 4 + (0 if h_bf is None else h_bf.numel() * 4)
    d2h = h_img.numel() * 8
    g = make_grid(krp, cfg, h_dens.numpy(), None if h_bf is None else h_bf.numpy(), weight)
    g.events_reserve(r["ev_cap"])

    copy_stream = torch.cuda.Stream(device=dev)
    hb = None if h_bf is None else h_bf.numpy()

    def one(i):
        first, cnt = shard.step_id_range(1000 + i, rank, world, batch)
        # This step's snapshot: its H2D copy was started during the step before (krp_grid_stage on a copy stream), so it ran
        # under that step's kernels; here the cells are re-packed from it.  The copy of the NEXT step's snapshot starts at once
        # and runs under this step's transport and imaging -- every step, the last one included, issues one full copy.
        g.update_staged()
        g.stage(h_dens.numpy(), hb, copy_stream=copy_stream)
        g.packet_id_set(first)
        g.image_reset()
        g.transport(cnt, seed)
        g.image(obs, npix, npix)
        g.image_get(out=h_img.numpy())                 # D2H, synchronises
        return float(h_img[:, 0].sum())                # the step's result, read on the host

    k = max(1, args.steps)
    g.stage(h_dens.numpy(), hb, copy_stream=copy_stream)
    one(0)
    torch.cuda.synchronize()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    t0 = time.perf_counter()
    for i in range(k):
        one(1 + i)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([dt], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dt = float(t.item())
    g.close()
    return {"value": k * batch * world / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
            "steps": k, "ms_per_step": 1e3 * dt / k,
            "path": "per step: krp_grid_update_staged (cells re-packed from the snapshot whose H2D copy ran under the step before) + "
                    "krp_grid_stage (pinned; the next snapshot's copy, on a copy stream) + krp_transport + krp_image + "
                    "krp_image_get(KRP_MEM_HOST, pinned)"}


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    r = run_krp(args)
    r["grid"].close()
    e2e = None if (args.no_e2e or args.form == "twostep") else run_e2e(args, r)
    if r["world"] > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if r["rank"] != 0:
        return 0
    cfg, tot = r["cfg"], r["tot"]
    cpu = None
    if r["world"] == 1 and not args.no_cpu_baseline:
        cpu = oracle_timed(cfg, args.cpu_seconds)
    sec = r["ms_total"] * 1e-3
    line = {
        "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": r["world"], "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": r["ms_total"] / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": ("f32 march with f64 optical depth, f64 image sums" if r["mode"] == "scalar"
                  else "f64 flights (event location), f32 imaging march, f64 image sums"), "data": "synthetic",
        "config": {"workload": cfg["name"], "grid": [cfg["nx"], cfg["ny"], cfg["nz"]], "packets_per_step_per_gpu": r["batch"],
                   "observers": len(cfg["observers"]), "npix": cfg["npix"], "cell_layout": r["mode"], "form": args.form,
                   "job_packets": cfg["n_packets"], "events_per_packet": r["epp"],
                   "l2": "flushed every step by a 256 MiB memset inside the timed region",
                   "launch": "flights: %s; imaging: one launch per observer over events ordered by cell bin" %
                             (("one kernel per batch, a lane follows a packet to its end (krp_k_packets_scalar)"
                               if r["roof"].get("kernels", {}).get("flight", {}).get("launches_per_step", 2) <= 1 else "static assignment, one launch per scattering order")
                              if r["mode"] == "scalar" else "persistent lanes, refill distance chosen from the measured flight length"),
                   "parallelism": "packet ids sharded over %d GPU(s), grid replicated, one fp64 image all-reduce at job end" % r["world"],
                   "reduced": bool(args.n)},
        "scatterings_per_s": tot["events"] / sec,
        "cell_steps_per_s": (tot["steps_transport"] + tot["steps_image"]) / sec,
        "kernel_ms": {"transport": r["t_tr"], "image": r["t_im"]},
        "clocks": r["clocks"], "roofline": r["roof"], "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(r["launches"]), "library": r["version"],
        "context": "paper: ~1.4e7 packets/s for its own (different) step 1 on an RTX 5090, ~1e2x over CPU codes (PAPER.md:125)",
    }
    print(json.dumps(line))
    return 0


if __name__ == "__main__":
    sys.exit(main())
