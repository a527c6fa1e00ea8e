#!/usr/bin/env python
"""bench.py -- throughput of the fp64 DG right-hand side fused into LSRK54 on one B200 (BASELINE.json metric).

A "step" is one LSRK54 time step of the whole hot path = 5 stages, each = auxiliary-gradient kernel +
fused tendency/low-storage-update kernel (rows a1-a5 of the scope table), on BASELINE config 5:
96x96x48 hexahedra at N=4, 6 prognostics, ~55.3 M nodes, moist Smagorinsky-Lilly, synthetic seeded state.
value = nodes * 5 * K / time  [DOF-stages/s], whole job (all ranks).  The state (2.65 GB/copy) is far larger
than the 126 MB L2, so no explicit L2 flush is needed between iterations.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--ne EX EY EZ] [--order N]

N > 1 (torchrun): the path does not shard in this build ("replicas only"): each rank runs an independent
replica on its own GPU, the timed region is bracketed by barriers and the max over ranks is taken.
--impl reference: the CPU oracle (oracle/), as it stands, on the host cores of rank 0, on a bounded cut of
the same workload (this tier's reference arm).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 DG RHS throughput (DOF-stages/s) at N=4; % of B200 HBM roofline"
UNIT = "DOF-stages/s"
# algorithmic bytes per node: each array once per sweep, fp64
B_GRAD = {5: (5 + 9) * 8, 6: (6 + 12) * 8}                  # sweep A: read Q, write packed SGS fluxes
B_TEND = {5: (5 + 9 + 5 + 5 + 5) * 8, 6: (6 + 12 + 6 + 6 + 6) * 8}   # sweep B: read Q, G, dQ; write dQ, Q
B_TEND_STAGE1 = {5: (5 + 9 + 5 + 5) * 8, 6: (6 + 12 + 6 + 6) * 8}    # stage 1 (A_1 = 0) does not read dQ


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def kernel_source_hash():
    """sha256 over the CUDA sources: ties a recorded ncu figure to the kernels it was captured on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2110_00853_b200", "csrc")
    for f in sorted(os.listdir(d)):
        with open(os.path.join(d, f), "rb") as fh:
            h.update(f.encode()); h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(order, ne):
    """dram bytes per launch of the dominant kernel from the committed ncu capture -- only if that capture was taken on
    the kernels of this tree (source hash) and on this workload; otherwise None."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        t = json.load(f)
    if t.get("source_hash") != kernel_source_hash() or t.get("order") != order or list(t.get("ne", [])) != list(ne):
        return None
    return t.get("tendency_dram_bytes_per_launch")


def record_traffic(args):
    """--record-traffic RAW.csv: reads dram__bytes_read.sum + dram__bytes_write.sum of the tendency kernel from an
    `ncu -i <rep> --page raw --csv` export and stores them with the source hash and the workload."""
    import csv
    rows = list(csv.reader(open(args.record_traffic)))
    hdr, units = rows[0], rows[1]
    best = None
    for r in rows[2:]:
        d = dict(zip(hdr, r))
        if "tendency" not in d.get("Kernel Name", ""):
            continue
        tot = 0.0
        for k in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            u = units[hdr.index(k)]
            tot += float(d[k]) * {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[u]
        best = (d["Kernel Name"], tot)
    assert best, "no tendency kernel in " + args.record_traffic
    out = {"tendency_dram_bytes_per_launch": best[1], "kernel": best[0], "source_hash": kernel_source_hash(),
           "order": args.order, "ne": list(args.ne), "source": os.path.basename(args.record_traffic)}
    with open(os.path.join(ROOT, "profiles", "traffic.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out))


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index; self.rows = []; self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True); self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def cut_of_config5(ne, order):
    """Config 5 with the full 3 km column and the same element size, on an Ex x Ey x Ez brick."""
    import workloads as W
    full = W.SWEEP5[order]
    hi = (6000.0 * ne[0] / full[0], 6000.0 * ne[1] / full[1], 3000.0 * ne[2] / full[2])
    return W.config5(ne=tuple(ne), N=order, hi=hi)


def time_oracle(sample_ne, order, steps, warmup=0):
    """Times the CPU oracle (kind "oracle") on a cut of config 5; returns (DOF-stages/s, threads, description, s/step)."""
    from oracle import oracle as om
    cfg, Q, dt = cut_of_config5(sample_ne, order)
    o = om.Oracle(cfg)
    nodes = Q.shape[0] * Q.shape[1]
    Qc = Q.copy(); dU = np.zeros_like(Q)
    for _ in range(warmup):
        for s in range(5):
            o.lsrk54_stage(Qc, dU, dt, s)
    t0 = time.perf_counter()
    for _ in range(steps):
        for s in range(5):
            o.lsrk54_stage(Qc, dU, dt, s)
    el = time.perf_counter() - t0
    desc = "config 5 cut %dx%dx%d elements at N=%d (%d nodes, full 3 km column), %d LSRK54 steps" % (*sample_ne, order, nodes, steps)
    return nodes * 5 * steps / el, om.num_threads(), desc, el / steps


def cpu_info():
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip(); break
    except OSError:
        pass
    return model, os.cpu_count()


def set_oracle_threads(n):
    """OpenMP thread count of the oracle library (libgomp's own entry point; the oracle is not modified for timing)."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def time_oracle_stage(cfg, Q, dt, reps=3):
    """Best of `reps` of ONE LSRK54 stage (gradient + RHS + update) of the oracle on the given config."""
    from oracle import oracle as om
    o = om.Oracle(cfg)
    Qc = Q.copy(); dU = np.zeros_like(Q)
    best = 1e300
    for _ in range(reps):
        t0 = time.perf_counter(); o.lsrk54_stage(Qc, dU, dt, 0); best = min(best, time.perf_counter() - t0)
    nodes = Q.shape[0] * Q.shape[1]
    return {"nodes": nodes, "ms_per_stage": 1e3 * best, "node_stages_per_s": nodes / best}


def cpu_baseline(order, full_ne, ne):
    """the oracle as it stands on the host cores -- all cores and one thread on cuts of config 5
    (full 3 km column), one stage of each of configs 1-4 at their stated sizes; CPU model, nproc and thread counts printed."""
    import workloads as W
    from oracle import oracle as om
    model, nproc = cpu_info()
    sample = (full_ne[0] // 4, full_ne[1] // 4, full_ne[2]) if tuple(ne) == tuple(full_ne) else tuple(ne)
    val, threads, desc, _ = time_oracle(sample, order, 3)
    out = {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc, "cpu_model": model, "nproc": nproc}
    small = (max(1, sample[0] // 3), max(1, sample[1] // 3), sample[2])
    if set_oracle_threads(1):
        v1, t1, d1, _ = time_oracle(small, order, 1)
        out["single_thread"] = {"value": v1, "unit": UNIT, "cores": t1, "sample": d1}
        set_oracle_threads(threads)
    per_cfg = {}
    for k in (1, 2, 3, 4):
        cfg, Q, dt = W.CONFIGS[k]()
        per_cfg["config%d" % k] = time_oracle_stage(cfg, Q, dt)
    out["one_stage_all_cores"] = per_cfg
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads as W
    full = W.SWEEP5[args.order]
    sample = (full[0] // 4, full[1] // 4, full[2])          # 1/16 of the columns, full 3 km height
    val, threads, desc, s_per_step = time_oracle(sample, args.order, args.steps, args.warmup)
    model, nproc = cpu_info()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * s_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, sample_note="each step = one LSRK54 step on the bounded sample: " + desc),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
                             "cpu_model": model, "nproc": nproc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# algorithmic bytes per node and LSRK stage of the extra legs (stage 1 of a step does not read the residual)
def stage_bytes(nvar, sgs, warped25):
    ngrad = {5: 9, 6: 12}[nvar]
    grad = (nvar + ngrad) * 8 if sgs else 0
    tend = (nvar + (ngrad if sgs else 0) + nvar + nvar + nvar) * 8 - nvar * 8 / 5.0
    geo = (2 + 2 + 2 + 1) * 8 if warped25 else 0          # z_xi, z_zeta per sweep, rho_r, rhoe_r, nodal z (SURVEY: 200 B for config 4)
    if warped25 and not sgs:
        geo = (2 + 2 + 1) * 8
    return grad + tend + geo


def bench_leg(P, torch, cfg, Q, dt, steps, peak, label, bytes_per_node_stage, tuning=None):
    """K LSRK54 steps of one further workload on the library stream, CUDA events; returns a small report dict."""
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        g = P.CmDg(cfg, stream=stream, tuning=tuning)
        Qd = torch.from_numpy(g.pack(Q)).to(g.device, non_blocking=False)
    stream.synchronize()
    nodes = g.n_elem * g.np
    for _ in range(3):                                   # call 2 captures the step as a CUDA graph, call 3 replays it
        g.lsrk_step(Qd, dt, 1)
    stream.synchronize()
    # pass 1: the shipped default (graph replay, no per-launch events) -> value / ms_per_step
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        g.lsrk_step(Qd, dt, 1)
    e1.record(stream); stream.synchronize()
    ms = e0.elapsed_time(e1)
    # pass 2: instrumented (events around every launch, which also switches the graph off): per-kernel times and the
    # plain-launch step time the graph is compared with
    ksteps = max(1, min(steps, 5))
    g.profile_begin()
    p0 = torch.cuda.Event(enable_timing=True); p1 = torch.cuda.Event(enable_timing=True)
    p0.record(stream)
    for _ in range(ksteps):
        g.lsrk_step(Qd, dt, 1)
    p1.record(stream); stream.synchronize()
    ks = g.profile_end()
    ms_plain = p0.elapsed_time(p1) / ksteps
    d = g.diagnostics(Qd)
    gbs = nodes * bytes_per_node_stage * 5 * steps / (ms * 1e-3) / 1e9
    out = {"workload": label, "nodes": nodes, "order": int(cfg["N"]), "steps": steps, "value": nodes * 5 * steps / (ms * 1e-3),
           "unit": UNIT, "ms_per_step": ms / steps, "ms_per_step_no_graph_instrumented": ms_plain,
           "ms_tendency": ks["ms_tendency"] / max(1, ks["launches_tendency"]),
           "ms_gradient": ks["ms_gradient"] / max(1, ks["launches_gradient"]),
           "algorithmic_bytes_per_node_stage": bytes_per_node_stage, "achieved_gbs": gbs, "frac_of_measured_hbm": gbs / peak,
           "n_nonfinite": d["n_nonfinite"]}
    g.close(); del Qd
    torch.cuda.empty_cache()
    return out


LEGS = {
    "c2": (lambda W: W.config2(), 50, "config 2 (density current, dry, closure on, flat) 40x1x20", (5, 1, False)),
    "c3": (lambda W: W.config3(), 20, "config 3 (dry CBL, SL, flat) 32x32x16", (5, 1, False)),
    "c3x": (lambda W: W.config3(ne=(96, 96, 48), hi=(19200.0, 19200.0, 9000.0)), 5, "config 3 scaled to 96x96x48 elements", (5, 1, False)),
    "c4": (lambda W: W.config4(), 20, "config 4 (mountain, inviscid, stored metrics) 120x1x30", (5, 0, True)),
    "c4x": (lambda W: W.config4(ne=(120, 96, 30)), 5, "config 4 extruded to 120x96x30 elements", (5, 0, True)),
    "c4s": (lambda W: W.config4(ne=(120, 96, 30), sgs=1), 5, "config 4 extruded to 120x96x30 elements, with the Smagorinsky-Lilly closure", (5, 1, True)),
}


def _next_leg(**over):
    """Config 5 on a 48x48x48 cut (13.8 M nodes, state 0.66 GB per copy: still far larger than L2) with one of the further
    options switched on: the throughput of the scope table's NEXT rows."""
    def make(W):
        if not _C5CUT_CACHE:
            _C5CUT_CACHE.append(W.config5(ne=(48, 48, 48), N=4, hi=(3000.0, 3000.0, 3000.0)))   # the same seeded state for every leg
        cfg, Q, dt = _C5CUT_CACHE[0]
        return dict(cfg, **over), Q, dt
    return make


_C5CUT_CACHE = []


_C5CUT = "config 5 cut 48x48x48, N=4, "
LEGS.update({
    "c5_vreman": (_next_leg(sgs=2, richardson=1), 3, _C5CUT + "Vreman closure + Richardson factor (NEXT-1)", (6, 1, False)),
    "c5_sponge_filter": (_next_leg(sponge_alpha=0.4, sponge_zs=2400.0, filter_order=64), 3, _C5CUT + "Rayleigh sponge + exponential filter after every step (NEXT-2)", (6, 1, False)),
    "c5_hllc": (_next_leg(riemann=1), 3, _C5CUT + "HLLC flux (NEXT-3; thread-per-node kernels)", (6, 1, False)),
    "c5_roe": (_next_leg(riemann=2), 3, _C5CUT + "Roe flux (NEXT-3; thread-per-node kernels)", (6, 1, False)),
    "c5_satadj": (_next_leg(satadj=1), 3, _C5CUT + "saturation-adjusted equation of state (NEXT-4; thread-per-node kernels)", (6, 1, False)),
    "c5_surface": (_next_leg(drag_cd=1.3e-3, lhf_bottom=147.2, evap_bottom=5.9e-5), 3, _C5CUT + "drag law + LHF + evaporation at the bottom wall (NEXT-4)", (6, 1, False)),
})
NEXT_LEGS = ("c5_vreman", "c5_sponge_filter", "c5_hllc", "c5_roe", "c5_satadj", "c5_surface")


def one_leg(P, torch, name, peak, tuning=None):
    """One of the further workloads by name (also `bench.py --leg NAME`, the command the ncu captures of the stored-metric
    kernels run).  For the stored-metric legs the bytes those kernels really move are reported beside the algorithmic
    ones: on a terrain-following mesh the tendency kernel reads 6 geometry fields (Ja^1_x, Ja^3_x, Ja^3_y, 1/J, z, tau_s) and
    2 reference fields per node where the 2.5-D-specialised count of SURVEY 8(d) has 5 values."""
    import workloads as W
    make, steps, label, sb = LEGS[name]
    cfg, Q, dt = make(W)
    out = bench_leg(P, torch, cfg, Q, dt, steps, peak, label, stage_bytes(*sb), tuning)
    out["leg"] = name
    if tuning:
        out["tuning"] = tuning
    if sb[2] and not tuning:
        moved = (5 + 5 + 5 + 5 - 1.0) * 8 + (6 + 2) * 8           # Q, residual (4 of 5 stages), residual out, Q out + geometry + reference
        if sb[1]:
            moved += (5 + 15 + 9) * 8 + 9 * 8                     # gradient sweep: Q, 15 geometry fields, G out; G read by the tendency
        out["moved_bytes_per_node_stage"] = moved
        out["moved_gbs"] = out["achieved_gbs"] * moved / out["algorithmic_bytes_per_node_stage"]
        out["moved_frac_of_measured_hbm"] = out["moved_gbs"] / peak
    return out


def extra_legs(P, torch, args, peak):
    """Order sweep of config 5 at ~55 M nodes (N = 3, 5, 6), dry config 3 and terrain config 4 (BASELINE size and a
    y-extruded variant that fills the GPU): throughput and whole-stage roofline fraction of each."""
    import workloads as W
    out = {"sweep": [], "configs": []}
    for N in (3, 5, 6):
        if N == args.order:
            continue
        ne = W.SWEEP5[N]
        cfg, Q, dt = W.config5(ne=ne, N=N, hi=(6000.0, 6000.0, 3000.0))
        out["sweep"].append(bench_leg(P, torch, cfg, Q, dt, 3, peak, "config 5 at N=%d, %dx%dx%d" % ((N,) + tuple(ne)), stage_bytes(6, 1, False)))
        del cfg, Q
    for name in ("c2", "c3", "c3x", "c4", "c4x", "c4s"):
        out["configs"].append(one_leg(P, torch, name, peak))
    out["next_rows"] = [one_leg(P, torch, name, peak) for name in NEXT_LEGS]
    return out


def workload_config(args, sample_note=None):
    ne = args.ne
    c = {"workload": "BASELINE config 5: moist shallow-cumulus-shaped box, %dx%dx%d hexahedra, N=%d, 6 fp64 prognostics, "
                     "Smagorinsky-Lilly, periodic x/y, no-flux z" % (ne[0], ne[1], ne[2], args.order),
         "elements": int(np.prod(ne)), "nodes": int(np.prod(ne)) * (args.order + 1) ** 3, "order": args.order, "nvar": 6,
         "step": "one LSRK54 step = 5 x (gradient kernel + fused tendency/update kernel)",
         "l2": "inputs larger than L2 (state 2.65 GB per copy vs 126 MB L2), no flush needed",
         "parallelism": "replicas only (one independent replica per GPU)"}
    if sample_note:
        c["sample"] = sample_note
    return c


def max_over_ranks(x, dist, device):
    """MAX of a scalar over the ranks of the default process group (identity when dist is None)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(nodes_per_rank, steps, ms_local, world, dist, device):
    """DOF-stages/s of the whole job: every rank advances its own replica (weak scaling, no data-path collective), the
    time is the max over ranks.  Returns (value, ms)."""
    ms = max_over_ranks(ms_local, dist, device)
    return world * nodes_per_rank * 5 * steps / (ms * 1e-3), ms


def run_ours(args):
    import torch
    import workloads as W
    import paper_2110_00853_b200 as P

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    t_gen = time.perf_counter()
    cfg, Q, dt = cut_of_config5(args.ne, args.order)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        g = P.CmDg(cfg, stream=stream, tuning=args.tuning)
        Qh = torch.from_numpy(g.pack(Q)).pin_memory()
        del Q
        Qd = Qh.to(g.device, non_blocking=True)
    stream.synchronize()
    t_gen = time.perf_counter() - t_gen
    nodes = g.n_elem * g.np
    nv = g.nvar
    K, Wm = args.steps, args.warmup

    # ---- device-resident throughput: K LSRK54 steps, CUDA events on the library stream
    d0 = g.diagnostics(Qd)
    for _ in range(Wm):
        g.lsrk_step(Qd, dt, 1)
    stream.synchronize()
    sampler = ClockSampler(local); sampler.start()
    time.sleep(0.3)
    ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
    barrier()
    # timed region: the shipped default path (after the warm-up the step is replayed from its CUDA graph; no per-launch events)
    ev0.record(stream)
    for _ in range(K):
        g.lsrk_step(Qd, dt, 1)
    ev1.record(stream)
    stream.synchronize()
    barrier()
    clocks = sampler.stop()
    value, ms = whole_job_value(nodes, K, ev0.elapsed_time(ev1), world, dist, g.device)
    # second, separate pass with CUDA events around every launch (plain launches): per-kernel times for the roofline
    Kp = max(1, min(K, 5))
    g.profile_begin()
    pv0 = torch.cuda.Event(enable_timing=True); pv1 = torch.cuda.Event(enable_timing=True)
    pv0.record(stream)
    for _ in range(Kp):
        g.lsrk_step(Qd, dt, 1)
    pv1.record(stream); stream.synchronize()
    ks = g.profile_end()
    ms_plain = pv0.elapsed_time(pv1) / Kp
    launches_per_step = (ks["launches_gradient"] + ks["launches_tendency"] + ks["launches_other"]) // Kp
    d1 = g.diagnostics(Qd)

    # ---- RHS alone (cm_dg_rhs), same state
    with torch.cuda.stream(stream):                  # allocate (and zero-fill) on the stream the library writes on
        dQ = g.empty(nv)
    for _ in range(3):
        g.rhs(Qd, dQ)
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    stream.synchronize(); e0.record(stream)
    nrhs = max(5, K)
    for _ in range(nrhs):
        g.rhs(Qd, dQ)
    e1.record(stream); stream.synchronize()
    rhs_ms = e0.elapsed_time(e1) / nrhs
    del dQ

    # ---- end to end through the host-buffer C-ABI call: H2D + step + D2H inside the timed region
    Ke = max(1, min(K, args.e2e_steps))
    g.lsrk_step_host(Qh, dt, 1)                      # warm-up (allocates the staging buffer)
    barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        g.lsrk_step_host(Qh, dt, 1)                  # synchronises the stream itself
    barrier()
    e2e_val, e2e_ms = whole_job_value(nodes, Ke, 1e3 * (time.perf_counter() - t0), world, dist, g.device)
    state_bytes = nv * g.stride * 8

    # ---- roofline of the dominant kernel (fused tendency + LSRK update), measured live with CUDA events
    peak, peak_src = measured_peaks()
    n_t = max(1, ks["launches_tendency"]); n_g = max(1, ks["launches_gradient"])
    t_tend = ks["ms_tendency"] / n_t; t_grad = ks["ms_gradient"] / n_g
    bytes_tend = nodes * (4 * B_TEND[nv] + B_TEND_STAGE1[nv]) / 5.0
    ach = bytes_tend / (t_tend * 1e-3) / 1e9
    stage_bytes = nodes * (B_GRAD[nv] + (4 * B_TEND[nv] + B_TEND_STAGE1[nv]) / 5.0)
    stage_gbs = stage_bytes * 5 * K / (ms * 1e-3) / 1e9
    if int(cfg.get("geom", 0)) == 0 and not args.tuning:
        kname = "cm10_tendency_kernel<Nq=%d,MOIST=%d,SGS=%d,MODE=1> (row sweep: fused tendency + LSRK update)" % (args.order + 1, int(nv == 6), int(cfg.get("sgs", 0) != 0))
        if args.order + 1 >= 7:
            kname = "cm7_tendency_kernel<Nq=%d,...> (CTA per element: fused tendency + LSRK update)" % (args.order + 1)
    else:
        kname = "tendency kernel selected by --tuning %r" % (args.tuning,)
    roof = {"bound": "hbm", "kernel": kname, "achieved": ach, "peak": peak,
            "unit": "GB/s", "frac": ach / peak, "traffic": ncu_traffic(args.order, args.ne), "peak_source": peak_src,
            "algorithmic_bytes_per_launch": bytes_tend, "ms_per_launch": t_tend,
            "share_of_step": ks["ms_tendency"] / (ks["ms_tendency"] + ks["ms_gradient"] + ks["ms_other"]),
            "gradient_kernel": {"achieved": nodes * B_GRAD[nv] / (t_grad * 1e-3) / 1e9, "ms_per_launch": t_grad,
                                "algorithmic_bytes_per_launch": nodes * B_GRAD[nv]},
            "whole_stage": {"achieved": stage_gbs, "frac": stage_gbs / peak, "frac_of_8TBs_nominal": stage_gbs / 8000.0,
                            "algorithmic_bytes_per_node_stage": stage_bytes / nodes},
            "rhs_only": {"ms": rhs_ms, "dof_per_s": nodes / (rhs_ms * 1e-3),
                         "achieved": nodes * (B_GRAD[nv] + B_TEND[nv] - nv * 16) / (rhs_ms * 1e-3) / 1e9}}
    roof["rhs_only"]["frac"] = roof["rhs_only"]["achieved"] / peak
    # the same figures as flat scalars (a consumer that keeps only the top level of `roofline` still sees them)
    roof.update({"rhs_only_ms": rhs_ms, "rhs_only_frac": roof["rhs_only"]["frac"],
                 "rhs_only_frac_of_8TBs": roof["rhs_only"]["achieved"] / 8000.0,
                 "whole_stage_frac": stage_gbs / peak, "gradient_ms": t_grad,
                 "gradient_frac": roof["gradient_kernel"]["achieved"] / peak,
                 "ms_per_step_no_graph_instrumented": ms_plain})

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(args),
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes,
                    "steps": Ke, "call": "cm_dg_lsrk_step_host (pinned host buffer)"},
            "gpu_launches": int(launches_per_step * K),   # kernels of the timed K steps (counted per step on the instrumented pass)
            "clocks": clocks, "roofline": roof,
            "conservation": {"rel_mass_change": (d1["mass"] - d0["mass"]) / d0["mass"],
                             "rel_energy_change": (d1["energy"] - d0["energy"]) / d0["energy"],
                             "n_nonfinite": d1["n_nonfinite"]},
            "setup_s": t_gen}
    if rank == 0 and world == 1 and not args.no_extra:
        g.close(); del Qd, Qh
        torch.cuda.empty_cache()
        line["extra"] = extra_legs(P, torch, args, peak)
        for leg in line["extra"]["sweep"]:
            roof["sweep_N%d_frac" % leg["order"]] = leg["frac_of_measured_hbm"]
        for leg in line["extra"]["next_rows"]:
            roof["%s_gdofs" % leg["leg"]] = leg["value"] / 1e9
        for leg in line["extra"]["configs"]:
            if leg.get("leg") in ("c2", "c3", "c4"):     # launch-bound meshes: graph replay against plain launches
                roof["%s_ms_per_step_graph" % leg["leg"]] = leg["ms_per_step"]
                roof["%s_ms_per_step_no_graph" % leg["leg"]] = leg["ms_per_step_no_graph_instrumented"]
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.order, W.SWEEP5[args.order], args.ne)
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--order", type=int, default=4, help="polynomial order N (config-5 sweep: 3..6)")
    ap.add_argument("--ne", type=int, nargs=3, default=None, help="element counts (default: the full config-5 mesh)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--record-traffic", default=None, metavar="RAW.csv",
                    help="store the tendency kernel's ncu DRAM bytes (ncu --page raw --csv export) in profiles/traffic.json")
    ap.add_argument("--no-extra", action="store_true", help="skip the extra legs (order sweep, configs 3 and 4)")
    ap.add_argument("--leg", default=None, choices=sorted(LEGS), help="run ONE of the further workloads and print its report")
    ap.add_argument("--tuning", nargs="*", default=None, metavar="KEY=VAL",
                    help="cm_dg_tuning fields for kernel experiments (e.g. kernel=7 row_len=16); default: the library's defaults")
    args = ap.parse_args()
    if args.tuning is not None:
        args.tuning = {kv.split("=")[0]: int(kv.split("=")[1]) for kv in args.tuning} or None
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    import workloads as W
    if args.ne is None:
        args.ne = list(W.SWEEP5[args.order])
    if args.record_traffic:
        record_traffic(args)
    elif args.leg:
        import torch
        import paper_2110_00853_b200 as P
        print(json.dumps(one_leg(P, torch, args.leg, measured_peaks()[0], args.tuning)))
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
