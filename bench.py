#!/usr/bin/env python
"""bench.py — zone-cycles/s of the full RK2 step (the whole hot path) on the headline workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference] [--graph 0|1]

One JSON line on stdout (rank 0).  Workload: BASELINE.json configs[3] = C4, the 256^3 MKS Fishbone-Moncrief
torus, PPM + LLF, fp64 (seeded synthetic stand-in for the paper's initial data).
N > 1 (torchrun): the path does not shard in this build ("replicas only"): every rank steps its own
copy, no data-path collective; value = N x zones x K / max-over-ranks time.

--impl reference: the CPU oracle as it stands, on the host cores, on a bounded sample of the same workload.
"""
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

METRIC = "zone-cycles/s per full RK2 step at 256^3 fp64 (1 B200); % of HBM roofline"
UNIT = "zone-cycles/s"
B_ALG = 1218.0          # algorithmic bytes per zone-cycle
# algorithmic bytes per zone and launch of each kernel class (SURVEY 8(d) accounting): flux: read P 64, write 7
# components 56; emf (generic path only): read 6 induction fluxes 48, write 3 EMFs 24; update (the fused kernel evaluates
# eq. 21 in place, so it reads the six induction-flux components instead of three EMFs): P^n 64 + hydro fluxes 5 x 3 x 8 =
# 120 + induction fluxes 6 x 8 = 48 + P-half 64 in the corrector only (mean of the two launches: 32) in, P 64 + flag 1 out
# = 64 + 120 + 48 + 32 + 65 = 329
KERNEL_BYTES = {"flux1": 120.0, "flux2": 120.0, "flux3": 120.0, "emf": 72.0, "update": 329.0}
# ncu --set full counters of this command at C4, per launch and averaged over the predictor and corrector launches
# (DRAM bytes read + written; fp64 DFMA/DMUL/DADD/DSETP warp instructions executed), are READ from the committed
# summary of the capture, never typed in here.  Only quoted for the workload they were captured on.
NCU_FILE = os.path.join(ROOT, "profiles", "ncu_c4_counters.json")


def ncu_counters():
    try:
        d = json.load(open(NCU_FILE))
        return d["kernels"], d.get("source", os.path.relpath(NCU_FILE, ROOT))
    except Exception:
        return {}, None


# fp64 pipe: 16 lanes per SM sub-partition = one warp instruction per 2 cycles per sub-partition
FP64_WARP_INST_PER_S = 148 * 4 * 1.965e9 / 2.0


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", d
    return 6650.0, "fallback (B200_PROFILING.md)", {}


class ClockSampler:
    """nvidia-smi clocks / power / throttle reasons sampled every 20 ms from before the warm-up until after the last
    timed region; every row carries its arrival time, so each timed region is summarised over its own window (a
    0.1 s region still sees the rows that arrived while it ran, plus the nearest one on either side)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def stop(self):
        if self.proc:
            self.proc.terminate()
            self.t.join(timeout=2)

    def window(self, t0, t1):
        """Summary of the rows that arrived in [t0, t1] (wall clock of this process), widened to the nearest row on
        either side when fewer than 3 fall inside."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        rows = [r for (t, r) in self.rows if t0 <= t <= t1]
        if len(rows) < 3:
            before = [r for (t, r) in self.rows if t < t0][-1:]
            after = [r for (t, r) in self.rows if t > t1][:1]
            rows = before + rows + after
        sm, mx, pw, reasons = [], [], [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for n, v in zip(self.NAMES, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "sm_min_mhz": sm[0] if sm else None, "power_w_max": max(pw) if pw else None,
                "reasons": sorted(reasons), "samples": len(sm), "window_s": round(t1 - t0, 3)}


def aggregate(ms_local, zones, steps, world, dist=None, device="cpu"):
    """Whole-job throughput of `world` independent replicas (the path does not shard in this build):
    max over ranks of the device-timed region, value = world x zones x steps / that time.  No data-path collective;
    this all-reduce of one scalar is the only exchange."""
    ms = float(ms_local)
    if dist is not None and world > 1:
        import torch
        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms, world * zones * steps / (ms * 1e-3)


def make_workload(name, **kw):
    from workloads import config
    from workloads.params import TORUS
    from workloads.torus import fm_torus
    p = config(name, **kw)
    prim, info = fm_torus(p, **TORUS[name])
    return p, prim


def oracle_sample(name, steps, n3_sample=None, threads=None, prebuilt=None):
    """The oracle as it stands on the `name` torus (n3_sample: a phi-slab of n3_sample zones of the same (r, theta)
    grid and scheme; None: the full grid; prebuilt = (params, host array) of that workload, stepped in place):
    (zone-cycles/s, threads used, description, seconds)."""
    import oracle
    kw = {} if n3_sample is None else {"n3": n3_sample}
    p, prim = prebuilt if prebuilt is not None else make_workload(name, **kw)
    oracle.set_threads(threads if threads else (os.cpu_count() or 1))
    g = oracle.Grid(p)
    g.bind(prim)
    dt = g.cfl_dt(0.45)
    t0 = time.perf_counter()
    for _ in range(steps):
        g.step(dt)
    sec = time.perf_counter() - t0
    zones = p["n1"] * p["n2"] * p["n3"]
    what = "full grid" if n3_sample is None else f"phi-slab of the {name} grid"
    used = oracle.get_threads()
    g.close()
    return zones * steps / sec, used, f"{name} torus, {p['n1']}x{p['n2']}x{p['n3']} ({what}), {steps} RK2 steps", sec


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    per_step = []
    p = None
    import oracle
    if args.threads:
        oracle.set_threads(args.threads)
    p, prim = make_workload(args.config, n3=args.ref_n3)
    g = oracle.Grid(p)
    g.bind(prim)
    dt = g.cfl_dt(0.45)
    zones = p["n1"] * p["n2"] * p["n3"]
    for _ in range(args.warmup):
        g.step(dt)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        g.step(dt)
    sec = time.perf_counter() - t0
    val = zones * args.steps / sec
    sample = f"{args.config} torus, {p['n1']}x{p['n2']}x{p['n3']} phi-slab of the {args.config} grid per step"
    out = {"metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * sec / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "impl": "reference",
           "config": {"workload": f"{args.config}: {sample} (CPU oracle, bounded sample)", "recon": p["recon"], "riemann": p["riemann"]},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.get_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def run_ours(args):
    import numpy as np
    import torch
    import paper_2205_02484_b200 as cu

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU path)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    p, prim_host = make_workload(args.config)
    zones = p["n1"] * p["n2"] * p["n3"]
    prim_pinned = torch.from_numpy(prim_host).pin_memory()
    s = cu.Solver(p, prim_pinned, device=f"cuda:{local}")
    dt = s.cfl_dt(0.45)                                   # fixed dt chosen beforehand (eq. 26, xi = 0.45)
    if args.graph:
        s.use_graph(True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()                  # before the warm-up, so that rows exist when a 0.1 s region starts
    for _ in range(args.warmup):
        s.step(dt)
    barrier()

    # ---- timed regions: device-resident inputs, CUDA events on the library's stream (= torch's current stream) ----
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def one_step():
        if args.cfl_each_step:           # second protocol -- a new dt every step from eq. 26, taken on the
            s.step_cfl(0.45)             # device from the previous predictor's face speeds (same graph, no host sync)
        else:
            s.step(dt)

    def timed(n):
        """n steps between two events, barrier + synchronize on both sides: (max-over-ranks ms, zone-cycles/s of the whole
        job, clock summary of the window, launches)."""
        l0 = s.launch_count()
        barrier()
        w0 = time.perf_counter()
        e0.record()
        for _ in range(n):
            one_step()
        e1.record()
        barrier()
        w1 = time.perf_counter()
        ms_, val_ = aggregate(e0.elapsed_time(e1), zones, n, world, dist, "cuda")
        return ms_, val_, (sampler.window(w0, w1) if rank == 0 else None), s.launch_count() - l0

    # (1) burst: the first K steps after the W warm-up steps -- a fraction of a second, before the board has ramped to its
    # power cap.  Reported as `burst`; NOT the headline (the metric's workload is hundreds of steps: 500 at C4).
    if not args.graph:
        s.set_timing(True)
    ms_b, val_b, clk_b, _ = timed(args.steps)
    timing = s.get_timing() if not args.graph else {}
    s.set_timing(False)
    burst = {"steps": args.steps, "ms_per_step": ms_b / args.steps, "value": val_b, "unit": UNIT, "clocks": clk_b,
             "note": "first K steps after the warm-up, board not yet at its power cap"}

    # (2) sustained: after >= sustain_warm_s seconds of the same load, >= 300 steps (and >= sustain_s seconds) timed the
    # same way; clocks, power and throttle reasons over that window ride along.
    sustained = None
    if args.sustain_s > 0:
        est = ms_b / args.steps
        n_warm = max(1, int(args.sustain_warm_s * 1e3 / est))
        n_sus = max(300, int(args.sustain_s * 1e3 / est))
        barrier()
        for _ in range(n_warm):
            one_step()
        ms_s, val_s, clk_s, _ = timed(n_sus)
        sustained = {"steps": n_sus, "warm_steps": n_warm, "ms_per_step": ms_s / n_sus, "value": val_s, "unit": UNIT,
                     "seconds": ms_s * 1e-3, "clocks": clk_s,
                     "divb_norm": s.divb()[1], "failed_inversions": int(s.stats()[0])}

    # (3) headline: EXACTLY K steps, timed straight after the sustained leg, i.e. with the board in the state the metric's
    # own run (BASELINE.json: 500 steps at C4) spends nearly all of its time in.  With --sustain-s 0 this region follows
    # the burst directly (use --steps 500 --sustain-s 0 to time the config's own step count as one region).
    ms, value, clocks, launches = timed(args.steps)
    if args.graph:
        # per-kernel durations for the roofline objects: a short pass of the same steps launched kernel by kernel with
        # CUDA events around each launch (a graph replay has no place for them), after the headline region
        s.use_graph(False)
        s.set_timing(True)
        barrier()
        for _ in range(min(args.steps, 5)):
            s.step(dt)
        barrier()
        timing = s.get_timing()
        s.set_timing(False)
        s.use_graph(True)
    divb = s.divb()[1]
    stats = s.stats()

    # ---- e2e: the same step through the public API with HOST buffers: H2D of the primitives from pinned memory,
    # one step, D2H of the result into pinned memory, every step inside the timed region.  Three solver objects on three
    # streams take the steps in turn (each step is an independent problem: fresh input, own output), so the H2D copy of
    # one step overlaps the D2H copy and the kernels of the other (PCIe is full duplex; 1.15 GB each way per step).
    e2e_steps = max(2, min(args.e2e_steps, args.steps))
    NLANE = 3                            # H2D 22 ms + kernels 6 ms + D2H 22 ms per step: three steps in flight keep both copy
    lanes = [(s, torch.cuda.current_stream(), torch.empty_like(prim_pinned).pin_memory())]   # engines busy (PCIe is full duplex)
    for _ in range(NLANE - 1):
        side = torch.cuda.Stream(device=local)
        with torch.cuda.stream(side):
            sx = cu.Solver(p, prim_pinned, device=f"cuda:{local}", stream=side)
            if args.graph:
                sx.use_graph(True)
            sx.step(dt)                  # records its graph outside the timed region
        side.synchronize()
        lanes.append((sx, side, torch.empty_like(prim_pinned).pin_memory()))
    barrier()
    e0.record()
    for _, st, _ in lanes[1:]:
        st.wait_event(e0)
    for n in range(e2e_steps):
        sol, st, out_pinned = lanes[n % NLANE]
        with torch.cuda.stream(st):
            sol.load(prim_pinned)          # H2D + ghost fill
            sol.step(dt)
            out_pinned.copy_(sol.prim, non_blocking=True)
    for _, st, _ in lanes[1:]:
        ev = torch.cuda.Event()
        ev.record(st)
        torch.cuda.current_stream().wait_event(ev)
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)
    for sx, _, _ in lanes[1:]:
        sx.close()
    ms_e2e, e2e_val = aggregate(ms_e2e, zones, e2e_steps, world, dist, "cuda")
    # the same through ONE solver as a time-dependent run: step n+1 loads the host array step n wrote, so nothing overlaps
    # (H2D -> ghost fill -> step -> D2H, one after the other on one stream)
    ser_steps = max(2, min(6, e2e_steps))
    host_state = lanes[0][2]
    host_state.copy_(prim_pinned)
    barrier()
    e0.record()
    for n in range(ser_steps):
        s.load(host_state)
        s.step(dt)
        host_state.copy_(s.prim, non_blocking=True)
    e1.record()
    barrier()
    _, e2e_serial = aggregate(e0.elapsed_time(e1), zones, ser_steps, world, dist, "cuda")
    nbytes = prim_pinned.numel() * 8
    if rank == 0:
        sampler.stop()

    if rank == 0:
        peak, peak_src, pk = peaks()
        ncu_all, ncu_src = ncu_counters()
        # dominant kernel class by measured device time
        roof = None
        roof_alu = None
        shares = {}
        per_kernel = []      # every kernel class: algorithmic GB/s against the HBM peak, ncu DRAM bytes, fp64 pipe fraction
        if timing:
            tot = sum(v[0] for v in timing.values())
            shares = {k: round(v[0] / tot, 4) for k, v in timing.items() if v[1]}
            dom = max((k for k in KERNEL_BYTES if timing[k][1]), key=lambda k: timing[k][0])
            per_launch_ms = timing[dom][0] / timing[dom][1]
            achieved = KERNEL_BYTES[dom] * zones / (per_launch_ms * 1e-3) / 1e9
            ncu = ncu_all.get(dom) if (args.config == "C4" and world == 1) else None
            if ncu:
                a_alu = ncu["fp64_warp_inst"] / (per_launch_ms * 1e-3)
                roof_alu = {"bound": "alu", "kernel": dom, "achieved": a_alu, "peak": FP64_WARP_INST_PER_S,
                            "unit": "fp64 warp-instructions/s", "frac": a_alu / FP64_WARP_INST_PER_S,
                            "peak_source": "148 SMs x 4 sub-partitions x 1.965 GHz / 2 cycles per fp64 warp instruction",
                            "count_source": f"ncu, {ncu_src}"}
            for k in KERNEL_BYTES:
                if not timing[k][1]:
                    continue
                ms_k = timing[k][0] / timing[k][1]
                nk = ncu_all.get(k) if (args.config == "C4" and world == 1) else None
                gbs = KERNEL_BYTES[k] * zones / (ms_k * 1e-3) / 1e9
                per_kernel.append({
                    "kernel": k, "launches_per_step": 2, "algorithmic_bytes_per_zone": KERNEL_BYTES[k],
                    "ms_per_launch": ms_k, "achieved": gbs, "unit": "GB/s", "frac": gbs / peak,
                    "traffic": nk["traffic"] if nk else None,
                    "traffic_over_algorithmic": nk["traffic"] / (KERNEL_BYTES[k] * zones) if nk else None,
                    "dram_frac": nk["traffic"] / (ms_k * 1e-3) / 1e9 / peak if nk else None,
                    "fp64_frac": nk["fp64_warp_inst"] / (ms_k * 1e-3) / FP64_WARP_INST_PER_S if nk else None,
                    "time_share": shares.get(k)})
            roof = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": ncu["traffic"] if ncu else None,
                    "traffic_source": f"ncu --set full, {ncu_src}" if ncu else None, "peak_source": peak_src,
                    "kernel_ms_per_launch": per_launch_ms, "kernel_time_shares": shares,
                    "step_frac_of_hbm_roofline": value / world * B_ALG / (peak * 1e9),
                    "note": "achieved = algorithmic bytes of the dominant kernel class per launch / its mean "
                            "CUDA-event duration in the timed region; step_frac = zone-cycles/s x 1218 B / peak"}
        else:
            roof = {"bound": "hbm", "kernel": "whole step", "achieved": value / world * B_ALG / 1e9,
                    "peak": peak, "unit": "GB/s", "frac": value / world * B_ALG / (peak * 1e9), "traffic": None,
                    "peak_source": peak_src}
        if sustained is not None:
            sustained["step_frac_of_hbm_roofline"] = sustained["value"] / world * B_ALG / (peak * 1e9)
        burst["step_frac_of_hbm_roofline"] = burst["value"] / world * B_ALG / (peak * 1e9)
        cpu = None
        if not args.no_cpu:
            # SURVEY 8(d) "CPU baseline": (i) all host cores, full steps of this config; (ii) one core at C3
            full = None if args.cpu_n3 <= 0 else args.cpu_n3
            v, cores, sample, sec = oracle_sample(args.config, args.cpu_steps, full,
                                                  prebuilt=(p, prim_host) if full is None else None)
            cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": sec}
            v1, c1, sample1, sec1 = oracle_sample("C3", 1, None, threads=1)
            cpu["single_core"] = {"value": v1, "unit": UNIT, "cores": c1, "kind": "oracle", "sample": sample1, "seconds": sec1}
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
               "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "f64", "data": "synthetic",
               "config": {"workload": f"{args.config}: {p['n1']}x{p['n2']}x{p['n3']} MKS Fishbone-Moncrief torus, "
                                      f"a={p['a']}, gam={p['gam']:.4f}, recon={'PPM' if p['recon'] else 'PLM-MC'}, "
                                      f"riemann={'HLL' if p['riemann'] else 'LLF'}, "
                                      + ("dt from eq. 26 every step (cuharm_step_cfl, xi = 0.45)" if args.cfl_each_step
                                         else "fixed dt from cfl_dt(0.45)"),
                          "newton_tol": p["newton_tol"], "newton_extra": p["newton_extra"], "newton_maxit": p["newton_maxit"],
                          "l2": "inputs larger than L2 (prim 1.15 GB, fluxes 3 GB per substep vs 126 MB L2)",
                          "parallelism": "replicas only" if world > 1 else "single GPU", "graph": bool(args.graph),
                          "cfl_each_step": bool(args.cfl_each_step),
                          "dt": dt},
               "clocks": clocks, "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": nbytes,
                                         "d2h_bytes_per_step": nbytes, "steps": e2e_steps,
                                         "pipeline": "3 solver objects on 3 streams, steps dealt round-robin (independent "
                                                     "one-step problems)",
                                         "serial": {"value": e2e_serial, "unit": UNIT, "steps": ser_steps,
                                                    "pipeline": "one solver, one stream; step n+1 loads the host array "
                                                                "step n wrote (a time-dependent run through host buffers)"}},
               "gpu_launches": int(launches), "roofline": roof, "roofline_alu": roof_alu,
               "roofline_per_kernel": per_kernel, "burst": burst, "sustained": sustained,
               "headline_region": ("K steps timed after the sustained leg (board at the steady state of the metric's "
                                   "500-step run)" if sustained is not None else "K steps after the warm-up and the burst leg"),
               "cpu_baseline": cpu,
               "checks": {"divb_norm": divb, "stats": stats}}
        print(json.dumps(out), flush=True)
    s.close()
    if dist is not None:
        dist.destroy_process_group()


def run_decomposed(args):
    """--decompose: the grid cut into WORLD_SIZE slabs along X1, one per rank / GPU (paper_2205_02484_b200/slab.py: halo
    exchange over NCCL after every substep, max of the face speeds over the ranks), strong scaling: the whole job is ONE
    grid.  Not measured on more than one GPU in this build; with one rank it times the split-step
    path (plain launches, one host synchronisation per substep for the repair's counts) against the replayed graph."""
    import numpy as np
    import torch
    import paper_2205_02484_b200 as cu
    from paper_2205_02484_b200 import slab
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    p, prim_host = make_workload(args.config)
    mine = np.ascontiguousarray(prim_host[:, slab.slab_slice(p, world, rank)])
    eng = cu.Solver(slab.slab_params(p, world, rank), torch.from_numpy(mine).pin_memory(), device=f"cuda:{local}")
    if world > 1:
        me = slab.SlabRank(eng, p, rank, world)
    else:
        me = slab.SlabGroup([eng], p)
    dt = me.cfl_dt(0.45)
    for _ in range(max(args.warmup, 3)):
        me.step(dt)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        me.step(dt)
    e1.record()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    if dist is not None:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    zones = p["n1"] * p["n2"] * p["n3"]
    if rank == 0:
        peak, peak_src, _ = peaks()
        value = zones * args.steps / (ms * 1e-3)
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                          "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                          "dtype": "f64", "data": "synthetic",
                          "config": {"workload": f"{args.config}: one {p['n1']}x{p['n2']}x{p['n3']} grid in {world} slab(s) along X1",
                                     "parallelism": f"slab decomposition x{world}, halo exchange per substep", "dt": dt},
                          "roofline": {"bound": "hbm", "kernel": "whole step", "achieved": value * B_ALG / 1e9 / world, "peak": peak,
                                       "unit": "GB/s", "frac": value * B_ALG / (peak * 1e9) / world, "traffic": None, "peak_source": peak_src},
                          "gpu_launches": int(eng.launch_count())}), flush=True)
    eng.close()
    if dist is not None:
        dist.destroy_process_group()


def run_repair_scaling(args):
    """Cost of the eq. 34 repair (cuharm_repair: list build + the grid-wide repair kernel) on the headline grid for
    1e3 / 1e5 / 1e6 failed zones: random isolated zones plus 4 x 3 patches (diagonal stencil, later
    passes, last-resort rule), timed with CUDA events, beside the time of a full step of the same grid."""
    import numpy as np
    import torch
    import paper_2205_02484_b200 as cu
    p, prim_host = make_workload(args.config)
    s = cu.Solver(p, torch.from_numpy(prim_host).pin_memory())
    dt = s.cfl_dt(0.45)
    s.use_graph(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(5):
        s.step(dt)
    e0.record()
    for _ in range(10):
        s.step(dt)
    e1.record(); torch.cuda.synchronize()
    step_ms = e0.elapsed_time(e1) / 10
    ng, n1, n2, n3 = p["ng"], p["n1"], p["n2"], p["n3"]
    r = np.random.Generator(np.random.PCG64(220502484))
    rows = []
    for target in (0, 1000, 100000, 1000000):
        bad = np.zeros((n1, n2, n3), dtype=bool)
        if target:
            bad |= r.random((n1, n2, n3)) < 0.8 * target / bad.size
            for _ in range(max(1, int(0.2 * target / 12))):
                i, j, k = r.integers(0, n1 - 4), r.integers(0, n2 - 3), r.integers(0, n3)
                bad[i:i + 4, j:j + 3, k] = True
        flag = np.zeros((n1 + 2 * ng, n2 + 2 * ng, n3 + 2 * ng), dtype=np.int32)
        flag[ng:-ng, ng:-ng, ng:-ng][bad] = 2
        dflag = torch.as_tensor(flag).cuda()
        work = s.prim.clone()
        st0 = s.stats()
        s.repair(work, dflag)                      # warm-up of this pattern (also makes the timed call idempotent in cost)
        work.copy_(s.prim)
        torch.cuda.synchronize()
        e0.record()
        s.repair(work, dflag)
        e1.record(); torch.cuda.synchronize()
        st = s.stats()
        rows.append({"failed_zones": int(bad.sum()), "repair_ms": e0.elapsed_time(e1),
                     "frac_of_step": e0.elapsed_time(e1) / step_ms, "last_resort": (st[7] - st0[7]) // 2})
    print(json.dumps({"repair_scaling": rows, "step_ms": step_ms, "config": args.config,
                      "note": "cuharm_repair = flag-array scan over the whole grid + fixup_kernel; inside cuharm_step the list "
                              "comes from the update kernel, so the scan (the cost at 0 failed zones) is not paid"}), flush=True)
    s.close()


def run_chain_cost(args):
    """--chain: what the inversion fallback chain of P:L229-239 costs where it is hot.  The headline grid
    with inv_chain = 1 and beta_min = 1e-2 (eq. 33: zones below it take the entropy method as first and only choice), the
    torus field scaled up until at least `--chain-frac` of the zones are eq. 33 zones; sustained-style timing of the same
    state with the chain off and on; chain counters per step in the line."""
    import torch
    import paper_2205_02484_b200 as cu
    p0, prim_host = make_workload(args.config)
    zones = p0["n1"] * p0["n2"] * p0["n3"]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def run(p, prim, nsteps):
        s = cu.Solver(p, torch.from_numpy(prim).pin_memory())
        dt = s.cfl_dt(0.45)
        s.use_graph(True)
        for _ in range(3):
            s.step(dt)
        c0, st0 = (s.chain_stats() if p["inv_chain"] else [0] * 4), s.stats()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(nsteps):
            s.step(dt)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / nsteps
        c1, st1 = (s.chain_stats() if p["inv_chain"] else [0] * 4), s.stats()
        out = {"ms_per_step": ms, "chain_per_step": [(b - a) / nsteps for a, b in zip(c0, c1)],
               "failed_inversions_per_step": (st1[0] - st0[0]) / nsteps, "repaired_per_step": (st1[1] - st0[1]) / nsteps,
               "divb_norm": s.divb()[1], "dt": dt}
        s.close()
        return out

    rows = []
    for bscale in ((args.chain_bscale,) if args.chain_bscale > 0 else (1.0, 30.0, 100.0, 300.0, 1000.0)):
        prim = prim_host.copy()
        prim[5:8] *= bscale
        on = run(dict(p0, inv_chain=1, beta_min=args.beta_min), prim, 3)
        frac = on["chain_per_step"][3] / (2.0 * zones)          # eq. 33 zones per substep / zones
        rows.append({"bscale": bscale, "eq33_zone_fraction": frac, "probe_ms_per_step": on["ms_per_step"]})
        if frac >= args.chain_frac:
            break
    prim = prim_host.copy()
    prim[5:8] *= rows[-1]["bscale"]
    off = run(dict(p0, inv_chain=0), prim, args.steps)
    on = run(dict(p0, inv_chain=1, beta_min=args.beta_min), prim, args.steps)
    base = run(dict(p0, inv_chain=1, beta_min=args.beta_min), prim_host.copy(), args.steps)
    print(json.dumps({"chain_cost": {"config": args.config, "beta_min": args.beta_min, "steps": args.steps, "search": rows,
                                     "bscale": rows[-1]["bscale"], "chain_off": off, "chain_on": on,
                                     "chain_on_unscaled_field": base,
                                     "extra_ms_per_step": on["ms_per_step"] - off["ms_per_step"],
                                     "extra_frac_of_step": on["ms_per_step"] / off["ms_per_step"] - 1.0,
                                     "chain_per_step_legend": ["2D failed -> chain", "recovered by 1D-W", "recovered by entropy",
                                                               "eq. 33 zones (entropy first and only)"]}}), flush=True)


def run_fp64_peak():
    """--fp64-peak: build and run bench_fp64_peak.cu (beside this file), the DFMA micro-benchmark behind the "alu" roofline
    peak: cycles per warp-level DFMA per SM sub-partition and the device-wide rate for ILP x
    resident-warps combinations.  A measurement aid; nothing in the library depends on it."""
    import tempfile
    src = os.path.join(ROOT, "bench_fp64_peak.cu")
    with tempfile.TemporaryDirectory() as tmp:
        exe = os.path.join(tmp, "fp64_peak")
        subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe, src], check=True)
        return subprocess.run([exe]).returncode


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--graph", type=int, default=1)
    ap.add_argument("--e2e-steps", type=int, default=18)
    ap.add_argument("--cpu-steps", type=int, default=2, help="cpu_baseline: RK2 steps of the oracle on all host cores")
    ap.add_argument("--cpu-n3", type=int, default=0, help="cpu_baseline: phi zones of the sample (0 = the full grid)")
    ap.add_argument("--ref-n3", type=int, default=32, help="--impl reference: phi zones of the per-step sample")
    ap.add_argument("--sustain-s", type=float, default=3.0, help="sustained leg: at least this many seconds (0 = skip)")
    ap.add_argument("--sustain-warm-s", type=float, default=2.0, help="sustained leg: load before its timed region")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cfl-each-step", action="store_true", help="a new dt every step from eq. 26 (cuharm_step_cfl)")
    ap.add_argument("--decompose", action="store_true", help="one grid cut into WORLD_SIZE slabs (strong scaling) instead of replicas")
    ap.add_argument("--repair-scaling", action="store_true", help="time the eq. 34 repair at 1e3 / 1e5 / 1e6 failed zones")
    ap.add_argument("--threads", type=int, default=0, help="reference arm: OpenMP threads of the oracle (0 = all)")
    ap.add_argument("--chain", action="store_true", help="cost of the inversion fallback chain on a magnetised state")
    ap.add_argument("--chain-frac", type=float, default=0.05, help="--chain: scale B until this fraction of zones are eq. 33 zones")
    ap.add_argument("--beta-min", type=float, default=1e-2, help="--chain: eq. 33 threshold")
    ap.add_argument("--chain-bscale", type=float, default=0.0, help="--chain: use this field scale instead of searching for one")
    ap.add_argument("--fp64-peak", action="store_true", help="run the DFMA micro-benchmark (bench_fp64_peak.cu) and exit")
    args = ap.parse_args()
    if args.fp64_peak:
        sys.exit(run_fp64_peak())
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.chain:
        run_chain_cost(args)
    elif args.repair_scaling:
        run_repair_scaling(args)
    elif args.decompose and args.impl == "ours":
        run_decomposed(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
