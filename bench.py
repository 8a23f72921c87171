#!/usr/bin/env python
"""bench.py -- Dhop throughput on B200 (BASELINE.json metric: GFlop/s at 1320 flop per output
5D site, and the fraction of the HBM roofline of the minimal-traffic model).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload c4]

Workload at N=1: BASELINE.json configs[3] ("C4"): 32^4 x Ls=16, complex fp32, near-unit gauge
(eps=0.2), Gaussian spinor on the even checkerboard.  One STEP = one red-black matvec as the
config states it, plus the reduction of the hot path's last row:
    chi_o = DhopOE psi_e ;  phi_e = DhopEO chi_o ;  n = norm2(phi_e) -> host (8 bytes)
(the last two through dwf_dhop_eo_norm2_async: the reduction runs in the epilogue of the DhopEO kernel; the host reads the
value of step k with dwf_reduction_wait while step k + 1 runs, all K values inside the timed region)
`value` counts 2 x 1320 x (V4/2 x Ls) flop per step (the norm2 flops are not counted).
Inputs are resident in HBM before the timed region; fields are far larger than L2 (805 MB per
half field, 604 MB of links), so no L2 flush is needed between iterations.

`e2e` is the same step through the C ABI with HOST buffers: every step imports psi_e from
pinned host memory (H2D + reorder), runs the three calls, and exports phi_e back to pinned
host memory (reorder + D2H).

`--impl reference` times the CPU oracle (oracle/, plain fp64 definition, OpenMP) on the host
cores on the same workload; there is no other reference implementation (the paper ships none).

`roofline.frac` is the event-timed DhopOE launch of the K timed steps; `roofline.frac_sustained` is the
same kernel in a >= 2 s loop of back-to-back half-Dhops with no host synchronisation inside
(the regime in which the board sits at its power limit), with its own clock record.

Multi-GPU: the path does not shard (north_star: one GPU, no halo exchange) -- "replicas only":
every rank runs the same workload on its own GPU, value = total sites / max time over ranks.
`--gpus N` without a launcher (no WORLD_SIZE in the environment) starts the N ranks itself.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE = 1320

WORKLOADS = {
    # name: dims, Ls, precision, bc_time, gauge kind, seed
    "c3": dict(dims=(16, 16, 16, 16), Ls=16, prec=4, bc=0, gauge="random", seed=1003),
    "c4": dict(dims=(32, 32, 32, 32), Ls=16, prec=4, bc=0, gauge="near_unit", seed=1004),
    "c4d": dict(dims=(32, 32, 32, 32), Ls=16, prec=8, bc=0, gauge="near_unit", seed=1004),
    # the paper's threshold volume per GPU ("24^4 and above") with the C4 recipe
    "c24": dict(dims=(24, 24, 24, 24), Ls=16, prec=4, bc=0, gauge="near_unit", seed=1004),
    "c24d": dict(dims=(24, 24, 24, 24), Ls=16, prec=8, bc=0, gauge="near_unit", seed=1004),
    "c64": dict(dims=(64, 16, 16, 32), Ls=16, prec=4, bc=0, gauge="near_unit", seed=1004),
    "c5": dict(dims=(48, 48, 48, 96), Ls=12, prec=4, bc=1, gauge="random", seed=1005),
    "tiny": dict(dims=(8, 8, 8, 8), Ls=8, prec=4, bc=1, gauge="random", seed=1002),
    # the Schur complement of the red-black Shamir DWF operator on the C4 shape
    "schur": dict(dims=(32, 32, 32, 32), Ls=16, prec=4, bc=0, gauge="near_unit", seed=1004, kind="schur"),
    # time-decomposed Dhop, every rank owns a C4-sized slab (weak scaling: global lattice 32^3 x 32 N)
    "c4slab": dict(dims=(32, 32, 32, 32), Ls=16, prec=4, bc=1, gauge="near_unit", seed=1004, kind="slab"),
    # 12-real link storage (third row rebuilt in the kernel), C4 shape
    "c4g12": dict(dims=(32, 32, 32, 32), Ls=16, prec=4, bc=0, gauge="near_unit", seed=1004, gauge12=1),
    # four right-hand sides sharing one gauge load, C4 shape
    "c4m4": dict(dims=(32, 32, 32, 32), Ls=16, prec=4, bc=0, gauge="near_unit", seed=1004, kind="mrhs", nrhs=4),
    # the solver the paper's workload is: CG on the Schur normal equations, a fixed number of iterations on the C4 shape
    "cg": dict(dims=(32, 32, 32, 32), Ls=16, prec=4, bc=1, gauge="near_unit", seed=1004, kind="cg"),
    "schurd": dict(dims=(32, 32, 32, 32), Ls=16, prec=8, bc=0, gauge="near_unit", seed=1004, kind="schur"),
    # spinor fields stored as fp16, fp32 links and arithmetic, C4 shape
    "c4h": dict(dims=(32, 32, 32, 32), Ls=16, prec=4, bc=0, gauge="near_unit", seed=1004, kind="f16"),
}


def workload_name(w):
    d = w["dims"]
    return (f"DWF even/odd Dhop {d[0]}x{d[1]}x{d[2]}x{d[3]} x Ls={w['Ls']} complex "
            f"fp{w['prec'] * 8}, {w['gauge']} SU(3) gauge" + (", 12-real link storage for the plain DhopOE" if w.get("gauge12") else "") +
            ", DhopOE then DhopEO then norm2")


def model_bytes_cb(w):
    """Minimal-traffic model of ONE half-Dhop: one spinor read + one write per
    output site, the whole gauge field once."""
    d = w["dims"]
    V4 = d[0] * d[1] * d[2] * d[3]
    link_reals = 48 if w.get("gauge12") else 72            # 12-real storage: two rows of every link
    return (V4 // 2) * w["Ls"] * 48 * w["prec"] + V4 * link_reals * w["prec"]


def make_inputs(w):
    import dwf_inputs as gen
    d = w["dims"]
    if w["gauge"] == "near_unit":
        U = gen.gauge_near_unit(d, w["seed"], 0.2, prec=w["prec"])
    else:
        U = gen.gauge_random(d, w["seed"], prec=w["prec"])
    psi_e = gen.spinor_gaussian(gen.volume(d) // 2, w["Ls"], w["seed"], prec=w["prec"])
    return U, psi_e


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.005)

    def start(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ---------------------------------------------------------------------------------------------
# the CPU oracle arm (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------
def oracle_step(w, U, psi_e):
    """One whole step of the workload on the host cores with the oracle as it stands."""
    import oracle
    d, Ls, bc = w["dims"], w["Ls"], w["bc"]
    t0 = time.perf_counter()
    chi_o = oracle.dhop_oe(d, Ls, bc, U, psi_e)
    phi_e = oracle.dhop_eo(d, Ls, bc, U, chi_o)
    n = oracle.norm2(phi_e)
    return time.perf_counter() - t0, n


def cpu_baseline(w, U, psi_e, steps=1):
    import oracle
    d = w["dims"]
    sites = (d[0] * d[1] * d[2] * d[3] // 2) * w["Ls"]
    runs = [oracle_step(w, U, psi_e) for _ in range(steps)]
    best = min(r[0] for r in runs)
    cpu_baseline.norm2 = runs[0][1]
    return {"value": 2 * FLOP_PER_SITE * sites / best / 1e9, "unit": "GFlop/s",
            "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"one whole step (DhopOE + DhopEO + norm2) of the same workload, {best:.2f} s, fp64"}


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    U, psi_e = make_inputs(w)
    d = w["dims"]
    sites = (d[0] * d[1] * d[2] * d[3] // 2) * w["Ls"]
    # each step is a bounded sample of the workload so that K steps end within minutes:
    # a whole step when it is cheap, else the OE/EO pair at a seeded sample of output sites
    probe, _ = oracle_step(w, U, psi_e)
    budget = 120.0
    whole = probe * (args.steps + args.warmup) <= budget
    if whole:
        for _ in range(max(0, args.warmup - 1)):
            oracle_step(w, U, psi_e)
        times = [oracle_step(w, U, psi_e)[0] for _ in range(args.steps)]
        per_step_sites, sample = 2 * sites, "whole steps"
    else:
        import dwf_inputs as gen
        par = gen.site_parity(d)
        rng = np.random.default_rng(w["seed"])
        n = max(1024, int(len(par) / 2 * budget / (probe * (args.steps + args.warmup))))
        odd = rng.choice(np.nonzero(par == 1)[0], n, replace=False)
        times = []
        for i in range(args.warmup + args.steps):
            t0 = time.perf_counter()
            oracle.dhop_sites(d, w["Ls"], w["bc"], U, psi_e, True, odd)
            if i >= args.warmup:
                times.append(time.perf_counter() - t0)
        per_step_sites, sample = n * w["Ls"], f"DhopOE at {n} sampled odd sites per step"
    tot = sum(times)
    val = FLOP_PER_SITE * per_step_sites * len(times) / tot / 1e9
    line = {
        "impl": "reference", "metric": "Dhop GFlop/s (1320 flop/5D site)", "value": val, "unit": "GFlop/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * tot / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(w), "name": args.workload, "dims": list(d), "Ls": w["Ls"],
                   "note": "CPU oracle on host cores: " + sample},
        "cpu_baseline": {"value": val, "unit": "GFlop/s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "GFlop/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------
def ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the
    `ncu --set full` capture summarised under profiles/ (profiles/traffic.json is written beside each
    summary: {workload: {"kernel": ..., "bytes": ..., "source": ...}}).  None when there is no capture of
    this workload with the kernel that actually ran."""
    try:
        rec = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))[workload]
    except Exception:
        return None, None
    if rec.get("kernel") and rec["kernel"] != kernel:
        return None, f"capture is of {rec['kernel']}, not of {kernel}"
    return rec.get("bytes"), rec.get("source")


def max_over_ranks(x, dist=None, device="cuda"):
    """Slowest rank's time (device-timed milliseconds): all-reduce MAX over the process group (N > 1)."""
    if dist is None:
        return x
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gflops(world, sites_per_half_dhop, ms_step):
    """Replicas only: every rank runs the same two half-Dhops per step, so the
    whole-job throughput is world x per-rank flop over the slowest rank's step time."""
    return world * 2 * FLOP_PER_SITE * sites_per_half_dhop / (ms_step * 1e-3) / 1e9


def run_gpu(args, w):
    import torch
    import paper_2203_06777_b200 as dwf

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit(f"bench.py: no CUDA device for rank {rank} of {world} (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dwf.load()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    d, Ls, prec = w["dims"], w["Ls"], w["prec"]
    V4 = d[0] * d[1] * d[2] * d[3]
    sites = (V4 // 2) * Ls                          # output 5D sites of one half-Dhop
    U, psi_e = make_inputs(w)

    g = dwf.Geometry(d, Ls, prec, w["bc"], device=local_rank)
    for kv in args.opt or []:
        k, v = kv.split("=")
        g.set_option(k, int(v))
    if w.get("gauge12"):
        g.set_option("gauge12", 1)
    g.load_gauge(U)
    f_in = g.import_spinor(psi_e, dwf.EVEN)
    f_mid, f_out = g.new_field(dwf.ODD), g.new_field(dwf.EVEN)

    def step():
        g.dhop_oe(f_in, f_mid)
        return g.dhop_eo_norm2(f_mid, f_out)[1]      # DhopEO with the norm2 of its result fused in

    for _ in range(args.warmup):
        n_gpu = step()

    # ---- timed region: K steps, device time, per-launch events on the launching stream ----
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(physical_gpu_index(local_rank))
    barrier()
    sampler.start()
    l0 = dwf.dwf_launch_count()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record()
    # the norm2 of step k is read by the host while step k + 1 runs (dwf_dhop_eo_norm2_async / dwf_reduction_wait): every
    # step's value is read inside the timed region, the GPU does not idle on the host in between
    pending = None
    for k in range(args.steps):
        ev[k][0].record()
        g.dhop_oe(f_in, f_mid)
        ev[k][1].record()
        _, ticket = g.dhop_eo_norm2_async(f_mid, f_out)
        ev[k][2].record()
        if pending is not None:
            n_gpu = g.reduction_wait(pending)
        pending = ticket
    n_gpu = g.reduction_wait(pending)
    t_end.record()
    barrier()
    launches = dwf.dwf_launch_count() - l0
    clocks = sampler.stop()
    ms_total = max_over_ranks(t_start.elapsed_time(t_end), dist)
    ms_step = ms_total / args.steps
    t_oe = float(np.mean([e[0].elapsed_time(e[1]) for e in ev]))
    t_eo = float(np.mean([e[1].elapsed_time(e[2]) for e in ev]))
    value = whole_job_gflops(world, sites, ms_step)

    # ---- sustained regime: >= 2 s of half-Dhops back to back, no host synchronisation inside ----
    # (north_star says "sustains": after ~60 ms the board reaches its power limit and the SM clock sags)
    sustained = None
    if args.sustain > 0:
        n_pairs = max(10, int(args.sustain / (2 * t_oe * 1e-3)) + 1)
        s_sampler = ClockSampler(physical_gpu_index(local_rank))
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        s_sampler.start()
        s0.record()
        for _ in range(n_pairs):
            g.dhop_oe(f_in, f_mid)
            g.dhop_eo(f_mid, f_out)
        s1.record()
        barrier()
        s_clocks = s_sampler.stop()
        ms_sus = max_over_ranks(s0.elapsed_time(s1), dist)
        sustained = {"seconds": ms_sus * 1e-3, "launches": 2 * n_pairs, "us_per_launch": 1e3 * ms_sus / (2 * n_pairs),
                     "clocks": s_clocks}

    # ---- small lattices: the same half-Dhops replayed from a CUDA graph (no launch gaps, no host in the loop) ----
    graph_line = None
    if psi_e.nbytes < 200e6:
        side = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        reps = 20
        with torch.cuda.stream(side):
            g.dhop_oe(f_in, f_mid)                  # warm the tensor-map cache of this thread outside the capture
            g.dhop_eo(f_mid, f_out)
            torch.cuda.synchronize()
            with torch.cuda.graph(graph, stream=side):
                for _ in range(reps):
                    g.dhop_oe(f_in, f_mid)
                    g.dhop_eo(f_mid, f_out)
        graph.replay()
        torch.cuda.synchronize()
        ga, gb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ga.record()
        for _ in range(5):
            graph.replay()
        gb.record()
        torch.cuda.synchronize()
        us_graph = 1e3 * ga.elapsed_time(gb) / (5 * 2 * reps)
        graph_line = {"us_per_half_dhop": us_graph, "frac": model_bytes_cb(w) / (us_graph * 1e-6) / 1e9 / peaks()[0],
                      "note": f"{reps} DhopOE + DhopEO pairs captured in one CUDA graph, replayed 5 times"}
        # the full-field operator dwf_dhop (fp32 staged geometries: ONE launch over both parities), event-timed with the
        # host in the loop and replayed from a graph; two half fields of traffic per launch
        ff_in, ff_out = g.new_field(dwf.FULL), g.new_field(dwf.FULL)
        ff_in.normal_()
        n_l0 = dwf.dwf_launch_count()
        g.dhop(ff_in, ff_out)
        launches_full = dwf.dwf_launch_count() - n_l0
        torch.cuda.synchronize()
        ga.record()
        for _ in range(2 * reps):
            g.dhop(ff_in, ff_out)
        gb.record()
        torch.cuda.synchronize()
        us_full = 1e3 * ga.elapsed_time(gb) / (2 * reps)
        graph2 = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            torch.cuda.synchronize()
            with torch.cuda.graph(graph2, stream=side):
                for _ in range(reps):
                    g.dhop(ff_in, ff_out)
        graph2.replay()
        torch.cuda.synchronize()
        ga.record()
        for _ in range(5):
            graph2.replay()
        gb.record()
        torch.cuda.synchronize()
        us_full_graph = 1e3 * ga.elapsed_time(gb) / (5 * reps)
        mb_full = 2 * model_bytes_cb(w)
        graph_line["full_dhop"] = {"launches_per_dhop": launches_full, "us_per_dhop": us_full, "us_per_dhop_graph": us_full_graph,
                                   "frac": mb_full / (us_full * 1e-6) / 1e9 / peaks()[0],
                                   "frac_graph": mb_full / (us_full_graph * 1e-6) / 1e9 / peaks()[0],
                                   "note": "dwf_dhop on a full field; fields of this size stay partly resident in the 126 MB L2 "
                                           "between launches, so the HBM model is an upper bound on the DRAM traffic (SURVEY.md 8(d))"}
        del ff_in, ff_out

    # ---- e2e: the same step through the C ABI with HOST buffers ----
    host_in = torch.empty(psi_e.shape, dtype=torch.from_numpy(psi_e).dtype, pin_memory=True)
    host_in.copy_(torch.from_numpy(psi_e))
    host_out = torch.empty_like(host_in, pin_memory=True)
    hin, hout = host_in.numpy(), host_out.numpy()

    # host transfers pipelined across steps (option "async_host"): the import of step k + 1 is issued on a side stream
    # into a second input field before the kernels of step k, and step k's export (D2H) runs under it (H2D): both copy
    # engines stay busy; dwf_host_wait inside the timed region waits for the last copies
    f_in2 = g.new_field(dwf.EVEN)
    in_bufs = [f_in, f_in2]
    in_stream = torch.cuda.Stream()
    in_done = [torch.cuda.Event(), torch.cuda.Event()]

    def issue_import(k):
        with torch.cuda.stream(in_stream):
            g.import_spinor(hin, dwf.EVEN, out=in_bufs[k & 1])
            in_done[k & 1].record(in_stream)

    def step_e2e(k, last):
        if not last:
            issue_import(k + 1)         # its buffer was last read by DhopOE of step k - 1, which the norm2 read-back synchronised
        torch.cuda.current_stream().wait_event(in_done[k & 1])
        g.dhop_oe(in_bufs[k & 1], f_mid)
        n = g.dhop_eo_norm2(f_mid, f_out)[1]
        g.export_spinor(f_out, dwf.EVEN, out=hout)
        return n

    g.set_option("async_host", 1)
    k_e2e = max(1, min(args.steps, 20))
    issue_import(0)
    for k in range(2):
        step_e2e(k, k == 1)
    g.host_wait()
    torch.cuda.synchronize()
    barrier()
    t0_e2e = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    issue_import(0)                     # k_e2e imports and k_e2e exports inside the timed region
    for k in range(k_e2e):
        n_e2e = step_e2e(k, k == k_e2e - 1)
    g.host_wait()
    torch.cuda.current_stream().wait_stream(in_stream)
    e1.record()
    torch.cuda.synchronize()
    barrier()
    g.set_option("async_host", 0)
    ms_e2e = max_over_ranks(e0.elapsed_time(e1), dist) / k_e2e
    e2e_val = whole_job_gflops(world, sites, ms_e2e)
    field_bytes = psi_e.nbytes

    # ---- optional: the NEXT-row kernels of SURVEY.md 8(f1), each event-timed on its own ----
    extra = None
    if args.extra_ops:
        def timed(fn, n=20):
            fn()
            e_a, e_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e_a.record()
            for _ in range(n):
                fn()
            e_b.record()
            torch.cuda.synchronize()
            return e_a.elapsed_time(e_b) / n
        t_dag = timed(lambda: g.dhop_eo_dag(f_mid, f_out))
        t_axpy = timed(lambda: g.dhop_eo_axpy(f_mid, f_in, 1.0, -0.25 / (4.3 * 4.3), f_out))
        mb_axpy = model_bytes_cb(w) + sites * 24 * prec          # + one read of x
        extra = {"dhop_eo_dag_ms": t_dag, "dhop_eo_axpy_ms": t_axpy,
                 "axpy_algorithmic_bytes_per_launch": mb_axpy,
                 "note": "a x + b DhopEO in one pass; model = half-Dhop model + one read of x"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = peaks()
    # the roofline kernel is the plain half-Dhop launch (DhopOE), bracketed by events on its own; the
    # DhopEO interval also holds the final sum of the fused norm2, the 8-byte D2H copy and the host wake-up
    t_dhop = t_oe
    mb = model_bytes_cb(w)
    achieved = mb / (t_dhop * 1e-3) / 1e9
    kernel = g.kernel_info()
    traffic, traffic_src = ncu_traffic(args.workload, kernel)
    fld_mb, gauge_mb = psi_e.nbytes / 1e6, 2 * U.nbytes / 1e6
    l2_note = (f"inputs larger than L2 ({fld_mb:.0f} MB half fields, {gauge_mb:.0f} MB links); no flush" if fld_mb > 200 else
               f"working set ({3 * fld_mb:.0f} MB of fields + {gauge_mb:.0f} MB links) is partly L2-resident across steps: "
               "model GB/s may exceed the HBM peak; no flush (SURVEY.md 8(d) caveat)")
    line = {
        "metric": "Dhop GFlop/s (1320 flop/5D site)", "value": value, "unit": "GFlop/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if prec == 4 else "f64", "data": "synthetic",
        "config": {"workload": workload_name(w), "name": args.workload, "dims": list(d), "Ls": Ls,
                   "l2": l2_note,
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": "GFlop/s", "ms_per_step": ms_e2e,
                "h2d_bytes_per_step": field_bytes, "d2h_bytes_per_step": field_bytes + 8},
        "gpu_launches": int(launches),
        "kernels_ms": {"dhop_oe": t_oe, "dhop_eo_norm2": t_eo},
        "dhop_only_gflops": FLOP_PER_SITE * sites / (t_dhop * 1e-3) / 1e9,
        "roofline": {"bound": "hbm", "kernel": kernel + " (DhopOE launches)", "achieved": achieved, "peak": peak,
                     "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": mb,
                     "traffic": traffic, "traffic_source": traffic_src},
    }
    if graph_line is not None:
        line["cuda_graph"] = graph_line
    if sustained is not None:
        ach_s = mb / (sustained["us_per_launch"] * 1e-6) / 1e9
        line["roofline"]["frac_sustained"] = ach_s / peak
        line["roofline"]["achieved_sustained"] = ach_s
        line["roofline"]["sustained"] = sustained
    if extra is not None:
        extra["dag_roofline_frac"] = mb / (extra["dhop_eo_dag_ms"] * 1e-3) / 1e9 / peak
        extra["axpy_roofline_frac"] = extra["axpy_algorithmic_bytes_per_launch"] / (extra["dhop_eo_axpy_ms"] * 1e-3) / 1e9 / peak
        line["next_rows"] = extra
    if world == 1 and not args.no_cpu:
        cb = cpu_baseline(w, U, psi_e)
        line["cpu_baseline"] = cb
        # free full-size sanity check: norm2 of the step's result, CUDA path (fp32/fp64) vs oracle (fp64)
        line["check"] = {"norm2_gpu": n_gpu, "norm2_oracle": cpu_baseline.norm2,
                         "rel_diff": abs(n_gpu - cpu_baseline.norm2) / cpu_baseline.norm2}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_gpu_schur(args, w):
    """--workload schur: SURVEY.md 8(f2) on the C4 shape: one application of the even-site Schur complement
    S = Mooee - 1/4 DhopEO Mooee^-1 DhopOE (four kernels) per step, plus every kernel of the sequence timed
    on its own against its own minimal-traffic model (one read + one write of the field for the
    fifth-dimension passes; + one read of x and the links for a x + b Dhop)."""
    import torch
    import paper_2203_06777_b200 as dwf
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dwf.load()
    d, Ls, prec = w["dims"], w["Ls"], w["prec"]
    V4 = d[0] * d[1] * d[2] * d[3]
    sites = (V4 // 2) * Ls
    M5, mass = 1.8, 0.01
    U, psi_e = make_inputs(w)
    g = dwf.Geometry(d, Ls, prec, w["bc"], device=local_rank)
    for kv in args.opt or []:
        k, v = kv.split("=")
        g.set_option(k, int(v))
    g.load_gauge(U)
    f_in = g.import_spinor(psi_e, dwf.EVEN)
    f_out, f_t, f_u = g.new_field(dwf.EVEN), g.new_field(dwf.ODD), g.new_field(dwf.ODD)
    work = g.new_work(dwf.dwf_schur_work_bytes(g.handle))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        g.schur(f_in, dwf.EVEN, M5, mass, out=f_out, work=work)

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(physical_gpu_index(local_rank))
    barrier()
    sampler.start()
    l0 = dwf.dwf_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    launches = dwf.dwf_launch_count() - l0
    clocks = sampler.stop()
    ms_step = max_over_ranks(e0.elapsed_time(e1), dist) / args.steps

    def timed(fn, n=max(10, args.steps // 2)):
        for _ in range(3):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    fb = psi_e.nbytes                                   # bytes of one half field
    gb = model_bytes_cb(w) - 2 * fb                      # the whole gauge field once
    peak, peak_src = peaks()
    parts = {
        "dhop_oe": (timed(lambda: g.dhop_oe(f_in, f_t)), 2 * fb + gb),
        "mooee_inv": (timed(lambda: g.mooee_inv(f_t, dwf.ODD, M5, mass, out=f_u)), 2 * fb),
        "mooee": (timed(lambda: g.mooee(f_in, dwf.EVEN, M5, mass, out=f_out)), 2 * fb),
        "dhop_eo_axpy": (timed(lambda: g.dhop_eo_axpy(f_u, f_out, 1.0, -0.25, out=f_out)), 3 * fb + gb),
    }
    kernels = {k: {"ms": t, "algorithmic_bytes": b, "achieved_gbs": b / (t * 1e-3) / 1e9, "frac": b / (t * 1e-3) / 1e9 / peak}
               for k, (t, b) in parts.items()}
    total_model = sum(b for _, b in parts.values())
    if rank == 0:
        t_inv, b_inv = parts["mooee_inv"]
        line = {
            "metric": "Dhop GFlop/s (1320 flop/5D site)", "value": whole_job_gflops(world, sites, ms_step), "unit": "GFlop/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if prec == 4 else "f64", "data": "synthetic",
            "config": {"workload": f"red-black Shamir DWF Schur complement S = Mooee - 1/4 DhopEO Mooee^-1 DhopOE on the even sites of "
                                   f"{d[0]}x{d[1]}x{d[2]}x{d[3]} x Ls={Ls} fp{8 * prec}, M5={M5}, m={mass} (SURVEY.md 8(f2)); value counts "
                                   "the two Dhops' 1320 flop/site only",
                       "name": args.workload, "dims": list(d), "Ls": Ls, "l2": "fields larger than L2; no flush",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "clocks": clocks, "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "kernel": "s_op_kernel (Mooee^-1, one read + one write of a half field)",
                         "achieved": b_inv / (t_inv * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": b_inv / (t_inv * 1e-3) / 1e9 / peak, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": b_inv, "traffic": ncu_traffic("schur", "s_op_kernel")[0]},
            "schur_step": {"algorithmic_bytes": total_model, "achieved_gbs": total_model / (ms_step * 1e-3) / 1e9,
                           "frac": total_model / (ms_step * 1e-3) / 1e9 / peak},
            "kernels": kernels,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_gpu_mrhs(args, w):
    """--workload c4m4: SURVEY.md 8(f4), nrhs right-hand sides per launch.  One step = DhopOE then DhopEO on
    all of them (2 launches); minimal-traffic model per launch: one read + one write of nrhs half fields and
    the whole gauge field ONCE: w (48 + 144 / (Ls nrhs)) bytes per output 5D site."""
    import torch
    import paper_2203_06777_b200 as dwf
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dwf.load()
    d, Ls, prec, nrhs = w["dims"], w["Ls"], w["prec"], w["nrhs"]
    V4 = d[0] * d[1] * d[2] * d[3]
    sites = (V4 // 2) * Ls * nrhs                      # output 5D sites of one launch
    U, psi_e = make_inputs(w)
    g = dwf.Geometry(d, Ls, prec, w["bc"], device=local_rank)
    for kv in args.opt or []:
        k, v = kv.split("=")
        g.set_option(k, int(v))
    g.load_gauge(U)
    one = g.import_spinor(psi_e, dwf.EVEN)
    f_in = torch.cat([one * (1.0 + 0.25 * r) for r in range(nrhs)])      # nrhs different right-hand sides
    f_mid, f_out = torch.empty_like(f_in), torch.empty_like(f_in)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        g.dhop_oe_mrhs(f_in, nrhs, out=f_mid)
        g.dhop_eo_mrhs(f_mid, nrhs, out=f_out)

    for _ in range(args.warmup):
        step()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    sampler = ClockSampler(physical_gpu_index(local_rank))
    barrier()
    sampler.start()
    l0 = dwf.dwf_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(args.steps):
        ev[k][0].record()
        g.dhop_oe_mrhs(f_in, nrhs, out=f_mid)
        ev[k][1].record()
        g.dhop_eo_mrhs(f_mid, nrhs, out=f_out)
    e1.record()
    barrier()
    launches = dwf.dwf_launch_count() - l0
    clocks = sampler.stop()
    ms_step = max_over_ranks(e0.elapsed_time(e1), dist) / args.steps
    t_oe = float(np.mean([e[0].elapsed_time(e[1]) for e in ev]))
    if rank == 0:
        peak, peak_src = peaks()
        mb = sites * 48 * prec + V4 * 72 * prec
        achieved = mb / (t_oe * 1e-3) / 1e9
        # the result of the last right-hand side equals the single-RHS call on the same input (bitwise)
        chk = bool(torch.equal(g.dhop_oe(f_in.view(nrhs, -1)[nrhs - 1].contiguous()), f_mid.view(nrhs, -1)[nrhs - 1]))
        line = {
            "metric": "Dhop GFlop/s (1320 flop/5D site)", "value": world * 2 * FLOP_PER_SITE * sites / (ms_step * 1e-3) / 1e9, "unit": "GFlop/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if prec == 4 else "f64", "data": "synthetic",
            "config": {"workload": f"DWF even/odd Dhop {d[0]}x{d[1]}x{d[2]}x{d[3]} x Ls={Ls} fp{8 * prec}, {nrhs} right-hand sides per launch "
                                   "sharing one gauge load (SURVEY.md 8(f4)), DhopOE then DhopEO",
                       "name": args.workload, "dims": list(d), "Ls": Ls, "nrhs": nrhs, "l2": "fields larger than L2; no flush",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "clocks": clocks, "gpu_launches": int(launches), "kernels_ms": {"dhop_oe_mrhs": t_oe},
            "roofline": {"bound": "hbm", "kernel": g.kernel_info() + f" ({nrhs} RHS, DhopOE launches)", "achieved": achieved, "peak": peak,
                         "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src, "algorithmic_bytes_per_launch": mb,
                         "traffic": ncu_traffic(args.workload, g.kernel_info())[0]},
            "check": {"last_rhs_equals_single_call_bitwise": chk},
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_gpu_f16(args, w):
    """--workload c4h: SURVEY.md 8(f4), spinor fields in fp16 storage, fp32 links and arithmetic.  One step = DhopOE then
    DhopEO (2 launches); minimal-traffic model per launch: one read + one write of a half field at 2 bytes per real plus
    the links of one parity in fp32: 96 + 576 / Ls bytes per output 5D site."""
    import torch
    import paper_2203_06777_b200 as dwf
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dwf.load()
    d, Ls, prec = w["dims"], w["Ls"], w["prec"]
    V4 = d[0] * d[1] * d[2] * d[3]
    sites = (V4 // 2) * Ls
    U, psi_e = make_inputs(w)
    g = dwf.Geometry(d, Ls, prec, w["bc"], device=local_rank)
    for kv in args.opt or []:
        k, v = kv.split("=")
        g.set_option(k, int(v))
    g.load_gauge(U)
    f32_in = g.import_spinor(psi_e, dwf.EVEN)
    f_in = g.to_f16(f32_in, dwf.EVEN)
    f_mid, f_out = g.new_field_f16(dwf.ODD), g.new_field_f16(dwf.EVEN)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        g.dhop_oe_f16(f_in, f_mid)
        g.dhop_eo_f16(f_mid, f_out)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    sampler = ClockSampler(physical_gpu_index(local_rank))
    barrier()
    sampler.start()
    l0 = dwf.dwf_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(args.steps):
        ev[k][0].record()
        g.dhop_oe_f16(f_in, f_mid)
        ev[k][1].record()
        g.dhop_eo_f16(f_mid, f_out)
    e1.record()
    barrier()
    launches = dwf.dwf_launch_count() - l0
    clocks = sampler.stop()
    ms_step = max_over_ranks(e0.elapsed_time(e1), dist) / args.steps
    t_oe = float(np.mean([e[0].elapsed_time(e[1]) for e in ev]))
    if rank == 0:
        peak, peak_src = peaks()
        mb = sites * 24 * 2 * 2 + (V4 // 2) * 8 * 18 * prec         # fp16 in + out, fp32 links of one parity
        achieved = mb / (t_oe * 1e-3) / 1e9
        # the fp32 path on the widened input, rounded once, gives the same bits
        chk = bool(torch.equal(g.dhop_oe(g.from_f16(f_in, dwf.EVEN)).to(torch.float16), f_mid))
        line = {
            "metric": "Dhop GFlop/s (1320 flop/5D site)", "value": world * 2 * FLOP_PER_SITE * sites / (ms_step * 1e-3) / 1e9, "unit": "GFlop/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"DWF even/odd Dhop {d[0]}x{d[1]}x{d[2]}x{d[3]} x Ls={Ls}, spinor fields stored as fp16, fp32 links and "
                                   "arithmetic (SURVEY.md 8(f4)), DhopOE then DhopEO",
                       "name": args.workload, "dims": list(d), "Ls": Ls, "storage": "f16", "l2": "fields larger than L2; no flush",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "clocks": clocks, "gpu_launches": int(launches), "kernels_ms": {"dhop_oe_f16": t_oe},
            "roofline": {"bound": "hbm", "kernel": g.kernel_info() + " (fp16 storage, DhopOE launches)", "achieved": achieved, "peak": peak,
                         "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src, "algorithmic_bytes_per_launch": mb,
                         "traffic": ncu_traffic(args.workload, g.kernel_info())[0]},
            "check": {"equals_fp32_path_rounded_once_bitwise": chk},
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_gpu_cg(args, w):
    """--workload cg: dwf_cg_schur on the C4 shape, `steps` CG iterations per solve (tolerance 0, so every iteration runs).
    One iteration = S p, S^dag (S p) (eight kernels of SURVEY.md 8(f2)), a fused x / r update with |r|^2, p = r + beta p, one
    norm2, and two scalar round trips to the host.  Minimal-traffic model per iteration: two Schur applications plus ten
    half-field passes of the vector algebra."""
    import torch
    import paper_2203_06777_b200 as dwf
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dwf.load()
    d, Ls, prec = w["dims"], w["Ls"], w["prec"]
    V4 = d[0] * d[1] * d[2] * d[3]
    sites = (V4 // 2) * Ls
    M5, mass = 1.8, 0.01
    U, b = make_inputs(w)
    g = dwf.Geometry(d, Ls, prec, w["bc"], device=local_rank)
    g.load_gauge(U)
    fb = g.import_spinor(b, dwf.EVEN)
    x = g.new_field(dwf.EVEN)
    work = g.new_work(dwf.dwf_cg_work_bytes(g.handle))
    iters = max(2, args.steps)
    g.cg_schur(fb, dwf.EVEN, M5, mass, 0.0, 2, x=x, work=work)              # warm-up
    sampler = ClockSampler(physical_gpu_index(local_rank))
    torch.cuda.synchronize()
    sampler.start()
    l0 = dwf.dwf_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    _, done, res = g.cg_schur(fb, dwf.EVEN, M5, mass, 0.0, iters, x=x, work=work)
    e1.record()
    torch.cuda.synchronize()
    launches = dwf.dwf_launch_count() - l0
    clocks = sampler.stop()
    ms_total = max_over_ranks(e0.elapsed_time(e1), dist)
    # the solve also applies S^dag once before and S once after the iterations: count them as one more iteration's matvecs
    ms_iter = ms_total / (done + 1)
    if rank == 0:
        peak, peak_src = peaks()
        half = b.nbytes
        gauge = model_bytes_cb(w) - 2 * half
        schur_bytes = (2 * half + gauge) + 2 * half + 2 * half + (3 * half + gauge)
        iter_bytes = 2 * schur_bytes + 10 * half
        line = {
            "metric": "Dhop GFlop/s (1320 flop/5D site)", "value": world * 4 * FLOP_PER_SITE * sites / (ms_iter * 1e-3) / 1e9, "unit": "GFlop/s",
            "n_gpus": world, "steps": int(done), "warmup": 2, "ms_per_step": ms_iter, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if prec == 4 else "f64", "data": "synthetic",
            "config": {"workload": f"CG on the normal equations of the red-black Shamir DWF Schur complement, {d[0]}x{d[1]}x{d[2]}x{d[3]} x Ls={Ls} "
                                   f"fp{8 * prec}, M5={M5}, m={mass}: {done} iterations (a step = one iteration: four half-Dhops counted in value)",
                       "name": args.workload, "dims": list(d), "Ls": Ls, "l2": "fields larger than L2; no flush",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "clocks": clocks, "gpu_launches": int(launches), "true_residual_after": res,
            "roofline": {"bound": "hbm", "kernel": "one CG iteration (8 operator kernels + 3 vector kernels + 2 reductions)",
                         "achieved": iter_bytes / (ms_iter * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": iter_bytes / (ms_iter * 1e-3) / 1e9 / peak, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": iter_bytes, "traffic": None},
        }
        print(json.dumps(line), flush=True)
    g.close()
    if dist is not None:
        dist.destroy_process_group()


def run_gpu_slab(args, w):
    """--workload c4slab: SURVEY.md 8(f3).  Every rank owns one time slab of `dims` (the global lattice is `world`
    slabs long in time, antiperiodic), one step = DhopOE then DhopEO of the decomposed operator: face pack, face
    exchange (NCCL point-to-point between neighbouring ranks; a copy when world = 1) on a side stream under the
    open-boundary bulk kernel, face terms.  Weak scaling: `value` = all ranks' sites over the slowest rank's time."""
    import torch
    import paper_2203_06777_b200 as dwf
    from paper_2203_06777_b200.dist import SlabDhop
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dwf.load()
    d, Ls, prec = w["dims"], w["Ls"], w["prec"]
    V4 = d[0] * d[1] * d[2] * d[3]
    sites = (V4 // 2) * Ls
    U, psi_e = make_inputs(w)                        # every rank uses the same slab data: timing does not depend on it
    gdims = d[:3] + (d[3] * world,)
    op = SlabDhop(gdims, Ls, prec, w["bc"], rank, world, device=local_rank)
    op.load_gauge(U)
    g = op.geometry
    f_in = g.import_spinor(psi_e, dwf.EVEN)
    f_mid, f_out = g.new_field(dwf.ODD), g.new_field(dwf.EVEN)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        op.dhop_oe(f_in, f_mid)
        op.dhop_eo(f_mid, f_out)

    for _ in range(args.warmup):
        step()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    sampler = ClockSampler(physical_gpu_index(local_rank))
    barrier()
    sampler.start()
    l0 = dwf.dwf_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(args.steps):
        ev[k][0].record()
        op.dhop_oe(f_in, f_mid)
        ev[k][1].record()
        op.dhop_eo(f_mid, f_out)
    e1.record()
    barrier()
    launches = dwf.dwf_launch_count() - l0
    clocks = sampler.stop()
    ms_step = max_over_ranks(e0.elapsed_time(e1), dist) / args.steps
    t_oe = float(np.mean([e[0].elapsed_time(e[1]) for e in ev]))
    # the same half-Dhop without decomposition (periodic slab): what the face traffic and kernels cost
    gp = dwf.Geometry(d, Ls, prec, dwf.PERIODIC, device=local_rank)
    gp.load_gauge(U)
    for _ in range(3):
        gp.dhop_oe(f_in, f_mid)
    pa, pb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pa.record()
    for _ in range(args.steps):
        gp.dhop_oe(f_in, f_mid)
    pb.record()
    torch.cuda.synchronize()
    t_plain = pa.elapsed_time(pb) / args.steps
    face = dwf.dwf_face_bytes(g.handle)
    if rank == 0:
        peak, peak_src = peaks()
        mb = model_bytes_cb(w) + 4 * face + 4 * (sites // d[3]) * 24 * prec     # + write/read of 2 faces each way, 2 layers of in and out
        achieved = mb / (t_oe * 1e-3) / 1e9
        line = {
            "metric": "Dhop GFlop/s (1320 flop/5D site)", "value": whole_job_gflops(world, sites, ms_step), "unit": "GFlop/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if prec == 4 else "f64", "data": "synthetic",
            "config": {"workload": f"time-decomposed DWF even/odd Dhop (SURVEY.md 8(f3)): {world} slab(s) of {d[0]}x{d[1]}x{d[2]}x{d[3]} x Ls={Ls} "
                                   f"fp{8 * prec} (global {gdims[0]}x{gdims[1]}x{gdims[2]}x{gdims[3]}, antiperiodic time), DhopOE then DhopEO",
                       "name": args.workload, "dims": list(d), "Ls": Ls, "l2": "fields larger than L2; no flush",
                       "parallelism": f"time slabs over {world} rank(s), half-spinor faces exchanged per half-Dhop" if world > 1 else
                                      "single GPU (the rank is its own neighbour: face exchange = device copy)"},
            "clocks": clocks, "gpu_launches": int(launches),
            "kernels_ms": {"decomposed_dhop_oe": t_oe, "plain_periodic_dhop_oe": t_plain},
            "halo": {"face_bytes": face, "sent_per_half_dhop": 2 * face, "overhead_vs_plain": t_oe / t_plain - 1.0},
            "roofline": {"bound": "hbm", "kernel": g.kernel_info() + " + face_pack / face_apply (decomposed DhopOE)", "achieved": achieved,
                         "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": mb, "traffic": None},
        }
        print(json.dumps(line), flush=True)
    gp.close()
    op.close()
    if dist is not None:
        dist.destroy_process_group()


def spawn_ranks(n: int, argv, check_devices: bool = True) -> int:
    """`python bench.py --gpus N` without a launcher: start N ranks of this script under
    torch.distributed.run on this node (one per GPU, rendezvous on 127.0.0.1) and return its exit
    code.  "Replicas only": the ranks share nothing but the timing all-reduce."""
    import socket
    import subprocess
    if check_devices:
        import torch
        have = torch.cuda.device_count()
        if have < n:
            print(f"bench.py: --gpus {n} but only {have} CUDA device(s) are visible", file=sys.stderr)
            return 2
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)        # a burst of ~15 ms; the regime over seconds is roofline.frac_sustained
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="dwf", choices=["dwf", "reference"])
    ap.add_argument("--workload", default="c4", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--extra-ops", action="store_true",
                    help="also time Dhop^dagger and the fused a x + b Dhop (SURVEY.md 8(f1)); adds `next_rows` to the line")
    ap.add_argument("--opt", action="append", help="kernel tunable key=value (dwf_set_option)")
    ap.add_argument("--sustain", type=float, default=2.2,
                    help="seconds of back-to-back half-Dhops for roofline.frac_sustained (0: skip)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "dwf" else args.warmup
    w = WORKLOADS[args.workload]
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "dwf":
        sys.exit(spawn_ranks(args.gpus, sys.argv[1:]))
    if args.impl == "reference":
        run_reference(args, w)
    elif w.get("kind") == "schur":
        run_gpu_schur(args, w)
    elif w.get("kind") == "mrhs":
        run_gpu_mrhs(args, w)
    elif w.get("kind") == "cg":
        run_gpu_cg(args, w)
    elif w.get("kind") == "f16":
        run_gpu_f16(args, w)
    elif w.get("kind") == "slab":
        run_gpu_slab(args, w)
    else:
        run_gpu(args, w)


if __name__ == "__main__":
    main()
