#!/usr/bin/env python
"""bench.py -- FIRE lattice site-updates/s of the fused LdG sweep on B200 (fp64).

One "step" = one FIRE step (one launch of the fused force+FIRE sweep kernel) over the whole
lattice.  Default workload: BASELINE.json config 4 (512^3 periodic, one-constant, random-director
quench), the largest single-GPU configuration and the one the >= 256^3 roofline target is quoted on.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4|3|5|5p|2|1] [--impl reference]

Prints ONE JSON line (rank 0).  Keys follow the driver's contract; see DESIGN.md section 8.
  value      N_sim * K / device time of lq_fire_minimize(K steps) with Q resident in HBM (CUDA events
             on the library's stream, max over ranks)
  e2e        same metric through the C ABI with HOST buffers: lq_set_Q(pinned host) +
             lq_fire_minimize(K) + lq_get_Q(pinned host), all inside the timed region
  roofline   algorithmic bytes (160 B per site-update, +1 flag byte with objects) x simulated sites
             per launch / average launch duration of the sweep (the library's CUDA events around its launch loop /
             sweep launches), against MEASURED_PEAKS.json's HBM copy bandwidth
  cpu_baseline  the oracle (oracle/, OpenMP, as it stands) timed on this box's host cores on a bounded
             crop of the same workload
Multi-GPU: the path is single-GPU by design (north_star); --gpus N runs N independent replicas
("replicas only"), value = N * units / max-over-ranks time, scaling "weak".
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
sys.path.insert(0, ROOT)

METRIC = "FIRE lattice site-updates/sec (fp64, 1 B200); achieved HBM GB/s vs peak"
UNIT = "site-updates/s"
FALLBACK_HBM_GBS = 6650.0   # B200_PROFILING.md fallback


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback"


class ClockSampler:
    """samples SM clock / throttle reasons during the timed region (pynvml, else nvidia-smi)"""

    def __init__(self, index=0, period=0.05):
        self.index, self.period = index, period
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

    def _loop(self):
        nv = self.nv
        names = {}
        for n in dir(nv):
            if n.startswith("nvmlClocksEventReason") or n.startswith("nvmlClocksThrottleReason"):
                v = getattr(nv, n)
                if isinstance(v, int) and v and n not in ("nvmlClocksEventReasonAll", "nvmlClocksThrottleReasonAll"):
                    names.setdefault(v, n.replace("nvmlClocksEventReason", "").replace("nvmlClocksThrottleReason", ""))
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit and bit & (bit - 1) == 0:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        s = sorted(self.samples)
        rs = sorted(x for x in self.reasons if x not in ("None", "GpuIdle", "ApplicationsClocksSetting"))
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz, "reasons": rs,
                "samples": len(s)}


def build_workload(name):
    from paper_1911_07045_b200 import workloads as wl
    return wl.make_config(name)


def oracle_problem(c):
    import oracle
    return oracle.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"],
                         mask=c["mask"], kind=c["kind"], W=c["W"], axis=c["axis"])


def crop_config(c, L):
    """bounded sample of the workload for the CPU oracle: the [0,L)^3 corner crop of every array (periodic
    wrap of the crop; same value distributions / structure, smaller lattice)"""
    Lx, Ly, Lz = min(L, c["Lx"]), min(L, c["Ly"]), min(L, c["Lz"])

    def crop(a, lead):
        if a is None:
            return None
        a = a.reshape(*lead, c["Lz"], c["Ly"], c["Lx"])[..., :Lz, :Ly, :Lx]
        return np.ascontiguousarray(a).reshape(*lead, -1)

    d = dict(c)
    d.update(Lx=Lx, Ly=Ly, Lz=Lz, N=Lx * Ly * Lz, q=crop(c["q"], (5,)), mask=crop(c["mask"], ()),
             kind=crop(c["kind"], ()), W=crop(c["W"], ()), axis=crop(c["axis"], (3,)))
    return d


def oracle_steps(o, s, q, steps, method="fire", eta=0.004, mu=0.8):
    """the oracle's minimiser for `method`, as it stands; returns the final q"""
    if method == "analyze":
        import oracle
        for _ in range(steps):
            oracle.analyze(q, s["mask"], 0.4)
        return q
    if method == "fire":
        return o.fire(q, steps, 0.0, s["fire"], variant=1)[0]
    return o.descent(q, 0 if method == "gd" else 1, steps, 0.0, eta, mu, variant=1)[0]


def time_oracle(c, target_s=15.0, crop=128, method="fire", eta=0.004, mu=0.8):
    """oracle minimiser steps on a crop; returns (site-updates/s, cores, sample description)"""
    import oracle
    oracle.build_oracle()
    s = crop_config(c, crop)
    o = oracle_problem(s)
    nsim = s["N"] if s["mask"] is None else int(np.sum(s["mask"] == 0))
    t0 = time.perf_counter()
    oracle_steps(o, s, s["q"], 1, method, eta, mu)
    t1 = time.perf_counter() - t0                      # 1 step (+ the initial force evaluation)
    steps = int(max(2, min(200, target_s / max(t1 / 2.0, 1e-4))))
    t0 = time.perf_counter()
    oracle_steps(o, s, s["q"], steps, method, eta, mu)
    dt = time.perf_counter() - t0
    val = nsim * steps / dt
    how = "numpy.linalg.eigh per site" if method == "analyze" else "oracle variant=factorised+OpenMP"
    desc = "%dx%dx%d corner crop of %s, %d %s steps, %s, %.1f s" % (
        s["Lx"], s["Ly"], s["Lz"], c["name"], steps, method, how, dt)
    return val, oracle.num_threads(), desc, dt, steps


def run_reference(args):
    """--impl reference: the oracle as it stands, on host cores, same metric/config keys"""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = build_workload(args.workload)
    per_step = []
    import oracle
    oracle.build_oracle()
    s = crop_config(c, args.ref_crop)
    o = oracle_problem(s)
    nsim = s["N"] if s["mask"] is None else int(np.sum(s["mask"] == 0))
    q = s["q"]
    for _ in range(args.warmup if args.warmup is not None else 1):
        q = oracle_steps(o, s, q, 1, args.method, args.eta, args.mu)
    K = args.steps if args.steps is not None else 5
    t0 = time.perf_counter()
    q = oracle_steps(o, s, q, K, args.method, args.eta, args.mu)
    dt = time.perf_counter() - t0
    val = nsim * K / dt
    sample = "%dx%dx%d corner crop of %s, %d %s steps per timed call" % (s["Lx"], s["Ly"], s["Lz"], c["name"], K, args.method)
    metric = METRIC if args.method == "fire" else METRIC.replace("FIRE", {"gd": "gradient-descent", "nesterov": "Nesterov", "analyze": "director/S/defect analysis"}[args.method])
    line = {"impl": "reference", "metric": metric, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
            "warmup": args.warmup if args.warmup is not None else 1, "ms_per_step": 1e3 * dt / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": c["name"], "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def aggregate(local_ms, local_units, world, dist=None, device=None):
    """max-over-ranks time and total units (replicas): used by the N>1 path and the gloo CPU test"""
    if world == 1 or dist is None:
        return local_ms, local_units
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([float(local_units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--workload", default="4")
    ap.add_argument("--impl", default="lq", choices=["lq", "reference"])
    ap.add_argument("--ref-crop", type=int, default=128)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--fire-path", type=int, default=0)
    ap.add_argument("--method", default="fire", choices=["fire", "gd", "nesterov", "analyze"],
                    help="minimiser whose step is timed (default: FIRE, the headline metric; gd / nesterov: SURVEY 8(f1))")
    ap.add_argument("--slabs", type=int, default=0,
                    help="FIRE only: cut the lattice into this many z-slab sub-domains ON THIS GPU (SURVEY 8(f4): sweeps per "
                         "slab + device-to-device halo copies + cross-domain reduction per step); 0 = undivided")
    ap.add_argument("--decomp", action="store_true",
                    help="FIRE only: the paper's domain decomposition (PAPER.md:215-221, 229) instead of replicas: the lattice "
                         "is cut into one z-slab per rank (torchrun: one rank per GPU, NCCL moves halo packages and reduction "
                         "rows between device buffers; parallel.fire_minimize_rank). Total work is fixed: scaling 'strong'. "
                         "With one rank the slab is the whole lattice and its halo wraps onto itself")
    ap.add_argument("--sustained-s", type=float, default=2.0,
                    help="length of the second timed block (seconds of device time) reported as roofline.sustained; 0 = skip")
    ap.add_argument("--eta", type=float, default=0.004)
    ap.add_argument("--mu", type=float, default=0.8)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_1911_07045_b200 import binding as lq, build
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1 or args.decomp:
        import torch.distributed as dist
        if world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29533")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
    build.build()
    K = args.steps if args.steps is not None else 200
    W = args.warmup if args.warmup is not None else 5
    if W < 3:
        W = 3

    c = build_workload(args.workload)
    N = c["N"]
    ctx = lq.lq_create(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"])
    stream = torch.cuda.current_stream()
    lq.lq_set_stream(ctx, stream.cuda_stream)
    lq.lq_set_option(ctx, "fire_path", args.fire_path)
    if c["mask"] is not None:
        lq.lq_set_sites(ctx, c["mask"], c["kind"], c["W"], c["axis"])
    nsim = int(lq.lq_get_info(ctx, "n_simulated"))
    # pinned host staging for the e2e leg
    hq = torch.empty((5, N), dtype=torch.float64, pin_memory=True)
    hq.numpy()[...] = c["q"]
    hout = torch.empty((5, N), dtype=torch.float64, pin_memory=True)
    lq.lq_set_Q(ctx, hq)

    slabs = None
    if args.decomp:
        if args.method != "fire" or args.slabs > 0:
            raise SystemExit("--decomp goes with --method fire and without --slabs")
        from paper_1911_07045_b200 import parallel
        z0, nz = parallel.split_z(c["Lz"], world)[rank]
        mine = parallel.make_slab(lq, c, z0, nz)
        lq.lq_set_stream(mine, stream.cuda_stream)
        lq.lq_set_option(mine, "fire_path", args.fire_path)
        nsim = int(lq.lq_get_info(mine, "n_simulated"))          # this rank's share; summed over ranks below
        comm = parallel.DistComm(dist, rank, world)
        slabs = [mine]

        def minimize(steps):
            return parallel.fire_minimize_rank(lq, mine, comm, steps, 0.0, c["fire"], staging="device")
    elif args.method == "fire" and args.slabs > 0:
        from paper_1911_07045_b200 import parallel
        slabs = parallel.make_slabs(lq, c, args.slabs)
        for s_ in slabs:
            lq.lq_set_stream(s_, stream.cuda_stream)
            lq.lq_set_option(s_, "fire_path", args.fire_path)

        def minimize(steps):
            return lq.lq_slabs_fire_minimize(slabs, steps, 0.0, c["fire"])
    elif args.method == "fire":
        def minimize(steps):
            return lq.lq_fire_minimize(ctx, steps, 0.0, c["fire"])
    elif args.method == "analyze":
        # a "step" = one pass of the director / S / defect-mask kernel over the lattice
        aS = torch.empty(N, dtype=torch.float64, device="cuda")
        aD = torch.empty((3, N), dtype=torch.float64, device="cuda")
        aM = torch.empty(N, dtype=torch.uint8, device="cuda")
        thr = 0.8 * lq.lq_get_S0(ctx)

        def minimize(steps):
            for _ in range(steps):
                lq.lq_analyze_device(ctx, thr, aS, aD, aM)
            return {"steps": steps, "sweep_launches": steps, "launches": steps}
    else:
        meth = lq.LQ_MIN_GD if args.method == "gd" else lq.LQ_MIN_NESTEROV

        def minimize(steps):
            return lq.lq_descent_minimize(ctx, meth, steps, 0.0, args.eta, args.mu)

    # warm-up: W steps (also builds the sweep plan / tensor maps)
    minimize(W)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    rep = minimize(K)
    e1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    assert rep["steps"] == K
    if dist is not None:
        dist.barrier()
    ms_max, units = aggregate(ms, nsim * K, world, dist, torch.device("cuda", local))
    value = units / (ms_max * 1e-3)

    # second timed block, long enough for the board to reach its power-capped clock (the K-step region above can be a
    # sub-100 ms burst at full clock): same call, same accounting, reported beside the headline as roofline.sustained
    sustained = None
    if args.sustained_s > 0 and ms > 0:
        Ks = max(K, int(np.ceil(args.sustained_s * 1e3 / (ms / K))))
        sampler2 = ClockSampler(local)
        sampler2.start()
        torch.cuda.synchronize()
        e0.record(stream)
        rep_s = minimize(Ks)
        e1.record(stream)
        torch.cuda.synchronize()
        clocks2 = sampler2.stop()
        ms_s = e0.elapsed_time(e1)
        loop_s = (rep_s.get("gpu_ms") or ms_s) if isinstance(rep_s, dict) else ms_s
        sustained = {"steps": Ks, "ms_per_step": ms_s / Ks, "loop_ms": loop_s, "sweep_launches": rep_s["sweep_launches"],
                     "sm_mhz": clocks2["sm_mhz"], "reasons": clocks2["reasons"]}

    # e2e: host buffers in, K steps, host buffers out -- all inside the timed region
    e2e = None
    if not args.no_e2e and slabs is None:
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        lq.lq_set_Q(ctx, hq)
        rep2 = minimize(K)
        lq.lq_get_Q(ctx, hout)
        torch.cuda.synchronize()
        t_e2e = (time.perf_counter() - t0) * 1e3
        t_max, units2 = aggregate(t_e2e, nsim * K, world, dist, torch.device("cuda", local))
        e2e = {"value": units2 / (t_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 40.0 * N / K,
               "d2h_bytes_per_step": 40.0 * N / K, "ms_total": t_max,
               "call": "lq_set_Q(pinned host) + %s + lq_get_Q(pinned host)" % (
                   {"fire": "lq_fire_minimize(%d)" % K, "analyze": "%d x lq_analyze" % K}.get(
                       args.method, "lq_descent_minimize(%d)" % K))}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_kind = measured_hbm_peak()
    flag_byte = 1.0 if lq.lq_get_info(ctx, "n_object") > 0 else 0.0
    # FIRE reads + writes q and v (+ flag byte).  GD: read q, write q; Nesterov: read q_k, q_{k-1}, write q_{k+1}
    alg_bytes_site = {"fire": 160.0, "gd": 80.0, "nesterov": 120.0, "analyze": 73.0}[args.method] + flag_byte
    # average duration of one launch of the dominant kernel over the timed region: the library's own CUDA events
    # around its launch loop (on the stream the kernels run on) / launches of that kernel.  Since Algorithm 1's
    # initialisation rides on the first sweep there is nothing else inside those events (masked three-constant
    # lattices: the sweep plus its fix-up launch).  Units per launch = simulated sites.
    loop_ms = rep.get("gpu_ms") or ms
    nlaunch = max(rep["sweep_launches"], 1)
    if slabs is not None:
        nlaunch = max(rep["sweep_launches"] // len(slabs), 1)    # one "launch" = the sweeps of all slabs of one step
    launch_ms = loop_ms / nlaunch
    # on-chip resident kernel (small lattices): ONE launch runs all K steps
    resident = args.method == "fire" and slabs is None and rep["sweep_launches"] == 1 and K > 1
    sites_per_launch = nsim * (K if resident else 1)
    achieved = alg_bytes_site * sites_per_launch / (launch_ms * 1e-3) / 1e9
    design_bytes_site = lq.lq_get_info(ctx, "sweep_bytes_per_site") if args.method == "fire" else alg_bytes_site
    three = c["L2"] != 0 or c["L3"] != 0
    if args.method == "analyze":
        kernel_name = "k_analyze"
    elif args.method != "fire":
        kernel_name = "k_descent" if args.fire_path == 1 else "k_descent_sweep"
    else:
        kernel_name = {1: "k_fire1_force"}.get(args.fire_path, "k_sweep" if (three or args.fire_path == 2) else "k_sweep_rc")
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic_cfg%s%s.json" % (args.workload, "" if args.method == "fire" else "_" + args.method))
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get("dram_bytes_per_launch")
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "peak_kind": peak_kind, "kernel": kernel_name,
                "algorithmic_bytes_per_site": alg_bytes_site, "design_bytes_per_site": design_bytes_site,
                "achieved_design_GBs": design_bytes_site * sites_per_launch / (launch_ms * 1e-3) / 1e9,
                "launch_ms": launch_ms, "launches_timed": rep["sweep_launches"], "sites_per_launch": sites_per_launch}
    # the secondary roof: fp64 FMA rate of this device, measured now by the library's register-only
    # microbenchmark (outside the timed region), and the fp64 work the timed kernel did against it
    if slabs is None:
        try:
            alu = lq.lq_get_info(ctx, "fp64_fma_tflops")
            # ~190 flop per one-constant force + update, ~340 with L2/L3; the recompute sweep
            # evaluates the one-constant force ~2.2 times per site-update (~340); GD / Nesterov drop FIRE's update
            flop_site = {"fire": 340.0, "gd": 300.0 if three else 150.0, "nesterov": 310.0 if three else 160.0,
                         "analyze": 250.0}[args.method]
            roofline["fp64_fma_peak_tflops"] = alu
            roofline["fp64_flop_per_site_estimate"] = flop_site
            roofline["fp64_frac_estimate"] = flop_site * sites_per_launch / (launch_ms * 1e-3) / 1e12 / alu
        except Exception:
            pass
    if sustained is not None:
        nl = max(sustained.pop("sweep_launches") // (len(slabs) if (slabs is not None and not args.decomp) else 1), 1)
        l_ms = sustained.pop("loop_ms") / nl
        per_launch = nsim * (sustained["steps"] if resident else 1)
        sustained["launch_ms"] = l_ms
        sustained["frac"] = alg_bytes_site * per_launch / (l_ms * 1e-3) / 1e9 / peak
        sustained["note"] = "same call run for >= %.1f s of device time right after the timed region (power-capped clock)" % args.sustained_s
        roofline["sustained"] = sustained
    if resident:
        roofline["kernel"] = "k_fire_resident"
        roofline["note"] = ("state resident on chip: the algorithmic bytes never touch HBM, the step is bound by its grid "
                            "barrier; no roofline claim (SURVEY 8(d): configs 1-2 are latency-bound)")

    cpu = None
    if not args.no_cpu_baseline:
        v, cores, desc, _, _ = time_oracle(c, target_s=15.0, crop=args.ref_crop, method=args.method, eta=args.eta, mu=args.mu)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

    metric = METRIC if args.method == "fire" else METRIC.replace("FIRE", {"gd": "gradient-descent", "nesterov": "Nesterov", "analyze": "director/S/defect analysis"}[args.method])
    line = {"metric": metric, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "strong" if args.decomp else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": c["name"], "lattice": [c["Lx"], c["Ly"], c["Lz"]], "n_simulated": nsim,
                       "elastic": "L1" if c["L2"] == 0 and c["L3"] == 0 else "L1+L2+L3",
                       "l2": "inputs_larger_than_L2" if 120.0 * N > 126e6 * 4 else "L2_resident_no_flush",
                       "multi_gpu": "z-slabs" if args.decomp else "replicas only", "fire_path": args.fire_path, "method": args.method,
                       "z_slabs_on_this_gpu": args.slabs},
            "clocks": clocks, "e2e": e2e, "gpu_launches": rep["launches"], "roofline": roofline,
            "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
