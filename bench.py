"""bench.py -- BASELINE.json's metric on its named workload, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3|1|2|4|5]

A "step" is one pass of the whole hot path over one batch of synthetic input: one gn_transport_run of the
workload (config 3 by default: 64^3 voxel phantom, 1e7 photons of 6 MeV from a 5-degree cone, fp32 -- the
configuration BASELINE.json's north_star quotes the target on), or for config 5 one gn_nav_locate +
gn_nav_compute_step over the query batch.  metric = transported photon steps/s (ComputeStep queries/s for
config 5).  Multi-GPU (torchrun, one rank per GPU): weak scaling, every rank transports its own contiguous
photon-id range of the same size on a replicated geometry; the per-volume tally is all-reduced (NCCL) at the
end of each step, inside the timed region.
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
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

import numpy as np  # noqa: E402

ALGO_BYTES = {("transport", 32): 96.0, ("transport", 64): 160.0, ("nav", 32): 64.0, ("nav", 64): 116.0}
# Algorithmic flops per step (configs 1-4) / per query (config 5): operation count of the oracle's algorithm on the config's own
# workload, measured with the oracle's counting Real (SURVEY 8(d) "instrumented oracle": + - * / sqrt compare = 1, fma = 2,
# transcendental = 1).  bench.py re-measures it in the cpu_baseline leg; these are the committed values of that measurement
# (oracle.transport_count_ops on the first 20000 photons / oracle.nav_count_ops on 20000 queries), used with --no-cpu-baseline.
ALGO_FLOPS = {1: 371.4, 2: 469.6, 3: 606.5, 4: 582.4, 5: 841.9}
PIPE_PEAK_FALLBACK = {32: 74.4, 64: 37.2}   # nominal TFLOP/s (148 SMs x 128 / 64 lanes x 2 x 1.965 GHz) when the self-test cannot run


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        self.lines, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


def workload(k):
    from paper_1209_5235_b200 import workloads as W
    wl = W.config(k)
    precision = 32 if 32 in wl.precisions else 64
    return wl, precision


# ------------------------------------------------------------------------------------------------ reference arm
def _oracle_worker(args):
    k, precision, first, count = args
    import oracle
    from paper_1209_5235_b200 import workloads as W
    wl = W.config(k)
    og = oracle.OracleGeometry(wl.geometry)
    t = time.perf_counter()
    if wl.source is not None:
        r = og.transport(wl.source, wl.seed, count, precision, first_id=first)
        units = r["stats"]["n_steps"]
    else:
        R = np.float32 if precision == 32 else np.float64
        pos, dirs = W.nav_queries(wl.geometry, count, seed=wl.seed, dtype=R, first=first)
        t = time.perf_counter()
        vol = og.locate(pos, dirs, precision); og.compute_step(pos, dirs, vol, None, precision)
        units = count
    return units, time.perf_counter() - t


def oracle_rate(k, precision, sample, cores=1):
    """units/s of the oracle as it stands on `cores` host cores (independent workers over disjoint id ranges,
    as the paper's OpenMP-over-particles version)."""
    if cores == 1:
        units, dt = _oracle_worker((k, precision, 0, sample))
        return units / dt, units, dt
    import multiprocessing as mp
    per = sample // cores
    with mp.get_context("spawn").Pool(cores) as pool:
        t = time.perf_counter()
        res = pool.map(_oracle_worker, [(k, precision, i * per, per) for i in range(cores)])
        wall = time.perf_counter() - t
    units = sum(u for u, _ in res)
    dt = max(d for _, d in res)            # excludes geometry construction, like the GPU side
    return units / dt, units, wall


def oracle_flops_per_unit(k, n_sample):
    """Flops per step / query of config k from the instrumented oracle (counting Real), on the first n_sample units."""
    import oracle
    from paper_1209_5235_b200 import workloads as W
    wl = W.config(k)
    og = oracle.OracleGeometry(wl.geometry)
    if wl.source is not None:
        c, st = og.transport_count_ops(wl.source, wl.seed, n_sample)
        return c["flops"] / max(1, st["n_steps"]), {n: v / max(1, st["n_steps"]) for n, v in c.items()}
    pos, dirs = W.nav_queries(wl.geometry, n_sample, seed=wl.seed)
    c = og.nav_count_ops(pos, dirs)
    return c["flops"] / n_sample, {n: v / n_sample for n, v in c.items()}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl, precision = workload(args.config)
    sample = {1: 10000, 2: 20000, 3: 100000, 4: 50000, 5: 300000}[args.config]
    _oracle_worker((args.config, precision, 0, max(1, sample // 10)))          # page in, build lib
    times, units = [], 0
    for _ in range(args.warmup):
        _oracle_worker((args.config, precision, 0, max(1, sample // 10)))
    for s in range(args.steps):
        u, dt = _oracle_worker((args.config, precision, s * sample, sample))
        units += u; times.append(dt)
    total = sum(times)
    value = units / total
    unit = "photon-steps/s" if wl.source is not None else "ComputeStep queries/s"
    line = {"impl": "reference", "metric": "transported photon steps/s" if wl.source is not None else "ComputeStep queries/s",
            "value": value, "unit": unit, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if precision == 32 else "f64", "data": "synthetic",
            "config": {"workload": wl.name, "precision": precision, "sample_per_step": sample},
            "cpu_baseline": {"value": value, "unit": unit, "cores": 1, "kind": "oracle",
                             "sample": f"{sample} of {wl.n} {'photons' if wl.source is not None else 'queries'} per step, single thread"},
            "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ the paper's own benchmark
PAPER_TABLE1 = {  # PAPER.md Table 1 (L176-181): execution time [ms] of phase 5 for N = 1e5 particles
    "random": {"cpu_1_thread_ms": 458.0, "cpu_12_threads_ms": 56.0, "gpu_gtx470_ms": 114.0},
    "regular": {"cpu_1_thread_ms": 442.0, "cpu_12_threads_ms": 54.0, "gpu_gtx470_ms": 33.0},
}


def freepath_inputs(which, precision, scale):
    from paper_1209_5235_b200 import workloads as W
    R = np.float32 if precision == 32 else np.float64
    if which == "random":
        pos, d, Y = W.random_particles(int(100000 * scale), seed=11, dtype=R)
    else:
        pos, d, Y = W.regular_particles(400, max(1, int(250 * scale)), dtype=R)
    return W.spheres_geometry(), pos, d, Y, W.MU_MASS_AL_1MEV


def run_freepath(args):
    """Configs 6 / 7: Algorithm 2 phase 5 on the Spheres geometry, N = 1e5 (x --scale).  A step = one
    gn_free_path_run over the whole particle set.  Context beside PAPER.md Table 1, not a BASELINE.json config."""
    which = "random" if args.config == 6 else "regular"
    precision = args.precision or 64                          # the paper's port is double-based
    geom, pos, d, Y, mu_mass = freepath_inputs(which, precision, args.scale)
    n = pos.shape[0]
    unit = "free paths/s"
    name = f"spheres_{which}"
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return 0
        import oracle
        og = oracle.OracleGeometry(geom)
        m = min(n, 20000)
        og.free_path(pos[:200], d[:200], Y[:200], mu_mass, precision)
        t = []
        for s_ in range(args.steps):
            lo = (s_ * m) % max(1, n - m + 1)
            t0 = time.perf_counter(); og.free_path(pos[lo:lo + m], d[lo:lo + m], Y[lo:lo + m], mu_mass, precision); t.append(time.perf_counter() - t0)
        v = m * args.steps / sum(t)
        print(json.dumps({"impl": "reference", "metric": "free paths/s (Algorithm 2 phase 5)", "value": v, "unit": unit, "n_gpus": args.gpus, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": 1e3 * sum(t) / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                          "dtype": "f32" if precision == 32 else "f64", "data": "synthetic", "config": {"workload": name, "precision": precision, "sample_per_step": m},
                          "cpu_baseline": {"value": v, "unit": unit, "cores": 1, "kind": "oracle", "sample": f"{m} of {n} particles per step, single thread"},
                          "e2e": {"value": v, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return 0
    import torch
    from paper_1209_5235_b200 import binding as B, build as lib_build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        lib_build.build()
    if world > 1:
        dist.barrier()
    dev = torch.device("cuda", local)
    geo = B.Geometry(geom)
    tp, td, tY = (torch.from_numpy(a).to(dev) for a in (pos, d, Y))
    T = torch.empty(n, dtype=tp.dtype, device=dev)
    for _ in range(max(args.warmup, 3)):
        B.free_path_run(geo, tp, td, tY, mu_mass, out=T, nsteps=False)
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * args.steps)]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2: written between timed runs
    for s_ in range(args.steps):
        flush.fill_(s_ & 255)
        ev[2 * s_].record()
        B.free_path_run(geo, tp, td, tY, mu_mass, out=T, nsteps=False)
        ev[2 * s_ + 1].record()
    torch.cuda.synchronize()
    ms = sum(ev[2 * s_].elapsed_time(ev[2 * s_ + 1]) for s_ in range(args.steps))
    tt = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX); ms = tt.item()
    clocks = sampler.stop() if rank == 0 else None
    # end to end = Algorithm 2 phases 4-6: host buffers in, T back on the host
    hp, hd, hY = (torch.from_numpy(a).pin_memory().numpy() for a in (pos, d, Y))
    B.free_path_run_host(geo, hp, hd, hY, mu_mass, precision)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        B.free_path_run_host(geo, hp, hd, hY, mu_mass, precision)
    e2e_dt = time.perf_counter() - t0
    if rank == 0:
        rs = 4 if precision == 32 else 8
        abytes = 8 * rs                                       # 3 + 3 + 1 Real in, 1 Real out per particle
        peak, peak_src = measured_peaks()
        achieved = n * abytes / (ms / args.steps * 1e-3) / 1e9
        cpu = None
        if not args.no_cpu_baseline:
            import oracle
            og = oracle.OracleGeometry(geom); m = min(n, 60000)
            t0 = time.perf_counter(); og.free_path(pos[:m], d[:m], Y[:m], mu_mass, precision); dt = time.perf_counter() - t0
            cpu = {"value": m / dt, "unit": unit, "cores": 1, "kind": "oracle", "sample": f"first {m} of {n} particles of {name}, fp{precision}, {dt:.1f} s"}
        line = {"metric": "free paths/s (Algorithm 2 phase 5)", "value": world * n * args.steps / (ms * 1e-3), "unit": unit, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if precision == 32 else "f64", "data": "synthetic",
                "config": {"workload": name, "precision": precision, "particles_per_gpu": n, "volumes": geo.n_places, "l2": "256 MB buffer written between timed runs (L2 flush)",
                           "parallelism": f"dp{world} (replicas)"},
                "clocks": clocks, "gpu_launches": args.steps,
                "e2e": {"value": world * n * args.steps / e2e_dt, "unit": unit, "h2d_bytes_per_step": 7 * rs * n, "d2h_bytes_per_step": (rs + 4) * n,
                        "note": "Algorithm 2 phases 4-6: particle states and lifetimes from pinned host memory, T (and step counts) back to the host"},
                "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                             "kernel": "free_path_kernel", "algorithmic_bytes_per_unit": abytes,
                             "note": "one thread walks one particle to completion (latency-bound at N = 1e5: 0.4 resident warps per scheduler)"},
                "cpu_baseline": cpu,
                "paper_table1": dict(PAPER_TABLE1[which], note="PAPER.md Table 1, N = 1e5, GTX 470 / 2 x Opteron 2427; context, other hardware, ball radius not printed in the paper")}
        print(json.dumps(line))
    if world > 1:
        dist.barrier(); dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1209_5235_b200 import binding as B, build as lib_build, workloads as W
    from paper_1209_5235_b200.sharding import allreduce_tally
    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        lib_build.build()
    if world > 1:
        dist.barrier()
    wl, precision = workload(args.config)
    if args.precision:
        precision = args.precision
    n = int(wl.n * args.scale)
    gopts = {}
    if args.steps_per_pass:
        gopts["steps_per_pass"] = args.steps_per_pass
    if args.tail_photons:
        gopts["tail_photons"] = args.tail_photons
    if args.first_pass_steps:
        gopts["first_pass_steps"] = args.first_pass_steps
    if args.regroup_percent:
        gopts["regroup_percent"] = args.regroup_percent
    if args.secondaries:
        gopts["secondaries"] = 1
    if args.refill:
        gopts["refill"] = 1
    geo = B.Geometry(wl.geometry, **gopts)
    transport = wl.source is not None
    dom = [0, 0.0]                                            # dominant kernel: steps taken in / summed duration of the lean step passes
    first_id = rank * n                                       # weak scaling: same work per GPU, disjoint ids
    dev = torch.device("cuda", local)
    if transport:
        edep = torch.empty(geo.n_places, dtype=torch.float64, device=dev)

        def step():
            r = B.transport_run(geo, wl.source, wl.seed, n, precision, first_photon_id=first_id, edep=edep)
            st = r["stats"]
            if world > 1:
                allreduce_tally(edep, st)
            dom[0] += st["n_steps_step_pass"]; dom[1] += st["step_pass_ms"]
            return st["n_steps"], st["n_kernel_launches"], st["kernel_ms"]
    else:
        rdt = torch.float32 if precision == 32 else torch.float64
        pos, dirs = W.nav_queries_torch(wl.geometry, n, wl.seed + 1000 * rank, rdt, dev)
        vol = torch.empty(n, dtype=torch.int32, device=dev)
        out = (torch.empty(n, dtype=rdt, device=dev), torch.empty(n, dtype=torch.int32, device=dev))
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]

        def step():
            ev[0].record()
            B.nav_locate(geo, pos, dirs, out=vol)
            B.nav_compute_step(geo, pos, dirs, vol, out=out)
            ev[1].record(); ev[1].synchronize()
            # locate_levels_kernel, sort_keys_kernel, sort_scatter_kernel, step_distance_kernel, sort_scatter_kernel, step_relocate_kernel
            return n, 6, ev[0].elapsed_time(ev[1])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3) if not args.allow_short_warmup else args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    units = launches = 0; kernel_ms = 0.0
    dom[0], dom[1] = 0, 0.0
    e0.record()
    for _ in range(args.steps):
        u, l, km = step()
        units += u; launches += l; kernel_ms += km
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    t = torch.tensor([ms, float(units), float(launches), kernel_ms], dtype=torch.float64, device=dev)
    if world > 1:
        tmax = t.clone(); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        tsum = t.clone(); dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
        ms, units, launches = tmax[0].item(), tsum[1].item(), tsum[2].item()
    clocks = sampler.stop() if rank == 0 else None

    # ---- end to end through the host-buffer C-ABI call (H2D / D2H inside the timed region)
    e2e = None
    if transport:
        cs_bytes = 88
        B.transport_run_host(geo, wl.source, wl.seed, n, precision, first_photon_id=first_id)      # untimed: the GPU idled while the clock sampler stopped
        t0 = time.perf_counter(); u2 = 0
        for _ in range(args.steps):
            r = B.transport_run_host(geo, wl.source, wl.seed, n, precision, first_photon_id=first_id)
            u2 += r["stats"]["n_steps"]
        dt = time.perf_counter() - t0
        e2e_val = torch.tensor([u2 / dt], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(e2e_val, op=dist.ReduceOp.SUM)
        e2e = {"value": e2e_val.item(), "unit": "photon-steps/s", "h2d_bytes_per_step": cs_bytes, "d2h_bytes_per_step": geo.n_places * 8 + 136,
               "note": "inputs of a run are the source description and the seed; the per-volume tally and stats come back to the host"}
    else:
        m = min(n, 1 << 24)
        R = np.float32 if precision == 32 else np.float64
        hp = torch.empty((m, 3), dtype=rdt).pin_memory(); hd = torch.empty((m, 3), dtype=rdt).pin_memory()
        hp.copy_(pos[:m]); hd.copy_(dirs[:m])
        hout = (torch.empty(m, dtype=torch.int32).pin_memory().numpy(), torch.empty(m, dtype=rdt).pin_memory().numpy(),
                torch.empty(m, dtype=torch.int32).pin_memory().numpy())
        B.nav_query_host(geo, hp.numpy(), hd.numpy(), precision, out=hout)          # untimed: sizes the handle's staging area
        reps = 3
        t0 = time.perf_counter()
        for _ in range(reps):
            B.nav_query_host(geo, hp.numpy(), hd.numpy(), precision, out=hout)
        dt = (time.perf_counter() - t0) / reps
        rs = 4 if precision == 32 else 8
        e2e = {"value": world * m / dt, "unit": "ComputeStep queries/s", "h2d_bytes_per_step": 6 * rs * m, "d2h_bytes_per_step": (8 + rs) * m,
               "note": f"{m} queries per call, inputs from and results to page-locked host memory, chunks of 2^22 on two streams"}

    pipe = None
    if rank == 0:
        try:
            pipe = B.selftest_pipe_peak(precision)            # FFMA / DFMA pipe peak at the clock of this run (after the timed region)
        except Exception:
            pipe = None
    if rank == 0:
        peak, peak_src = measured_peaks()
        kind = "transport" if transport else "nav"
        abytes = ALGO_BYTES[(kind, precision)]
        cpu = None
        flops_per_unit, flops_src, op_mix = ALGO_FLOPS[args.config], "committed measurement of the instrumented oracle (bench.py ALGO_FLOPS)", None
        if not args.no_cpu_baseline:
            sample = {1: 10000, 2: 100000, 3: 1500000, 4: 400000, 5: 20000000}[args.config]
            v1, u1, d1 = oracle_rate(args.config, precision, sample, 1)
            cpu = {"value": v1, "unit": "photon-steps/s" if transport else "ComputeStep queries/s", "cores": 1, "kind": "oracle",
                   "sample": f"first {sample} of {wl.n} {'photons' if transport else 'queries'} of {wl.name}, fp{precision}, {d1:.1f} s"}
            if args.cpu_all_cores:
                nc = os.cpu_count() or 1
                vN, uN, dN = oracle_rate(args.config, precision, sample * min(nc, 8), nc)
                cpu["all_cores"] = {"value": vN, "cores": nc, "wall_s": dN}
            flops_per_unit, op_mix = oracle_flops_per_unit(args.config, 20000)
            flops_src = "instrumented oracle (counting Real) on the first 20000 units of this workload, this run"
        pipe_tflops = pipe["tflops"] if pipe else PIPE_PEAK_FALLBACK[precision]
        pipe_src = f"gn_selftest_pipe_peak ({'FFMA' if precision == 32 else 'DFMA'} chains, {pipe['sm_mhz']:.0f} MHz)" if pipe else "nominal (self-test unavailable)"
        # per-unit roofline: the slower of algorithmic bytes at HBM bandwidth and algorithmic flops at pipe peak
        t_hbm, t_alu = abytes / (peak * 1e9), flops_per_unit / (pipe_tflops * 1e12)
        bound = "hbm" if t_hbm >= t_alu else "alu"

        def fracs(rate):                                       # units / s -> (frac_hbm, frac_alu)
            return (rate * t_hbm, rate * t_alu) if rate else (None, None)
        whole_rate = (units / world) / (kernel_ms * 1e-3) if kernel_ms > 0 else None
        # dominant kernel = the lean step pass (voxel_pass for phantoms): steps taken inside its timed launches / their summed
        # CUDA-event durations (one event pair per launch on the launching stream, inside gn_transport_run)
        dom_rate = dom[0] / (dom[1] * 1e-3) if (transport and dom[1] > 0) else whole_rate
        dh, da = fracs(dom_rate); wh, wa = fracs(whole_rate)
        traffic = None
        tpath = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tpath):
            try:
                traffic = json.load(open(tpath)).get(f"{wl.name}_fp{precision}")
            except Exception:
                traffic = None
        traffic_note = None
        if isinstance(traffic, dict):                          # per launch of the dominant kernel, from the committed ncu capture
            traffic, traffic_note = traffic.get("dram_bytes_per_launch"), traffic.get("note")
        if bound == "hbm":
            ach, pk, un, fr = (dom_rate * abytes / 1e9 if dom_rate else None), peak, "GB/s", dh
        else:
            ach, pk, un, fr = (dom_rate * flops_per_unit / 1e12 if dom_rate else None), pipe_tflops, "TFLOP/s", da
        voxel = transport and wl.name.startswith(("config3", "config2"))      # geometries of regular voxels / slabs run the voxel schedule (gn_geometry::voxel_sched)
        roofline = {"bound": bound, "achieved": ach, "peak": pk, "unit": un, "frac": fr, "traffic": traffic,
                    "peak_source": peak_src if bound == "hbm" else pipe_src,
                    "kernel": ("voxel_pass (regular-voxel step pass)" if voxel else "transport_pass<R,0,0,0> (lean wavefront step pass)") if transport else "locate_levels_kernel + query sort + step_distance_kernel + step_relocate_kernel",
                    "algorithmic_bytes_per_unit": abytes, "flops_per_unit": flops_per_unit, "flops_source": flops_src,
                    "hbm_peak_gbs": peak, "pipe_peak_tflops": pipe_tflops, "pipe_peak_source": pipe_src,
                    "frac_hbm": dh, "frac_alu": da,
                    "kernel_steps_per_run": dom[0] / args.steps if transport else None, "kernel_ms_per_run": dom[1] / args.steps if transport else kernel_ms / args.steps,
                    "whole_run": {"frac": wh if bound == "hbm" else wa, "frac_hbm": wh, "frac_alu": wa, "ms_per_run": kernel_ms / args.steps,
                                  "note": "all kernels of a run: units of the run / CUDA-event time of the whole launch sequence"},
                    "note": "bound = the slower of (algorithmic bytes / measured HBM bandwidth) and (algorithmic flops / measured pipe peak) per unit; "
                            "a fraction above 1 on the HBM leg means the kernel does not move the algorithmic bytes: a pass keeps the photon in registers "
                            "for up to K steps, so the record is read and written once per pass, not once per step (traffic = ncu dram bytes of one launch of the dominant kernel, profiles/traffic.json)"}
        if traffic_note:
            roofline["traffic_note"] = traffic_note
        if op_mix:
            roofline["ops_per_unit"] = op_mix
        line = {"metric": "transported photon steps/s" if transport else "ComputeStep queries/s",
                "value": units / (ms * 1e-3), "unit": "photon-steps/s" if transport else "ComputeStep queries/s",
                "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if precision == 32 else "f64", "data": "synthetic",
                "config": {"workload": wl.name, "precision": precision, ("photons_per_gpu" if transport else "queries_per_gpu"): n,
                           "volumes": geo.n_places, "l2": "photon state queues (2 x %d MB) exceed the 126 MB L2; no explicit flush" % (n * (64 if precision == 32 else 112) // 10 ** 6)
                           if transport else "query arrays (%d MB) exceed the 126 MB L2" % (n * 6 * (4 if precision == 32 else 8) // 10 ** 6),
                           "parallelism": f"dp{world} (photon-id ranges, replicated geometry)", **({"secondaries": 1} if args.secondaries else {}), **({"refill": 1} if args.refill else {})},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
                "units_per_step": units / args.steps / world}
        print(json.dumps(line))
    if world > 1:
        dist.barrier(); dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5, 6, 7],
                    help="1-5: BASELINE.json configs; 6 / 7: the paper's own benchmark, Spheres geometry with the Random / Regular set")
    ap.add_argument("--precision", type=int, default=0, choices=[0, 32, 64])
    ap.add_argument("--scale", type=float, default=1.0, help="fraction of the workload's photons/queries (diagnostics only)")
    ap.add_argument("--steps-per-pass", type=int, default=0)
    ap.add_argument("--tail-photons", type=int, default=0, help="diagnostics: override gn_opts.tail_photons")
    ap.add_argument("--first-pass-steps", type=int, default=0, help="diagnostics: override gn_opts.first_pass_steps")
    ap.add_argument("--regroup-percent", type=int, default=0, help="diagnostics: override gn_opts.regroup_percent")
    ap.add_argument("--secondaries", action="store_true",
                    help="variant (not BASELINE.json's workload): gn_opts.secondaries = 1, annihilation photons of pair events are transported; no cpu_baseline leg")
    ap.add_argument("--refill", action="store_true",
                    help="variant: gn_opts.refill = 1, the paper's refill scheduling (PAPER.md L195) as one persistent kernel instead of the wavefront passes")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-all-cores", action="store_true")
    ap.add_argument("--allow-short-warmup", action="store_true")
    args = ap.parse_args()
    if args.secondaries:
        args.no_cpu_baseline = True
    if args.config in (6, 7):
        return run_freepath(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
