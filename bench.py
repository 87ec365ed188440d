#!/usr/bin/env python
"""bench.py -- headline benchmark of BASELINE.json: Metropolis spin-flip attempts/s at
L=4096, q=8, sigma=0.3, 128 replicas (configs[3]), swap event every sweep.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--variant auto|direct|field]
                  [--workload cfg3|cfg4|paper:L[:R]]

One STEP = one sweep of every replica (L Metropolis steps each, Eq. 8) + the per-slot observables +
one replica-exchange event (Eq. 9) = n_rep*L attempts, i.e. one pass of the whole hot path.  The
default K = 2000 is the full configs[3] run.  Prints ONE JSON line (rank 0).  For N > 1 (torchrun)
every rank runs its own ensemble of configs[3] (ens_base = rank: independent random streams, no
data-path collective), so scaling is "weak" and `value` is the sum over ranks / max time.
`--workload paper:L` (not the headline) times the same path on the shape of the paper's own
benchmark runs instead: q=3, 400 replicas on a uniform ladder, L in 512..10240 (
inputs.paper_benchmark; `paper:L:R` takes R replicas instead of 400, the replica-count scan of Fig. 5, :224), and says
so in `metric` and `config.workload`.
"""
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

from paper_1308_5426_b200 import inputs  # noqa: E402

METRIC = "Metropolis spin-flip attempts/s at L=4096 q=8 128 replicas"
UNIT = "attempts/s"
# ALU roofline: the algorithmic work of one attempt is L pair terms, each ONE integer
# multiply-accumulate (16-bit coupling half x 8-bit weight); IDP.2A does two of them per lane and issues at a measured
# 64 lanes/clk/SM on the FMA-heavy pipe (profiles/r1_a_direct_v1a.md), so peak = 148 SMs x 64 x 2 MAC x f_SM.
IDP_LANES_PER_CLK_PER_SM = 64    # fallback only: the line carries the rate pt_measure_peaks measured in this run
MACS_PER_IDP_LANE = 2
# dram__bytes_read.sum + dram__bytes_write.sum of ONE persistent sweep_direct_kernel launch on configs[3], from ncu
# --set full captures of a 20-sweep and a 40-sweep launch (profiles/r2_a_headline.md): a fixed part (couplings, spins,
# ladder, permutation: read once) plus a part per sweep (energies and arrival counters of the swap events)
DRAM_BYTES_PER_LAUNCH_FIXED = 412.7e3
DRAM_BYTES_PER_SWEEP = 0.165e3
N_SM = 148


_JSON_OUT = sys.stdout   # main() points this at the process's original stdout


def emit(line):
    _JSON_OUT.write(json.dumps(line) + "\n")
    _JSON_OUT.flush()


def pick_workload(args):
    if args.workload in ("cfg3", "configs[3]"):
        return inputs.config(3)
    if args.workload in ("cfg0", "cfg1", "cfg2"):
        return inputs.config(int(args.workload[3]))
    if args.workload.count(":") == 3 and not args.workload.startswith("paper:"):   # L:q:sigma:R, geometric T in [0.6, 2.5]
        L, q, sigma, R = args.workload.split(":")
        return inputs.Workload("custom[L=%s,q=%s,sigma=%s,R=%s]" % (L, q, sigma, R), int(L), int(q), float(sigma), 1,
                               int(R), 0.6, 2.5, 1000, seed=inputs.SEED_BASE + 0x900 + int(L))
    if args.workload.startswith("paper:"):
        parts = args.workload.split(":")
        return inputs.paper_benchmark(int(parts[1]), int(parts[2]) if len(parts) > 2 else 400)
    raise SystemExit("bench.py: --workload must be cfg0..cfg4, paper:L, paper:L:R or L:q:sigma:R")


def label(w):
    if w.name.startswith("cfg"):
        return "configs[%s]" % w.name[3] + ("" if w.name == "cfg3" else " (not the headline config)")
    if w.name.startswith("custom"):
        return "custom shape (not BASELINE's config)"
    return "the paper's benchmark shape (PAPER.md:136,202; not BASELINE's config)"


def metric_name(w):
    return METRIC if w.name == "cfg3" else "Metropolis spin-flip attempts/s at L=%d q=%d %d replicas" % (w.L, w.q, w.n_rep)


def workload_config(w, variant, n_gpus):
    return {"workload": "%s: L=%d q=%d sigma=%.1f, 1 ensemble x %d replicas per GPU, T %s in "
                        "[%.1f,%.1f], hot start, swap every sweep"
                        % (label(w), w.L, w.q, w.sigma, w.n_rep, w.ladder, w.T_lo, w.T_hi),
            "step": "1 sweep of all replicas + observables + 1 swap event = %d attempts per GPU" % (w.L * w.n_rep),
            "variant": variant, "parallelism": "ensembles sharded over %d GPU(s), no collective" % n_gpus,
            "l2": "not flushed: per-step state is %d KB of packed spins per GPU, resident in shared memory/L2 by "
                  "design; the path is ALU-bound, not HBM-bound" % (w.n_rep * w.L // 2 // 1024)}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML during the timed region."""
    REASONS = {0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x10: "sync_boost",
               0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
               0x100: "display_clock_setting"}

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.mask, self.max_mhz, self.err = index, False, [], 0, None, None
        self.ready, self.first = threading.Event(), 0

    def run(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
            self.ready.set()
            while True:   # at least one sample, also for a timed region shorter than the sampling period
                self.sm.append(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                self.mask |= int(pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                if self.stop_flag:
                    break
                time.sleep(0.01)
        except Exception as ex:  # NVML missing: report, do not fake
            self.err = repr(ex)
        self.ready.set()

    def start_sampling(self):
        """Starts the thread and returns once NVML is initialised, so that the timed region is not over before the
        first sample (nvmlInit takes tens of milliseconds)."""
        self.start()
        self.ready.wait(timeout=5.0)
        self.first = len(self.sm)   # samples from here on lie in the timed region (or just after its end)

    def result(self):
        self.stop_flag = True
        self.join(timeout=2.0)
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "error": self.err}
        sm = self.sm[self.first:] or self.sm[-1:]
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": self.max_mhz, "samples": len(sm),
                "reasons": [n for b, n in self.REASONS.items() if self.mask & b]}


def measured_hbm_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except Exception:
        return 6650.0   # fallback stated in the profiling guide


def oracle_threads():
    return max(1, os.cpu_count() or 1)


def time_oracle_step(o, replicas_done_per_step, threads):
    t0 = time.perf_counter()
    o.sweeps(1, 1, field=False, threads=threads)
    return time.perf_counter() - t0


def cpu_baseline_leg(w, budget_s=12.0):
    """The oracle as it stands (direct O(L) sum per step, the paper's way), all host cores, full configs[3]
    ensemble, as many sweeps as fit the budget (at least 1)."""
    from oracle import pt_oracle
    threads = oracle_threads()
    o = pt_oracle.Oracle(w.L, w.q, w.sigma, 1, w.n_rep, inputs.betas(w), w.seed)
    n, t = 0, 0.0
    while n < 1 or (t < budget_s and n < 64 and t + t / n < 2.5 * budget_s):
        t += time_oracle_step(o, w.n_rep, threads)
        n += 1
    o.close()
    return {"value": n * w.n_rep * w.L / t, "unit": UNIT, "cores": min(threads, w.n_rep), "kind": "oracle",
            "sample": "%d sweep(s) (+swap events) of the full %s ensemble (%d replicas), direct-sum mode, "
                      "%d std::threads, g++ -O2, %.1f s" % (n, label(w), w.n_rep, min(threads, w.n_rep), t)}


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host cores; a step = one sweep (+swap event) of a bounded
    sample of r evenly spaced slots of configs[3]."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import pt_oracle
    pt_oracle.build()
    w = pick_workload(args)
    threads = oracle_threads()
    betas = inputs.betas(w)
    # calibrate on one replica, then size the sample so that (K+W) steps take <= ~150 s
    o1 = pt_oracle.Oracle(w.L, w.q, w.sigma, 1, 1, betas[:1], w.seed)
    t1 = time_oracle_step(o1, 1, 1)
    o1.close()
    total_steps = args.steps + args.warmup
    per_step_budget = 150.0 / max(1, total_steps)
    r = int(per_step_budget / t1 * min(threads, w.n_rep) * 0.7)
    r = max(1, min(w.n_rep, r))
    idx = np.unique(np.linspace(0, w.n_rep - 1, r).round().astype(int))
    r = len(idx)
    use_threads = min(threads, r)
    o = pt_oracle.Oracle(w.L, w.q, w.sigma, 1, r, betas[idx], w.seed)
    for _ in range(args.warmup):
        time_oracle_step(o, r, use_threads)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.sweeps(1, 1, field=False, threads=use_threads)
    dt = time.perf_counter() - t0
    o.close()
    value = args.steps * r * w.L / dt
    sample = ("each step = 1 sweep + swap event of %d of the %d slots of %s (evenly spaced in the ladder), "
              "direct-sum mode, %d std::threads" % (r, w.n_rep, label(w), use_threads))
    line = {"impl": "reference", "metric": metric_name(w), "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32",
            "data": "synthetic", "config": workload_config(w, "oracle", args.gpus),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": use_threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    emit(line)
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1308_5426_b200 import build as ptbuild
    ptbuild.build()
    from paper_1308_5426_b200 import pt, shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libpt has no CPU path")
    torch.cuda.set_device(local_rank)
    # under torch.distributed.run (RANK set) the process group is always used, also for one rank, so that a
    # single-GPU launch exercises the same barrier / max-over-ranks code as N > 1
    use_dist = world > 1 or "RANK" in os.environ
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    w = pick_workload(args)
    betas = inputs.betas(w)
    K, W_ = args.steps, args.warmup
    ens_base, n_ens_local = shard.ensemble_shard(world, world, rank)   # one configs[3] ensemble per GPU
    g = pt.PT(w.L, w.q, w.sigma, n_ens_local, w.n_rep, betas, w.seed, ens_base=ens_base, variant=args.variant)
    variant = g.get_variant()
    peaks = pt.measure_peaks()   # instruction rates per SM and clock, measured now: ~1 s
    stream = torch.cuda.Stream()
    g.use_torch_stream(stream)

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K steps = K sweeps, a swap event after each ----
    with torch.cuda.stream(stream):
        g.sweeps_async(W_, w.swap_every)
        g.sync()
        barrier()
        sampler = ClockSampler(local_rank)
        sampler.start_sampling()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        launches = g.sweeps_async(K, w.swap_every)
        ev1.record(stream)
        g.sync()
        barrier()
        clocks = sampler.result()
    ms = ev0.elapsed_time(ev1)
    if use_dist:
        ms = shard.max_over_ranks(ms, dist, device="cuda")
    attempts_per_gpu = K * w.n_rep * w.L
    value = world * attempts_per_gpu / (ms * 1e-3)
    obs = g.observables()
    acc = float(obs["flip_accepts"].sum()) / float(obs["flip_attempts"].sum())

    # ---- end to end through the C ABI with host buffers: upload a start configuration, K steps, read back ----
    start, E0, _, sweep0 = g.get_state()
    barrier()
    t0 = time.perf_counter()
    g.set_state(start, E0, None, sweep0)     # H2D: n_rep*L bytes of spins + n_rep*8 bytes of energies (pinned staging)
    g.sweeps(K, w.swap_every)
    spins = g.get_spins()                    # D2H: n_rep*L bytes
    E = g.energy()                           # D2H: n_rep*8 bytes
    ob = g.observables()                     # D2H: n_rep*144 bytes
    barrier()
    e2e_s = time.perf_counter() - t0
    if use_dist:
        e2e_s = shard.max_over_ranks(e2e_s, dist, device="cuda")
    assert spins.shape == start.shape and E.size == w.n_rep and ob["n_samples"].min() > 0
    e2e = {"value": world * attempts_per_gpu / e2e_s, "unit": UNIT,
           "h2d_bytes_per_step": (start.nbytes + E0.nbytes) / K,
           "d2h_bytes_per_step": (spins.nbytes + E.nbytes + w.n_rep * 144) / K,
           "what": "pt_set_state(host spins + energies) + pt_sweeps(K) + pt_get_spins + pt_energy + pt_observables "
                   "(host buffers), wall clock"}

    if rank == 0:
        f_hz = (clocks.get("sm_mhz") or 1965.0) * 1e6
        # one multiply-accumulate per pair term (i, j); a persistent launch covers all K sweeps (swap events inside)
        macs_per_launch = K * w.n_rep * w.L * w.L / max(1, launches)
        launch_s = ms * 1e-3 / max(1, launches)              # CUDA events on the launching stream
        achieved = macs_per_launch / launch_s / 1e12
        dram_per_launch = DRAM_BYTES_PER_LAUNCH_FIXED + DRAM_BYTES_PER_SWEEP * K / max(1, launches)
        lanes = peaks["idp2a"][1] or IDP_LANES_PER_CLK_PER_SM          # IDP.2A alone, 2 warps per sub-partition
        lanes_mix = peaks["prmt+2idp2a (idp2a counted)"][1]            # ... next to one PRMT per two IDP.2A
        lanes_tile = peaks["bulk tile, near form (idp2a counted)"][1]  # ... in the kernel's own tile
        peak = N_SM * lanes * MACS_PER_IDP_LANE * f_hz / 1e12
        persistent = launches == 1 and K > 1 and variant == "direct"
        roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tmac/s", "frac": achieved / peak,
                    "traffic": dram_per_launch if persistent and w.name == "cfg3" else None,
                    "kernel": "sweep_%s_kernel" % variant,
                    "idp2a_lanes_per_clk_per_sm": lanes, "idp2a_lanes_in_bulk_mix": lanes_mix,
                    "frac_of_mix_ceiling": achieved / peak * lanes / lanes_mix if lanes_mix else None,
                    # the rate at which an SM runs the kernel's own bulk tile (8 sites x 16 steps on table and coupling
                    # registers, nothing else on the SM): what the instruction mix allows on 148 SMs
                    "idp2a_lanes_in_bulk_tile": lanes_tile,
                    "frac_of_tile_ceiling": achieved / peak * lanes / lanes_tile if lanes_tile else None,
                    "launch": "persistent (cooperative, swap events inside the kernel)" if persistent
                              else "one launch per swap interval",
                    "note": "algorithmic work = sweeps*n_rep*L^2 = %.3e integer multiply-accumulates per launch (one per "
                            "pair term; %d sweeps per launch); peak = 148 SMs x %.1f IDP.2A lanes/clk/SM (pt_measure_peaks, "
                            "this run) x 2 MAC x "
                            "sampled SM clock %.0f MHz -- a derived ALU peak, not MEASURED_PEAKS.json (its HBM and "
                            "tensor figures do not bound this path%s)"
                            % (macs_per_launch, K // max(1, launches), lanes, f_hz / 1e6,
                               ": %.0f KB of DRAM traffic per launch = %.2f GB/s of the measured %.0f GB/s; 128 of 148 "
                               "SMs carry a replica" % (dram_per_launch / 1e3, dram_per_launch / launch_s / 1e9,
                                                        measured_hbm_gbs()) if w.name == "cfg3" else "")}
        line = {"metric": metric_name(w), "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W_,
                "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": {"fp32": "f32", "fp64": "f64"}.get(variant, "int32"), "data": "synthetic",
                "config": dict(workload_config(w, variant, world), launch_plan=g.describe()), "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "flip_acceptance": acc, "pair_evaluations_per_s": value * (w.L - 1)}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline_leg(w)
        emit(line)
    g.close()
    if use_dist:
        dist.destroy_process_group()
    return 0


def run_cfg4(args):
    """--workload cfg4 (BASELINE.json configs[4], not the headline): the sigma-q scan, 40 independent handles of 32
    replicas (L=2048, q in {3,5,7,9} x sigma in {0.1..1.0}), one CUDA stream per handle, swap event every sweep.
    One step = one sweep + swap event of all 1280 replicas.  Single GPU only."""
    import torch
    from paper_1308_5426_b200 import build as ptbuild
    ptbuild.build()
    from paper_1308_5426_b200 import pt
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libpt has no CPU path")
    import torch.distributed as dist
    from paper_1308_5426_b200 import shard
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    use_dist = world > 1 or "RANK" in os.environ
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    # the 40 members are independent: rank r takes a contiguous block of them (no data-path collective; scaling "strong")
    base, n_loc = shard.ensemble_shard(40, world, rank)
    ws_all = inputs.config4()
    ws = ws_all[base:base + n_loc]
    K, W_ = args.steps, args.warmup
    streams = [torch.cuda.Stream() for _ in ws]
    gs = []
    for w, st in zip(ws, streams):
        g = pt.PT(w.L, w.q, w.sigma, 1, w.n_rep, inputs.betas(w), w.seed, variant=args.variant)
        g.use_torch_stream(st)
        gs.append(g)
    main_s = torch.cuda.current_stream()

    def steps(n):
        launches = 0
        c = max(1, args.sweeps_per_call)
        for k in range(0, n, c):     # interleaved, so that all 40 streams hold work from the start
            for g in gs:
                launches += g.sweeps_async(min(c, n - k), 1)
        return launches

    steps(W_)
    torch.cuda.synchronize()
    if use_dist:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start_sampling()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(main_s)
    for st in streams:
        st.wait_event(ev0)
    launches = steps(K)
    for st in streams:
        main_s.wait_stream(st)
    ev1.record(main_s)
    torch.cuda.synchronize()
    clocks = sampler.result()
    ms = ev0.elapsed_time(ev1)
    if use_dist:
        ms = shard.max_over_ranks(ms, dist, device="cuda")
    attempts = K * sum(w.n_rep * w.L for w in ws_all)       # whole job: all 40 members over all ranks
    value = attempts / (ms * 1e-3)

    starts = [g.get_spins() for g in gs]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for g, s0 in zip(gs, starts):
        g.set_spins(s0)
    steps(K)
    d2h = 0
    for g, w in zip(gs, ws):
        sp, E, ob = g.get_spins(), g.energy(), g.observables()
        d2h += sp.nbytes + E.nbytes + w.n_rep * 144
        assert ob["n_samples"].min() > 0
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    if use_dist:
        e2e_s = shard.max_over_ranks(e2e_s, dist, device="cuda")
        launches = int(shard.max_over_ranks(float(launches), dist, device="cuda")) * world
    if rank != 0:
        for g in gs:
            g.close()
        dist.destroy_process_group()
        return 0
    f_hz = (clocks.get("sm_mhz") or 1965.0) * 1e6
    macs = K * sum(w.n_rep * w.L * w.L for w in ws_all) / world     # per GPU
    achieved = macs / (ms * 1e-3) / 1e12
    peak = N_SM * IDP_LANES_PER_CLK_PER_SM * MACS_PER_IDP_LANE * f_hz / 1e12
    line = {"metric": "Metropolis spin-flip attempts/s on the sigma-q scan (40 ensembles x 32 replicas, L=2048)",
            "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W_, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "strong" if world > 1 else "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": "configs[4] (not the headline config): L=2048, q in {3,5,7,9} x sigma in {0.1..1.0} = "
                                   "40 handles x 32 replicas, T geometric in [0.4,3.0], hot start, swap every sweep, "
                                   "40 CUDA streams", "variant": gs[0].get_variant(),
                       "step": "1 sweep + swap event of all 1280 replicas = %d attempts" % (attempts // K),
                       "l2": "not flushed: the per-step state (1.3 MB of packed spins) is resident by design",
                       "launch_plans": {p: n for p, n in sorted(__import__("collections").Counter(g.describe() for g in gs).items())}},
            "clocks": clocks,
            "e2e": {"value": attempts / e2e_s, "unit": UNIT, "h2d_bytes_per_step": sum(s0.nbytes for s0 in starts) / K,
                    "d2h_bytes_per_step": d2h / K,
                    "what": "per handle pt_set_spins(host) + K x pt_sweeps_async(1) + pt_get_spins + pt_energy + "
                            "pt_observables (host buffers), wall clock"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tmac/s", "frac": achieved / peak,
                         "traffic": None, "kernel": "sweep_%s_kernel" % gs[0].get_variant(),
                         "note": "algorithmic work = sum over handles of sweeps*n_rep*L^2 multiply-accumulates over the "
                                 "whole timed region (40 streams run concurrently, so per-launch durations overlap); "
                                 "peak as for the headline config"}}
    emit(line)
    for g in gs:
        g.close()
    if use_dist:
        dist.destroy_process_group()
    return 0


def run_sharded(args):
    """--sharded: ONE configs[3] ensemble with its 128 slots spread over the ranks; every rank sweeps
    its configurations, at every swap event the ranks all-gather the running energies (n_rep int64 over NCCL: the only
    data that crosses GPUs) and take the same decisions (shard.ShardedEnsemble).  Scaling "strong".  One launch per
    sweep per rank (no persistent kernel: the swap barrier spans GPUs)."""
    import torch
    import torch.distributed as dist
    from paper_1308_5426_b200 import build as ptbuild
    ptbuild.build()
    from paper_1308_5426_b200 import pt, shard
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    use_dist = world > 1 or "RANK" in os.environ
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    w = pick_workload(args)
    K, W_ = args.steps, args.warmup
    ens = shard.ShardedEnsemble(pt, w.L, w.q, w.sigma, w.n_rep, inputs.betas(w), w.seed, dist=dist if use_dist else None)
    ens.sweeps(W_, w.swap_every)
    torch.cuda.synchronize()
    if use_dist:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start_sampling()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    ens.sweeps(K, w.swap_every)
    ev1.record()
    torch.cuda.synchronize()
    if use_dist:
        dist.barrier()
    clocks = sampler.result()
    ms = ev0.elapsed_time(ev1)
    if use_dist:
        ms = shard.max_over_ranks(ms, dist, device="cuda")
    value = K * w.n_rep * w.L / (ms * 1e-3)
    if rank == 0:
        emit({"metric": metric_name(w) + " (one ensemble sharded over the GPUs)", "value": value, "unit": UNIT,
              "n_gpus": world, "steps": K, "warmup": W_, "ms_per_step": ms / K, "higher_is_better": True,
              "scaling": "strong", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
              "config": dict(workload_config(w, "direct", world),
                             parallelism="slots of one ensemble sharded over %d GPU(s); all-gather of %d int64 energies "
                                         "per swap event (NCCL)" % (world, w.n_rep)),
              "clocks": clocks, "gpu_launches": 2 * K, "e2e": None, "roofline": None})
    ens.close()
    if use_dist:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", default="auto", choices=["auto", "direct", "field", "fp32", "fp64"])
    ap.add_argument("--sharded", action="store_true", help="one ensemble with its slots sharded over the GPUs (SURVEY.md 8(e)(2))")
    ap.add_argument("--peaks", action="store_true", help="print the instruction-rate micro-benchmarks (pt_measure_peaks) and exit")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweeps-per-call", type=int, default=1,
                    help="cfg4: sweeps per pt_sweeps_async call and handle (swap event after every sweep either way)")
    ap.add_argument("--workload", default="cfg3", help="cfg3 (BASELINE.json's headline config, default), cfg4, paper:L or paper:L:R")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    # stdout carries exactly one JSON line: libraries that write to file descriptor 1 on their own (NCCL prints its
    # version banner there at communicator creation, compilers their progress) are sent to stderr instead
    global _JSON_OUT
    sys.stdout.flush()
    _JSON_OUT = os.fdopen(os.dup(1), "w")
    os.dup2(2, 1)
    if args.peaks:
        from paper_1308_5426_b200 import build as ptbuild
        ptbuild.build()
        from paper_1308_5426_b200 import pt
        emit({"peaks": pt.measure_peaks(), "unit": "lane-operations per clock and SM (lds128: bytes), for 1, 2, 3, 4 warps "
              "per SM sub-partition; clock64() inside the kernel"})
        return 0
    if args.sharded:
        return run_sharded(args)
    if args.workload == "cfg4":
        if args.impl == "reference":
            raise SystemExit("bench.py: --impl reference times the headline config or a paper:L shape")
        return run_cfg4(args)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
