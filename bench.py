#!/usr/bin/env python
"""bench.py -- site-updates/s and SMC wall-clock to beta=1 of the batched tempered-particle update.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C1]

A "step" is one pass of the whole hot path: a complete adaptive-tempering SMC-RW run from fresh
N(0,I) particles to beta = 1 (P1-P4, C1, C2 and k x (M1-M4) per temperature) on BASELINE.json's
configuration (default C1 = configs[1]: L=10, N=16384, k=20, ESS 0.5).  value = N*V*(mutation steps
executed) / time, summed over ranks.  The path does not shard ("replicas only"): with
--gpus N every rank runs an independent replica with its own seed, no collective on the data path.

One JSON line on stdout (rank 0).  Besides the headline workload it carries
  peaks_measured  dense tcgen05 kind::tf32 / kind::f16, FP32 FMA and IMAD.WIDE rates measured in this run through
                  phi4_measure_peaks (the roofline denominators MEASURED_PEAKS.json does not hold)
  large_v         the same measurement on C3 and C4 (first --max-temps temperatures per step), where
                  the rooflines mean something: the tcgen05 proposal GEMM against the measured peak of the
                  MMA kind it issues (kind::f16 for the scaled 3xFP16 split, kind::tf32 with --path 3) and
                  the population step against the HBM peak, with per-phase device times
--impl reference times the FP64 CPU oracle on the host cores.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

ALU_OPS_PER_SITE_UPDATE = 40          # Philox ~20 int + Box-Muller ~6 + action ~14
# HMC: per site per leapfrog step: neighbour sum 3, 4a-nb 1, a^2 1, lam4*a^2+m0sq 1,
# *a 1, + 1, beta*gs+a 1, kick 1, drift 1
ALU_OPS_PER_LEAPFROG_SITE = 11
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, copied from the
# committed `ncu --set full` captures (not measured by this run): C1 the fused mutation kernel,
# C3 / C4 the proposal GEMM.
NCU_TRAFFIC = {"C1": (6815000, "profiles/r02_ncu_tables.md"),
               "C3": (1035600000, "profiles/r02_ncu_tables.md (capture r02d: the launch also writes the next "
                                  "step's normals, 0.21 GB)"),
               "C4": (13807000000, "profiles/r02_ncu_tables.md (capture r02d: the launch also writes the next "
                                   "step's normals, 2.1 GB)")}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "source": "MEASURED_PEAKS.json"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0,
            "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None
        self.ready = threading.Event()          # NVML is up: the caller waits for this before timing

    def begin(self):
        self.start()
        self.ready.wait(10.0)
        return self

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                     nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                     nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                     nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
            self.ready.set()
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(0.005)
        except Exception as e:                      # pragma: no cover - depends on the box
            self.reasons.add("nvml_unavailable:%s" % type(e).__name__)
        self.ready.set()

    def finish(self):
        self.stop_flag = True
        self.join()
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


def oracle_run(cfg, n_sample, seed, max_temps=4096):
    """One oracle SMC run on a reduced population; returns (site_updates, seconds, T, threads)."""
    from oracle import oracle as O
    t0 = time.perf_counter()
    if cfg.get("irmh"):
        r = O.smc_irmh_run(cfg["L"], cfg["m0sq"], cfg["lam"], n_sample, seed, cfg["k"],
                           ess_target=cfg["ess"], max_temps=max_temps)
    elif cfg.get("hmc"):
        eps, nfrog = cfg["hmc"]
        r = O.smc_hmc_run(cfg["L"], cfg["m0sq"], cfg["lam"], n_sample, seed, cfg["k"],
                          ess_target=cfg["ess"], eps=eps, nfrog=nfrog, max_temps=max_temps)
    else:
        r = O.smc_run(cfg["L"], cfg["m0sq"], cfg["lam"], n_sample, seed, cfg["k"], ess_target=cfg["ess"],
                      max_temps=max_temps)
    dt = time.perf_counter() - t0
    V = cfg["L"] ** 2
    return n_sample * V * cfg["k"] * units_per_step(cfg) * r["T"], dt, r["T"], O.num_threads()


def units_per_step(cfg):
    """Site-updates per site per mutation step: 1 for RW-Metropolis; an HMC transition updates every
    site once per leapfrog step."""
    return cfg["hmc"][1] if cfg.get("hmc") else 1


def default_max_temps(cfg, arg):
    return arg if arg > 0 else (6 if cfg["L"] ** 2 >= 1024 else 4096)


def run_reference(args, cfg):
    """--impl reference: the oracle as it stands, on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    V = cfg["L"] ** 2
    n_sample = min(cfg["N"], args.ref_particles if V < 1024 else 128)
    max_temps = args.max_temps if args.max_temps > 0 else (1 if V >= 1024 else 4096)
    for w in range(args.warmup):
        oracle_run(cfg, n_sample, 1000 + w, max_temps)
    tot_su, tot_t, Ts = 0, 0.0, []
    for s in range(args.steps):
        su, dt, T, thr = oracle_run(cfg, n_sample, s, max_temps)
        tot_su += su
        tot_t += dt
        Ts.append(T)
    value = tot_su / tot_t
    sample = "N=%d of %d particles, %s per step" % (
        n_sample, cfg["N"], "full adaptive tempering run to beta=1" if max_temps >= 4096
        else "first %d temperature(s)" % max_temps)
    line = {"impl": "reference", "metric": "site-updates/s", "value": value, "unit": "site-updates/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args.workload, cfg, args.gpus, temps=Ts),
            "cpu_baseline": {"value": value, "unit": "site-updates/s", "cores": thr, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": "site-updates/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------ nested sampling workloads --
def ns_config(name, cfg, gpus, iters):
    return {"workload": "%s: nested sampling, phi^4 L=%d (V=%d) m0sq=%g lambda=%g, %d live points from "
                        "N(0,I), %d deleted per iteration, %d %s steps per replacement, run to remaining "
                        "evidence < %g" % (name, cfg["L"], cfg["L"] ** 2, cfg["m0sq"], cfg["lam"],
                                           cfg["n_live"], cfg["k_del"], cfg["n_walk"],
                                           "slice-sampling" if cfg.get("inner") == "slice"
                                           else "constrained RW-Metropolis", cfg["stop_frac"]),
            "L": cfg["L"], "V": cfg["L"] ** 2, "n_live": cfg["n_live"], "k_delete": cfg["k_del"],
            "n_walk": cfg["n_walk"], "parallelism": "replicas x%d (no sharding)" % gpus,
            "l2": "flushed between timed steps (256 MiB write)", "iterations_per_step": iters,
            "unit_definition": "one site of one walker in one inner step"}


def ns_oracle_run(cfg, seed, max_iter):
    from oracle import oracle as O
    t0 = time.perf_counter()
    r = O.ns_run(cfg["L"], cfg["m0sq"], cfg["lam"], cfg["n_live"], cfg["k_del"], cfg["n_walk"], seed,
                 stop_frac=cfg["stop_frac"], max_iter=max_iter, inner=cfg.get("inner", "rw"))
    dt = time.perf_counter() - t0
    return float(r["iters"]) * cfg["k_del"] * cfg["n_walk"] * cfg["L"] ** 2, dt, r["iters"], O.num_threads()


def run_ns_reference(args, cfg):
    """--impl reference on a nested-sampling workload: the oracle, a bounded number of iterations."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    max_iter = 8 if cfg.get("inner") == "slice" else 64
    for w in range(args.warmup):
        ns_oracle_run(cfg, 1000 + w, 2)
    su, tt, its, thr = 0.0, 0.0, [], 1
    for s in range(args.steps):
        a, dt, it, thr = ns_oracle_run(cfg, s, max_iter)
        su += a; tt += dt; its.append(it)
    value = su / tt
    print(json.dumps({"impl": "reference", "metric": "site-updates/s", "value": value,
                      "unit": "site-updates/s", "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * tt / args.steps, "higher_is_better": True,
                      "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": ns_config(args.workload, cfg, args.gpus, its),
                      "cpu_baseline": {"value": value, "unit": "site-updates/s", "cores": thr,
                                       "kind": "oracle",
                                       "sample": "first %d iterations of the run per step" % max_iter},
                      "e2e": {"value": value, "unit": "site-updates/s", "h2d_bytes_per_step": 0,
                              "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


def run_ns(args, cfg):
    """A nested-sampling workload (BASELINE configs[2] = C2, or PNS10): a step is one whole run."""
    import torch
    import torch.distributed as dist
    from paper_2511_15196_b200 import binding as B
    from paper_2511_15196_b200 import build, replicas
    rank, world, local = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    B.load()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    pk = peaks()
    mp = B.phi4_measure_peaks(args.peak_seconds, device=dev)
    L, V, n, kd, nw = cfg["L"], cfg["L"] ** 2, cfg["n_live"], cfg["k_del"], cfg["n_walk"]
    h = B.ns_init(L, cfg["m0sq"], cfg["lam"], n, kd, nw, 0, cfg["stop_frac"], 4096, device=dev)
    if cfg.get("inner") == "slice":
        B.ns_set_params(h, inner=1)

    def step(seed, e2e):
        flush.fill_(seed & 0xFF)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        B.smc_reset(h, seed)
        it = B.ns_run(h)
        e1.record()
        nbytes = 0
        if e2e:                                   # D2H: the dead-point log (S_E, M, log w) and log Z
            d = B.ns_get_dead(h)
            B.log_Z(h)
            nbytes = sum(v.nbytes for v in d.values() if hasattr(v, "nbytes")) + 8
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) * 1e3 if e2e else e0.elapsed_time(e1), it, nbytes

    for w in range(max(args.warmup, 1)):
        step(replicas.replica_seed(1000 + w, rank), False)
    barrier()
    sampler = ClockSampler(local).begin()
    l0 = B.phi4_kernel_launches()
    ms, its = 0.0, []
    for s in range(args.steps):
        dt, it, _ = step(replicas.replica_seed(s, rank), False)
        ms += dt; its.append(it)
    launches = B.phi4_kernel_launches() - l0
    barrier()
    clocks = sampler.finish()
    e2e_ms, e2e_its, nbytes = 0.0, [], 0
    for s in range(args.steps):
        dt, it, nbytes = step(replicas.replica_seed(s, rank), True)
        e2e_ms += dt; e2e_its.append(it)
    barrier()
    su, e2e_su = float(sum(its)) * kd * nw * V, float(sum(e2e_its)) * kd * nw * V
    tmax, usum = replicas.reduce_stats({"ms": ms, "e2e_ms": e2e_ms}, {"su": su, "e2e_su": e2e_su}, device=dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    ms, e2e_ms, su, e2e_su = tmax["ms"], tmax["e2e_ms"], usum["su"], usum["e2e_su"]
    cpu = None
    if not args.no_cpu_baseline:
        a, dt, it, thr = ns_oracle_run(cfg, 0, 4 if cfg.get("inner") == "slice" else 48)
        cpu = {"value": a / dt, "unit": "site-updates/s", "cores": thr, "kind": "oracle",
               "sample": "first %d iterations of one run, %.1f s of CPU time" % (it, dt)}
    achieved = ALU_OPS_PER_SITE_UPDATE * su / world / (ms * 1e-3) / 1e12
    line = {"metric": "site-updates/s", "value": su / (ms * 1e-3), "unit": "site-updates/s", "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 1), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": ns_config(args.workload, cfg, world, its),
            "us_per_iteration": 1e3 * ms / max(1, sum(its)), "logZ_last": B.log_Z(h),
            "e2e": {"value": e2e_su / (e2e_ms * 1e-3), "unit": "site-updates/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": int(nbytes), "ms_per_step": e2e_ms / args.steps,
                    "note": "the live points are drawn on the device (INIT Philox stream): no host input"},
            "gpu_launches": int(launches), "clocks": clocks,
            "roofline": {"bound": "alu", "kernel": "whole iteration (select, evidence, covariance, Cholesky, "
                         "walk): the walk runs on k_delete / 128 CTAs and is latency-bound",
                         "achieved": achieved, "peak": mp["ffma_tlaneops"], "unit": "T lane-op/s",
                         "frac": achieved / mp["ffma_tlaneops"],
                         "ops": "lane-ops (FMA = 1), %d per walker site-update" % ALU_OPS_PER_SITE_UPDATE,
                         "peak_source": "phi4_measure_peaks FP32 FMA rate of this run", "traffic": None},
            "peaks_measured": dict(mp, hbm_gbs=pk["hbm_gbs"], bf16_tflops=pk["bf16_tflops"]),
            "cpu_baseline": cpu}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def workload_config(name, cfg, gpus, temps=None, max_temps=None):
    c = {"workload": "%s: phi^4 L=%d (V=%d) m0sq=%g lambda=%g, N=%d particles from N(0,I), adaptive "
                     "tempering to beta=1 at ESS %.2f, %d %s per temperature, systematic resampling"
                     % (name, cfg["L"], cfg["L"] ** 2, cfg["m0sq"], cfg["lam"], cfg["N"],
                        cfg["ess"], cfg["k"],
                        "HMC transitions (%d leapfrog steps of %g, diagonal mass matrix; a site-update "
                        "is one site in one leapfrog step)" % (cfg["hmc"][1], cfg["hmc"][0])
                        if cfg.get("hmc") else
                        "independent-MH steps from the fitted Gaussian N(mu, Sigma)" if cfg.get("irmh") else
                        "RW-Metropolis steps, dense VxV covariance-Cholesky proposal"),
         "L": cfg["L"], "V": cfg["L"] ** 2, "N": cfg["N"], "k_steps": cfg["k"], "ess_target": cfg["ess"],
         "parallelism": "replicas x%d (no sharding)" % gpus,
         "l2": "flushed between timed steps (256 MiB write)"}
    if temps is not None:
        c["temperatures_per_step"] = temps
    if cfg["L"] ** 2 >= 1024:
        c["note"] = ("the full schedule to beta=1 takes 100+ temperatures at this size: a step runs the "
                     "first %s temperatures" % (max_temps if max_temps else "max_temps"))
    return c


def rooflines(name, cfg, ph, pk, mp, timed_region_s, path=0):
    """Roofline records of the dominant mutation kernel and of the population step.
    ph: per-phase device times in ms; pk: MEASURED_PEAKS.json; mp: phi4_measure_peaks of this run."""
    L, N, k = cfg["L"], cfg["N"], cfg["k"]
    V, upm = L * L, units_per_step(cfg)
    mut_ms = ph["mutation_k_steps"]
    traffic, tsrc = NCU_TRAFFIC.get(name, (None, None))
    derived_alu = 148 * 128 * pk["sm_max_mhz"] * 1e6 / 1e12
    if cfg.get("hmc") or V <= 112:
        # plain-ALU bound (DESIGN.md 5.1 / 5.5): lane-ops, an FMA = 1
        per = ALU_OPS_PER_LEAPFROG_SITE if cfg.get("hmc") else ALU_OPS_PER_SITE_UPDATE
        work = per * float(N) * V * k * upm
        achieved = work / (mut_ms * 1e-3) / 1e12
        peak = mp["ffma_tlaneops"]
        roof = {"bound": "alu", "kernel": ("hmc_kernel" if cfg.get("hmc") else "mutate_tc_kernel") +
                " x%d steps, one launch" % k,
                "achieved": achieved, "peak": peak, "unit": "T lane-op/s", "frac": achieved / peak,
                "ops": "lane-ops (FMA = 1), %d per site-update" % per,
                "peak_source": "phi4_measure_peaks FP32 FMA rate of this run (derived 148 SM x 128 lanes x "
                               "%.0f MHz = %.1f; IMAD.WIDE rate %.1f)" % (pk["sm_max_mhz"], derived_alu,
                                                                         mp["imad_wide_tlaneops"]),
                "traffic": traffic if not cfg.get("hmc") else None,
                "traffic_source": tsrc if not cfg.get("hmc") else None,
                "site_updates_per_s": float(N) * V * k * upm / (mut_ms * 1e-3), "ms": mut_ms}
    else:
        # tensor bound: the proposal GEMM of ONE step, timed alone.  Algorithmic
        # work: the triangular product in three-product split precision (north_star), 3 products x
        # 2 flop x N V (V+1) / 2; the FP32-equivalent ("useful") flop are a third of that.  The
        # operands are FP16 pairs (scaled 3xFP16, same 11-bit significands as TF32) unless
        # --path 3 asks for 3xTF32: the peak is the measured dense rate of the kind the kernel issues.
        t = ph["proposal_gemm"] * 1e-3
        issued = 3.0 * float(N) * V * (V + 1)
        achieved = issued / t / 1e12
        sustained = timed_region_s >= 0.25
        kind = "tf32" if path == 3 else "f16"
        peak = mp[kind + "_tflops_sustained"] if sustained else mp[kind + "_tflops_burst"]
        roof = {"bound": "tensor", "kernel": "propose_tc_kernel<%s>, one launch = one mutation step"
                                             % ("false" if path == 3 else "true"),
                "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "useful_frac": achieved / 3.0 / peak,
                "ops": "%s flop of the triangular L*z in %s split precision, 3 N V (V+1) per "
                       "step; useful_frac counts the FP32-equivalent N V (V+1)"
                       % (("TF32", "3xTF32") if path == 3 else ("FP16", "scaled 3xFP16")),
                "peak_source": "phi4_measure_peaks dense tcgen05 kind::%s of this run, %s (burst %.0f, "
                               "sustained %.0f; kind::tf32 %.0f / %.0f; bf16 of MEASURED_PEAKS.json %.0f)"
                               % (kind, "sustained: the launch was timed inside a >= 0.25 s region" if sustained
                                  else "burst", mp[kind + "_tflops_burst"], mp[kind + "_tflops_sustained"],
                                  mp["tf32_tflops_burst"], mp["tf32_tflops_sustained"], pk["bf16_tflops"]),
                "proposal_gemm_3xtf32_ms": ph.get("proposal_gemm_3xtf32"),
                "traffic": traffic, "traffic_source": tsrc,
                "site_updates_per_s": float(N) * V / t, "ms": ph["proposal_gemm"],
                "mutation_step_ms": mut_ms / k}
    pop_ms = ph["resample_gather"]
    pop_bytes = 8.0 * N * V + 12.0 * N                 # 4 read + 4 written per site, 12 per particle
    gat = 8.0 * N * V / (ph["gather"] * 1e-3) / 1e9
    population = {"bound": "hbm", "kernel": "resample (scan, ancestors) + gather",
                  "achieved": pop_bytes / (pop_ms * 1e-3) / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s",
                  "frac": pop_bytes / (pop_ms * 1e-3) / 1e9 / pk["hbm_gbs"], "ms": pop_ms,
                  "gather_alone": {"achieved": gat, "frac": gat / pk["hbm_gbs"], "ms": ph["gather"]},
                  "peak_source": pk["source"], "state_in_l2": bool(8.0 * N * V < 126e6)}
    return roof, population


def measure_workload(name, cfg, args, env, steps, warmup, max_temps, want_e2e):
    """Times `steps` whole runs of one workload on this rank; returns raw times and records."""
    import torch
    B, replicas, dev, rank, local, flush = (env[k] for k in ("B", "replicas", "dev", "rank", "local", "flush"))
    L, N, k, V = cfg["L"], cfg["N"], cfg["k"], cfg["L"] ** 2
    upm = units_per_step(cfg)
    h = B.smc_init(L, cfg["m0sq"], cfg["lam"], N, 0, device=dev)
    if cfg.get("hmc"):
        B.smc_set_params(h, k_steps=k, ess_target=cfg["ess"], kernel=1, hmc_eps=cfg["hmc"][0],
                         hmc_leapfrog=cfg["hmc"][1])
    elif cfg.get("irmh"):
        B.smc_set_params(h, k_steps=k, ess_target=cfg["ess"], kernel=2)
    else:
        B.smc_set_params(h, k_steps=k, ess_target=cfg["ess"], mutation_path=args.path)

    def device_step(seed):
        """inputs resident in HBM: particles are drawn on the device by the INIT Philox stream."""
        flush.fill_(seed & 0xFF)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        B.smc_reset(h, seed)
        T = B.smc_run(h, max_temps)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1), T

    for w in range(warmup):
        device_step(replicas.replica_seed(1000 + w, rank))
    env["barrier"]()
    sampler = ClockSampler(local).begin()
    l0 = B.phi4_kernel_launches()
    ms, Ts = 0.0, []
    for s in range(steps):
        dt, T = device_step(replicas.replica_seed(s, rank))
        ms += dt
        Ts.append(T)
    launches = B.phi4_kernel_launches() - l0
    env["barrier"]()
    clocks = sampler.finish()
    out = {"ms": ms, "Ts": Ts, "launches": int(launches), "clocks": clocks,
           "site_updates": float(N) * V * k * upm * sum(Ts), "logZ": B.log_Z(h)}

    if want_e2e:
        # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
        h_in = torch.empty((V, N), dtype=torch.float32, pin_memory=True)
        h_in.normal_(generator=torch.Generator().manual_seed(1234 + rank))
        phi_in = h_in.numpy()
        h_out = {"phi": torch.empty((V, N), dtype=torch.float32, pin_memory=True).numpy(),
                 "S": torch.empty(N, dtype=torch.float32, pin_memory=True).numpy(),
                 "U0": torch.empty(N, dtype=torch.float32, pin_memory=True).numpy()}

        def e2e_step(seed):
            flush.fill_(seed & 0xFF)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            B.smc_reset(h, seed)
            B.smc_set_state(h, phi_in, 0.0, 0)            # H2D: V*N fp32 initial particles
            T = B.smc_run(h, max_temps)
            B.smc_get_state(h, out=h_out)                 # D2H: final particles, S_E, U0
            B.log_Z(h)
            torch.cuda.synchronize()
            return (time.perf_counter() - t0) * 1e3, T

        e2e_step(999)
        e2e_ms, e2e_T = 0.0, []
        env["barrier"]()
        for s in range(steps):
            dt, T = e2e_step(replicas.replica_seed(s, rank))
            e2e_ms += dt
            e2e_T.append(T)
        env["barrier"]()
        out["e2e_ms"] = e2e_ms
        out["e2e_su"] = float(N) * V * k * upm * sum(e2e_T)

    # ---- phases, timed alone at a mid-schedule state with CUDA events on the library's stream ----
    B.smc_reset(h, 4242)
    for _ in range(3):
        B.smc_step(h, want_info=False)
    torch.cuda.synchronize()
    reps = 5
    ph = {}
    B.smc_time_phase(h, "mutation", 1)                         # warm
    t0 = time.perf_counter()
    ph["mutation_k_steps"] = B.smc_time_phase(h, "mutation", reps)
    region_s = time.perf_counter() - t0
    if V > 112 and not cfg.get("hmc") and not cfg.get("irmh") and args.path != 1:
        for key, p in (("proposal_gemm", "proposal"), ("normals", "normals"), ("accept", "accept")):
            B.smc_time_phase(h, p, 1)
            t0 = time.perf_counter()
            ph[key] = B.smc_time_phase(h, p, reps * 2)
            if key == "proposal_gemm":
                region_s = time.perf_counter() - t0
        if args.path != 3:
            # the same product in 3xTF32 (mutation_path 3), for the record: same accuracy, twice the MMAs
            B.smc_set_params(h, k_steps=k, ess_target=cfg["ess"], mutation_path=3)
            B.smc_time_phase(h, "proposal", 1)
            ph["proposal_gemm_3xtf32"] = B.smc_time_phase(h, "proposal", reps * 2)
            B.smc_set_params(h, k_steps=k, ess_target=cfg["ess"], mutation_path=args.path)
    B.smc_reset(h, 4242)
    for _ in range(3):
        B.smc_step(h, want_info=False)
    B.smc_reweight(h)                                          # weights at the ESS target
    B.smc_resample(h)
    ph["resample_gather"] = B.smc_time_phase(h, "resample", reps)
    ph["gather"] = B.smc_time_phase(h, "gather", reps)
    ph["cov_chol"] = B.smc_time_phase(h, "covchol", reps)
    ph["reweight"] = B.smc_time_phase(h, "reweight", reps)
    out["phases_ms"] = ph
    out["phase_region_s"] = region_s
    h.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C1")
    ap.add_argument("--path", type=int, default=0, help="mutation path: 0 auto, 1 generic, 2 fused, 3 auto with the large-V proposal in 3xTF32")
    ap.add_argument("--ref-particles", type=int, default=16384)
    ap.add_argument("--kernel", default="rw", choices=["rw", "hmc", "irmh"],
                    help="rejuvenation kernel: RW-Metropolis (BASELINE metric), HMC (NEXT row f1) or "
                         "independent MH (NEXT row f2)")
    ap.add_argument("--k-steps", type=int, default=-1, help="override the workload's steps per temperature")
    ap.add_argument("--hmc-eps", type=float, default=0.1)
    ap.add_argument("--hmc-leapfrog", type=int, default=20)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--max-temps", type=int, default=-1,
                    help="temperatures per step; -1: to beta=1 (C0-C2), 6 for C3/C4 whose full schedule "
                         "takes 100+ temperatures")
    ap.add_argument("--large-v", default="C3,C4",
                    help="workloads measured beside the headline one as `large_v` sub-records (1 GPU "
                         "only); '' to skip")
    ap.add_argument("--peak-seconds", type=float, default=2.0,
                    help="length of the sustained tcgen05 TF32 peak measurement")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    from paper_2511_15196_b200 import inputs
    cfg = dict(inputs.CONFIGS[args.workload])
    if cfg["kind"] == "ns":                            # C2 (BASELINE configs[2]), PNS10
        if args.impl == "reference":
            run_ns_reference(args, cfg)
        else:
            run_ns(args, cfg)
        return
    if args.kernel == "hmc":
        cfg["hmc"] = (args.hmc_eps, args.hmc_leapfrog)
        cfg["k"] = 2                                   # "short HMC trajectories"
    if args.kernel == "irmh":
        cfg["irmh"] = True
    if args.k_steps > 0:
        cfg["k"] = args.k_steps
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    from paper_2511_15196_b200 import binding as B
    from paper_2511_15196_b200 import build, replicas

    rank, world, local = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    B.load()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    env = {"B": B, "replicas": replicas, "dev": dev, "rank": rank, "local": local, "barrier": barrier,
           "flush": torch.empty(256 << 20, dtype=torch.uint8, device=dev)}
    pk = peaks()
    mp = B.phi4_measure_peaks(args.peak_seconds, device=dev)      # every rank: keeps the ranks in step

    L, N, k, V = cfg["L"], cfg["N"], cfg["k"], cfg["L"] ** 2
    max_temps = default_max_temps(cfg, args.max_temps)
    m = measure_workload(args.workload, cfg, args, env, args.steps, args.warmup, max_temps, True)

    # ---- reduce over ranks: MAX of the times, SUM of the work (no data-path collective) ---------
    tmax, usum = replicas.reduce_stats({"ms": m["ms"], "e2e_ms": m["e2e_ms"]},
                                       {"su": m["site_updates"], "e2e_su": m["e2e_su"]}, device=dev)
    ms, e2e_ms = tmax["ms"], tmax["e2e_ms"]
    site_updates, e2e_su = usum["su"], usum["e2e_su"]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    roof, population = rooflines(args.workload, cfg, m["phases_ms"], pk, mp, m["phase_region_s"], args.path)

    # ---- large-V sub-records: where the rooflines mean something ------------------
    large = {}
    if world == 1 and args.kernel == "rw" and args.large_v:
        for name in [x for x in args.large_v.split(",") if x and x != args.workload]:
            c = dict(inputs.CONFIGS[name])
            mt = default_max_temps(c, args.max_temps)
            st, wu = (3, 3) if c["L"] >= 64 else (5, 3)
            r = measure_workload(name, c, args, env, st, wu, mt, False)
            rf, pop = rooflines(name, c, r["phases_ms"], pk, mp, r["phase_region_s"], args.path)
            large[name] = {"config": workload_config(name, c, 1, temps=r["Ts"], max_temps=mt),
                           "steps": st, "warmup": wu, "ms_per_step": r["ms"] / st,
                           "value": r["site_updates"] / (r["ms"] * 1e-3), "unit": "site-updates/s",
                           "ms_per_temperature": r["ms"] / max(1, sum(r["Ts"])),
                           "gpu_launches": r["launches"], "clocks": r["clocks"], "roofline": rf,
                           "population_step": pop, "phases_ms": r["phases_ms"]}

    cpu = None
    if not args.no_cpu_baseline:
        # the oracle as it stands on the host cores: full runs of the same workload until ~10 s of
        # CPU work (large lattices: a reduced population, the per-particle work is independent)
        n_s = min(N, args.ref_particles if V < 1024 else 128)
        mt = max_temps if V < 1024 else 1
        su_tot, dt_tot, runs, T, thr = 0.0, 0.0, 0, 0, 1
        while dt_tot < 10.0 and runs < 12:
            su, dt, T, thr = oracle_run(cfg, n_s, runs, mt)
            su_tot += su
            dt_tot += dt
            runs += 1
        cpu = {"value": su_tot / dt_tot, "unit": "site-updates/s", "cores": thr, "kind": "oracle",
               "sample": "%d oracle runs of N=%d of %d particles, %d temperatures each, %.1f s of CPU time"
               % (runs, n_s, N, T, dt_tot)}

    line = {"metric": "site-updates/s", "value": site_updates / (ms * 1e-3), "unit": "site-updates/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": workload_config(args.workload, cfg, world, temps=m["Ts"], max_temps=max_temps),
            "smc_wall_clock_ms_to_beta1": ms / args.steps if max_temps >= 4096 else None,
            "logZ_last": m["logZ"],
            "e2e": {"value": e2e_su / (e2e_ms * 1e-3), "unit": "site-updates/s",
                    "h2d_bytes_per_step": V * N * 4, "d2h_bytes_per_step": V * N * 4 + 8 * N + 8,
                    "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": m["launches"], "clocks": m["clocks"], "roofline": roof,
            "population_step": population, "phases_ms": m["phases_ms"],
            "peaks_measured": dict(mp, hbm_gbs=pk["hbm_gbs"], bf16_tflops=pk["bf16_tflops"],
                                   hbm_bf16_source=pk["source"],
                                   how="phi4_measure_peaks (csrc/measure.cu): dense tcgen05 kind::tf32 "
                                       "M128 N256 K8 (and kind::f16, K16) from resident smem operands on all SMs, burst = best "
                                       "of 5 launches, sustained = back to back for %.1f s; FP32 FMA and "
                                       "IMAD.WIDE+LOP3 (and FP64 FMA, dfma_tlaneops): 8 chains/thread, 2048 "
                                       "threads/SM" % args.peak_seconds),
            "large_v": large, "cpu_baseline": cpu}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
