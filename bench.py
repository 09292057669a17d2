#!/usr/bin/env python
"""bench.py -- site-updates/s and SMC wall-clock to beta=1 of the batched tempered-particle update.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C1]

A "step" is one pass of the whole hot path: a complete adaptive-tempering SMC-RW run from fresh
N(0,I) particles to beta = 1 (P1-P4, C1, C2 and k x (M1-M4) per temperature) on BASELINE.json's
configuration (default C1 = configs[1]: L=10, N=16384, k=20, ESS 0.5).  value = N*V*(mutation steps
executed) / time, summed over ranks.  The path does not shard ("replicas only"): with
--gpus N every rank runs an independent replica with its own seed, no collective on the data path.

One JSON line on stdout (rank 0).  --impl reference times the FP64 CPU oracle on the host cores.
"""
import argparse
import json
import math
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
# dram__bytes_read.sum + dram__bytes_write.sum of one mutation launch (profiles/, ncu --set full)
# (C1: the fused kernel; C3 / C4: the proposal GEMM, the dominant kernel of the large-V step)
NCU_DRAM_BYTES = {"C1": 6815744, "C3": 1127837175, "C4": 15380342000}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0,
            "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None

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
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(0.02)
        except Exception as e:                      # pragma: no cover - depends on the box
            self.reasons.add("nvml_unavailable:%s" % type(e).__name__)

    def result(self):
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


def run_reference(args, cfg):
    """--impl reference: the oracle as it stands, on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    V = cfg["L"] ** 2
    n_sample = min(cfg["N"], args.ref_particles if V < 1024 else 256)
    max_temps = args.max_temps if args.max_temps > 0 else (6 if V >= 1024 else 4096)
    for w in range(args.warmup):
        oracle_run(cfg, n_sample, 1000 + w, max_temps)
    tot_su, tot_t, Ts = 0, 0.0, []
    for s in range(args.steps):
        su, dt, T, thr = oracle_run(cfg, n_sample, s, max_temps)
        tot_su += su
        tot_t += dt
        Ts.append(T)
    value = tot_su / tot_t
    sample = "N=%d of %d particles, full adaptive tempering run to beta=1 per step" % (n_sample, cfg["N"])
    line = {"impl": "reference", "metric": "site-updates/s", "value": value, "unit": "site-updates/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, cfg, temps=Ts),
            "cpu_baseline": {"value": value, "unit": "site-updates/s", "cores": thr, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": "site-updates/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(args, cfg, temps=None):
    c = {"workload": "%s: phi^4 L=%d (V=%d) m0sq=%g lambda=%g, N=%d particles from N(0,I), adaptive "
                     "tempering to beta=1 at ESS %.2f, %d %s per temperature, systematic resampling"
                     % (args.workload, cfg["L"], cfg["L"] ** 2, cfg["m0sq"], cfg["lam"], cfg["N"],
                        cfg["ess"], cfg["k"],
                        "HMC transitions (%d leapfrog steps of %g, diagonal mass matrix; a site-update "
                        "is one site in one leapfrog step)" % (cfg["hmc"][1], cfg["hmc"][0])
                        if cfg.get("hmc") else
                        "independent-MH steps from the fitted Gaussian N(mu, Sigma)" if cfg.get("irmh") else
                        "RW-Metropolis steps, dense VxV covariance-Cholesky proposal"),
         "L": cfg["L"], "V": cfg["L"] ** 2, "N": cfg["N"], "k_steps": cfg["k"], "ess_target": cfg["ess"],
         "parallelism": "replicas x%d (no sharding)" % args.gpus,
         "l2": "flushed between timed steps (256 MiB write)"}
    if temps is not None:
        c["temperatures_per_step"] = temps
    if cfg["L"] ** 2 >= 1024:
        c["note"] = "full schedule to beta=1 takes 100+ temperatures at this size: each step runs the first max_temps"

    return c


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C1")
    ap.add_argument("--path", type=int, default=0, help="mutation path: 0 auto, 1 generic, 2 fused")
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
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    from paper_2511_15196_b200 import inputs
    cfg = dict(inputs.CONFIGS[args.workload])
    assert cfg["kind"] == "smc", "bench.py times SMC workloads (C0, C0g, C1, C3, C4, P10, P15, P18)"
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

    import numpy as np
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

    L, N, k, V = cfg["L"], cfg["N"], cfg["k"], cfg["L"] ** 2
    max_temps = args.max_temps if args.max_temps > 0 else (6 if V >= 1024 else 4096)
    h = B.smc_init(L, cfg["m0sq"], cfg["lam"], N, 0, device=dev)
    upm = units_per_step(cfg)
    if cfg.get("hmc"):
        B.smc_set_params(h, k_steps=k, ess_target=cfg["ess"], kernel=1, hmc_eps=cfg["hmc"][0],
                         hmc_leapfrog=cfg["hmc"][1])
    elif cfg.get("irmh"):
        B.smc_set_params(h, k_steps=k, ess_target=cfg["ess"], kernel=2)
    else:
        B.smc_set_params(h, k_steps=k, ess_target=cfg["ess"], mutation_path=args.path)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

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

    # ---- device-resident timing -------------------------------------------------------------
    for w in range(args.warmup):
        device_step(replicas.replica_seed(1000 + w, rank))
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = B.phi4_kernel_launches()
    ms, Ts = 0.0, []
    for s in range(args.steps):
        dt, T = device_step(replicas.replica_seed(s, rank))
        ms += dt
        Ts.append(T)
    launches = B.phi4_kernel_launches() - l0
    barrier()
    sampler.stop_flag = True
    sampler.join()
    site_updates = float(N) * V * k * upm * sum(Ts)
    logZ = B.log_Z(h)

    # ---- end to end through the C ABI with HOST buffers ---------------------------------------
    h_in = torch.empty((V, N), dtype=torch.float32, pin_memory=True)
    h_in.normal_(generator=torch.Generator().manual_seed(1234 + rank))
    phi_in = h_in.numpy()
    # results land in pinned host memory too (pageable destinations are staged by the driver)
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
        st = B.smc_get_state(h, out=h_out)            # D2H: final particles, S_E, U0
        lz = B.log_Z(h)
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) * 1e3, T, lz

    e2e_step(999)
    e2e_ms, e2e_T = 0.0, []
    barrier()
    for s in range(args.steps):
        dt, T, _ = e2e_step(replicas.replica_seed(s, rank))
        e2e_ms += dt
        e2e_T.append(T)
    barrier()
    e2e_su = float(N) * V * k * upm * sum(e2e_T)

    # ---- dominant kernel: the mutation, timed alone at a mid-schedule state -------------------
    B.smc_reset(h, 4242)
    for _ in range(3):
        B.smc_step(h, want_info=False)
    torch.cuda.synchronize()
    for _ in range(2):
        B.smc_mutate(h, k, want=False)
    reps = 5
    l1 = B.phi4_kernel_launches()
    # CUDA events on the library's own stream around `reps` back-to-back k-step mutations
    mut_ms = B.smc_time_mutation(h, k, reps)                  # k steps
    mut_launches = (B.phi4_kernel_launches() - l1 - 2) // reps    # minus the two counter resets

    # ---- population step: resample (integer scan, ancestors) + gather, device-resident weights ----
    B.smc_reweight(h)                                          # weights at the ESS target
    B.smc_resample(h)
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pe0.record()
    for _ in range(reps):
        B.smc_resample(h, want=False)                          # P3 + P4, nothing but the control block read back
    pe1.record()
    torch.cuda.synchronize()
    pop_ms = pe0.elapsed_time(pe1) / reps

    # ---- reduce over ranks: MAX of the times, SUM of the work (no data-path collective) ---------
    tmax, usum = replicas.reduce_stats({"ms": ms, "e2e_ms": e2e_ms, "mut_ms": mut_ms, "pop_ms": pop_ms},
                                       {"su": site_updates, "e2e_su": e2e_su}, device=dev)
    ms, e2e_ms, mut_ms, pop_ms = tmax["ms"], tmax["e2e_ms"], tmax["mut_ms"], tmax["pop_ms"]
    site_updates, e2e_su = usum["su"], usum["e2e_su"]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    pk = peaks()
    # Roofline of the dominant kernel, the fused mutation: plain-ALU bound; the
    # algorithmic work is 40 lane-ops per site-update (Philox ~20, Box-Muller ~6, action ~14;
    # SURVEY 8(d)); the proposal product rides on the tensor pipe.  Peak: 148 SM x 128 lanes x clock
    # (an FMA counts as one lane-op).  traffic: dram bytes per launch from the committed ncu capture.
    work = ALU_OPS_PER_SITE_UPDATE * float(N) * V * k
    alu_peak = 148 * 128 * pk["sm_max_mhz"] * 1e6 / 1e12
    achieved = work / (mut_ms * 1e-3) / 1e12
    if cfg.get("hmc"):
        work = ALU_OPS_PER_LEAPFROG_SITE * float(N) * V * k * upm
        achieved = work / (mut_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "hmc_kernel x%d transitions (%d launches)" % (k, mut_launches),
                    "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s", "frac": achieved / alu_peak,
                    "ops": "lane-ops (FMA = 1), 11 per site per leapfrog step", "traffic": None,
                    "peak_source": "derived: 148 SM x 128 lanes x %.0f MHz (%s clocks)"
                    % (pk["sm_max_mhz"], pk["source"]),
                    "site_updates_per_s": float(N) * V * k * upm / (mut_ms * 1e-3), "ms": mut_ms}
    elif V <= 112:
        roofline = {"bound": "alu", "kernel": "mutation x%d steps (%d launches)" % (k, mut_launches),
                    "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s", "frac": achieved / alu_peak,
                    "ops": "lane-ops (FMA = 1), 40 per site-update",
                    "traffic": NCU_DRAM_BYTES.get(args.workload),
                    "peak_source": "derived: 148 SM x 128 lanes x %.0f MHz (%s clocks)"
                    % (pk["sm_max_mhz"], pk["source"]),
                    "site_updates_per_s": float(N) * V * k / (mut_ms * 1e-3), "ms": mut_ms}
    else:
        # Large V: the mutation is the 3xTF32 tcgen05 proposal GEMM plus HBM-bound
        # normals / accept kernels.  Algorithmic work = the triangular product, (V+1) flop per
        # site-update in FP32-equivalent flop; every such flop costs three TF32 MMAs, so 1/3 is the
        # ceiling of this fraction.  Peak: measured dense BF16 x 1/2 (nominal TF32 : BF16 ratio).
        tf32_peak = 0.5 * pk["bf16_tflops"]
        achieved = (V + 1) * float(N) * V * k / (mut_ms * 1e-3) / 1e12
        roofline = {"bound": "tensor", "kernel": "mutation x%d steps (%d launches)" % (k, mut_launches),
                    "achieved": achieved, "peak": tf32_peak, "unit": "TFLOP/s", "frac": achieved / tf32_peak,
                    "ops": "FP32-equivalent flop of the triangular L*z, (V+1) per site-update; 3xTF32 "
                           "issues 3 MMAs per flop (ceiling 1/3)",
                    "traffic": NCU_DRAM_BYTES.get(args.workload),
                    "peak_source": "%s bf16 %.0f TFLOP/s x 1/2" % (pk["source"], pk["bf16_tflops"]),
                    "site_updates_per_s": float(N) * V * k / (mut_ms * 1e-3), "ms": mut_ms}
    # Population step (P3 + P4): 8 bytes per site (4 read + 4 written) + 12 bytes per particle.
    pop_bytes = 8.0 * N * V + 12.0 * N
    population = {"bound": "hbm", "kernel": "resample + gather", "achieved": pop_bytes / (pop_ms * 1e-3) / 1e9,
                  "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": pop_bytes / (pop_ms * 1e-3) / 1e9 / pk["hbm_gbs"],
                  "ms": pop_ms, "state_in_l2": bool(8.0 * N * V < 126e6),
                  "note": "integer CDF scan + ancestor search + gather, one control-block readback per call"}

    cpu = None
    if not args.no_cpu_baseline:
        # the oracle as it stands on the host cores: full runs of the same workload until ~10 s of
        # CPU work (large lattices: a reduced population, the per-particle work is independent)
        n_s = min(N, args.ref_particles if V < 1024 else 256)
        su_tot, dt_tot, runs, T, thr = 0.0, 0.0, 0, 0, 1
        while dt_tot < 10.0 and runs < 12:
            su, dt, T, thr = oracle_run(cfg, n_s, runs, max_temps)
            su_tot += su
            dt_tot += dt
            runs += 1
        cpu = {"value": su_tot / dt_tot, "unit": "site-updates/s", "cores": thr, "kind": "oracle",
               "sample": "%d oracle runs of N=%d of %d particles, %d temperatures each, %.1f s of CPU time"
               % (runs, n_s, N, T, dt_tot)}

    line = {"metric": "site-updates/s", "value": site_updates / (ms * 1e-3), "unit": "site-updates/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": workload_config(args, cfg, temps=Ts),
            "smc_wall_clock_ms_to_beta1": ms / args.steps, "logZ_last": logZ,
            "e2e": {"value": e2e_su / (e2e_ms * 1e-3), "unit": "site-updates/s",
                    "h2d_bytes_per_step": V * N * 4, "d2h_bytes_per_step": V * N * 4 + 8 * N + 8,
                    "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": int(launches), "clocks": sampler.result(), "roofline": roofline,
            "population_step": population, "cpu_baseline": cpu}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
