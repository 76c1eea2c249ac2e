#!/usr/bin/env python
"""bench.py -- the driver's measurement contract for libhea_b200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--mc-steps n]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Workload (BASELINE.json:configs[3], "c4"): fcc 40x40x40 = 256,000 atoms, 4 species at 0.25, shells 1-2, non-zero
first-shell target (seed 11), 16 chains per GPU x 1e7 MC steps, K = 128 candidates per step, chain seed 4.
One bench "step" is one pass of the whole hot path over that batch, exactly the config: `hea_sro_full` of the 16 seeded
random start configurations (counts, alpha, J) followed by ONE `hea_mc_run` of the whole 1e7-step trajectory of every
chain (about 70,000 steps in the accept regime, the rest in the reject regime; `regimes` reports both separately).
--mc-steps n shortens the trajectory (exploration; stated in `config`).
`value` = swap trials/s = chains * mc-steps * K / device time of the whole step, inputs resident in HBM.
`e2e` = the same metric through the host-buffer C-ABI call `hea_mc_run_host` (H2D of the occupancies from pinned
memory, recount, MC, D2H of occupancies + counts + stats inside the timed region).
Multi-GPU: chains are independent, so rank r runs chains [16 r, 16 r + 16) with no data-path collective ("weak").

`roofline` is for the dominant kernel of the step (the MC kernel; ALU-issue bound, model in DESIGN.md section 6);
`recount_roofline` is for the table-driven recount kernel (sro_engine = 1) on the sweep point of configs[4] where the
neighbour table exceeds L2 (fcc 100^3 = 4,000,000 atoms, 3 shells, batch 1; HBM bound, 4*Z+1 = 169 B/atom);
`recount_stencil` is the table-free kernel `hea_sro_full` runs by default on the same point (1 B/atom of HBM traffic;
bound by instruction issue, model in DESIGN.md section 6.1b) with its atoms/s beside the table kernel's.
`cpu_baseline` / `--impl reference`: the CPU oracle (oracle/hea_oracle.c), as it stands, on the host cores, on a
bounded sample (the first steps of the same trajectory).
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

MC_REJECT_WARP_INSTR = 14_961_870_598 / 6.4e7     # per 32 trials: smsp__inst_executed.sum of the 1e6-step reject launch
MC_REJECT_WAVEFRONTS = 1_703_546_922 / 6.4e7       # l1tex__data_pipe_lsu_wavefronts_mem_shared.sum of the same launch
MC_REJECT_L2_SECTORS = 3_854_036_651 / 6.4e7       # l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum (site-histogram table words, via L2)
MC_FULL_WARP_INSTR = 151_253_341_748.0             # whole c4 launch (16 chains x 1e7 steps)
DTYPE = ("int32 counts + f64 objective (D6 order, no FMA); long windows pass a conservative fp32 reject filter on shell 1 "
         "first (rigorous error bound in its threshold, survivors evaluated in f64: accept decisions are the f64 ones); its "
         "inputs are per-site integer neighbour counts kept in a table")
METRIC = "delta-SRO swap trials/sec (c4: fcc 40^3, 256,000 atoms, 16 chains x 1e7 steps, K=128) incl. the full-SRO recount of the start"
UNIT = "swap-trials/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


# Figures that only a profiler can give, copied from the committed `ncu --set full` captures under profiles/ (bench.py
# never runs under a profiler); every use below names its source file in the JSON line.
NCU = {
    # whole c4 trajectory, one launch: dram__bytes_read.sum + dram__bytes_write.sum
    "mc_c4_full_dram_bytes": (8_003_584 + 69_541_120, "profiles/r2_mc_halo_c4_full.md"),
    "mc_c4_full_warp_instr": (MC_FULL_WARP_INSTR, "profiles/r2_mc_halo_c4_full.md"),
    # reject regime of c4 (1e6 steps after the trajectory): executed warp-instructions and shared-memory data-pipe
    # wavefronts per 32 trials (smsp__inst_executed.sum, l1tex__data_pipe_lsu_wavefronts_mem_shared.sum over 6.4e7 warp-trials)
    "mc_reject_warp_instr_per_32_trials": (MC_REJECT_WARP_INSTR, "profiles/r2_mc_halo_reject.md"),
    "mc_reject_smem_wavefronts_per_32_trials": (MC_REJECT_WAVEFRONTS, "profiles/r2_mc_halo_reject.md"),
    "mc_reject_l2_sectors_per_32_trials": (MC_REJECT_L2_SECTORS, "profiles/r2_mc_halo_reject.md"),
    "recount_table_L100_dram_bytes": (680_581_888 + 4_061_184, "profiles/r2_recount.md"),
    "recount_stencil_L100_dram_bytes": (4_028_928, "profiles/r2_recount.md"),
    # table-free recount on fcc 100^3, batch 1: smsp__inst_executed.sum of one launch
    "recount_stencil_L100_warp_instr": (17_792_245, "profiles/r2_recount.md"),
}


# ALU-issue model of one swap trial: thread-instructions the method needs per candidate.
def mc_ops_per_trial(Z, S, M):
    philox = 10 * 4 + 4                 # 10 rounds x (2 wide multiplies + 2 three-input xors) + 4 bounded draws
    gather = 2 * Z * 5                  # per neighbour entry: index, species load, 2 compares folded, shift, add
    objective = S * M * M * 6 + S * M + S * 2   # per cell: cvt, mul, sub, sub, mul, add; row/shell/weight combines
    return philox + gather + objective


def stencil_ops_per_atom(Z, S, M):
    """Thread-instructions the table-free recount needs per atom as it is formulated: Z/2 shared-memory
    loads and Z/2 adds of the half-shell histogram, per shell and wide word one extract and M multiply-adds of the row
    select (2 words for M <= 5, 4 above), M own-species flags."""
    nw = 2 if M <= 5 else 4
    return Z // 2 + Z // 2 + S * nw * (1 + M) + M


def issue_peak(n_sms, sm_mhz):
    """T thread-instr/s: SMs x 128 lanes/clk x clock."""
    return n_sms * 128 * sm_mhz * 1e6 / 1e12


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
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
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.t.join(timeout=2)
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------ oracle legs (CPU)
def oracle_mc_sample(w, n_chains, n_steps, threads):
    """Times the oracle (all K candidates evaluated every step) on n_chains x n_steps of workload w."""
    from oracle import hea_oracle
    o = hea_oracle.Oracle(*w.create_args())
    occ = o.init_random(n_chains, w.seed)
    cnt, _, _ = o.sro_full(occ, n_threads=threads)
    t0 = time.perf_counter()
    o.sro_full(occ, n_threads=threads)
    t_rc = time.perf_counter() - t0
    t0 = time.perf_counter()
    o.mc_run(occ, cnt, n_steps, w.K, w.seed, n_threads=threads, eval_all=True)
    t_mc = time.perf_counter() - t0
    return t_rc, t_mc, min(threads, n_chains)


def cpu_baseline(w, budget_s=12.0):
    cores = os.cpu_count() or 1
    n_chains = w.n_chains
    t_rc, t_mc, used = oracle_mc_sample(w, n_chains, 200, cores)          # calibration
    n_steps = int(max(200, min(2_000_000, 200 * budget_s / max(t_mc, 1e-6))))
    t_rc, t_mc, used = oracle_mc_sample(w, n_chains, n_steps, cores)
    trials = n_chains * n_steps * w.K
    return {"value": trials / (t_rc + t_mc), "unit": UNIT, "cores": used, "kind": "oracle",
            "sample": f"{n_chains} chains x {n_steps} MC steps x K={w.K} of c4 (all K evaluated) after one recount of "
                      f"the {n_chains} configurations; oracle/hea_oracle.c, gcc -O2, one thread per chain",
            "mc_trials_per_s": trials / t_mc, "recount_atoms_per_s": n_chains * w.n_sites / t_rc,
            "seconds": t_rc + t_mc}


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same metric/config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2411_18906_b200 import workloads
    w = workloads.config(4)
    cores = os.cpu_count() or 1
    n_steps = args.ref_mc_steps
    for _ in range(args.warmup):
        oracle_mc_sample(w, w.n_chains, max(1, n_steps // 10), cores)
    t_all, used = 0.0, 1
    for _ in range(args.steps):
        t_rc, t_mc, used = oracle_mc_sample(w, w.n_chains, n_steps, cores)
        t_all += t_rc + t_mc
    trials = w.n_chains * n_steps * w.K
    value = trials * args.steps / t_all
    sample = (f"per step: one recount of {w.n_chains} configurations + {n_steps} MC steps x K={w.K} on "
              f"{w.n_chains} chains of c4 (all K evaluated)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_all / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32 counts + f64 objective (the oracle: D6 order, no FMA, no filter)", "data": "synthetic",
        "config": {"workload": "c4: fcc 40x40x40 (256,000 atoms), 4 species 0.25 each, shells 1-2, target seed 11, "
                               "16 chains, K=128", "mc_steps_per_step": n_steps,
                   "sample": f"the FIRST {n_steps} steps of the 1e7-step trajectory (accept regime), all K evaluated; the "
                             "GPU arm runs the whole trajectory"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))



# ------------------------------------------------------------------------------------------ configs[4]: throughput sweeps
def run_sweep(args):
    """BASELINE.json:configs[4]: full-SRO recount on fcc L^3 (L = 10..100) x batch 1..1024, and the MC chain-count sweep
    1..65,536 chains on the 2,000-atom bcc cell (steady state after a warm-up run).  Prints one JSON object; not the
    driver's bench line."""
    import torch
    from paper_2411_18906_b200 import binding, workloads
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    hbm_peak, _, _ = load_peaks()
    out = {"sweep": "configs[4]", "recount": [], "mc_chains": []}
    for L in workloads.RECOUNT_SWEEP_L:
        wr = workloads.recount_sweep_workload(L, 1)
        hr = binding.Hea(*wr.create_args(), device=0)
        Z = sum(hr.z)
        for B in workloads.RECOUNT_SWEEP_B:
            if B * hr.N > (6 << 30):
                continue
            occ = hr.init_random(B, wr.seed)
            cnt = torch.empty((B, hr.S, hr.M, hr.M), dtype=torch.int32, device=dev)
            reps = max(3, min(50, int(2e9 // (B * hr.N)) or 3))
            t_eng = {}
            for engine in (1, 2):                      # 1 = table-driven kernel, 2 = table-free stencil kernel (default)
                hr.set_option("sro_engine", engine)
                for _ in range(2):
                    hr.sro_full(occ, counts=cnt, want_alpha=False, want_obj=False)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                for _ in range(reps):
                    hr.sro_full(occ, counts=cnt, want_alpha=False, want_obj=False)
                e1.record()
                torch.cuda.synchronize()
                t_eng[engine] = e0.elapsed_time(e1) * 1e-3 / reps
            t = t_eng[1]
            table_bytes, occ_bytes = 4 * Z * hr.N, B * hr.N
            out["recount"].append({"L": L, "atoms": hr.N, "batch": B, "us": 1e6 * t, "atoms_per_s": B * hr.N / t,
                                   "model_GBps_table_once": (table_bytes + occ_bytes) / t / 1e9,
                                   "frac_hbm_table_once": (table_bytes + occ_bytes) / t / 1e9 / hbm_peak,
                                   "table_MB": table_bytes / 1e6,
                                   "stencil_us": 1e6 * t_eng[2], "stencil_atoms_per_s": B * hr.N / t_eng[2],
                                   "stencil_frac_issue": B * hr.N / t_eng[2] * stencil_ops_per_atom(Z, hr.S, hr.M) / 1e12
                                   / issue_peak(148, 1965.0)})
            del occ, cnt
        hr.close()
    for C in workloads.CHAIN_SWEEP_C:
        wm = workloads.chain_sweep_workload(C)
        hm = binding.Hea(*wm.create_args(), device=0)
        occ = hm.init_random(C, wm.seed)
        cnt, _, _ = hm.sro_full(occ, want_alpha=False, want_obj=False)
        st = hm.new_stats(C)
        n_warm, n_time = 20_000, 20_000
        hm.mc_run(occ, cnt, n_warm, wm.K, wm.seed, stats=st)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a0 = int(binding.stats_to_numpy(st)["n_accept"].sum())
        e0.record()
        hm.mc_run(occ, cnt, n_time, wm.K, wm.seed, step0=n_warm, stats=st)
        e1.record()
        torch.cuda.synchronize()
        t = e0.elapsed_time(e1) * 1e-3
        a1 = int(binding.stats_to_numpy(st)["n_accept"].sum())
        out["mc_chains"].append({"chains": C, "mc_steps": n_time, "K": wm.K, "ms": 1e3 * t,
                                 "trials_per_s": C * n_time * wm.K / t, "us_per_step": 1e6 * t / n_time,
                                 "accept_rate": (a1 - a0) / (C * n_time)})
        hm.close()
    print(json.dumps(out))

def run_configs(args):
    """BASELINE.json configs c1..c4 as configured (full length from the seeded start, all chains, one hea_mc_run call
    each): device time, trials/s, accept rate.  Prints one JSON object; not the driver's bench line."""
    import torch
    from paper_2411_18906_b200 import binding, workloads
    torch.cuda.set_device(0)
    out = {"configs": []}
    for ci in (1, 2, 3, 4, 0):
        w = workloads.config(ci) if ci else workloads.large_m_workload()     # 0: the cell only the window engine holds
        h = binding.Hea(*w.create_args(), device=0)
        for kv in args.opt:
            name, val = kv.split("=")
            h.set_option(name, int(val))
        best = None
        for rep in range(3):
            occ = h.init_random(w.n_chains, w.seed)
            e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            e[0].record()
            cnt, _, _ = h.sro_full(occ)
            e[1].record()
            st, _ = h.mc_run(occ, cnt, w.n_steps, w.K, w.seed)
            e[2].record()
            torch.cuda.synchronize()
            t_rc, t_mc = e[0].elapsed_time(e[1]) * 1e-3, e[1].elapsed_time(e[2]) * 1e-3
            if best is None or t_mc < best[1]:
                best = (t_rc, t_mc)
        stn = binding.stats_to_numpy(st)
        trials = w.n_chains * w.n_steps * w.K
        out["configs"].append({"config": w.name, "lattice": w.lattice, "dims": list(w.dims), "atoms": w.n_sites,
                               "species": w.n_species, "shells": w.n_shells, "chains": w.n_chains, "steps": w.n_steps, "K": w.K,
                               "recount_us": 1e6 * best[0], "mc_ms": 1e3 * best[1], "trials": trials,
                               "trials_per_s": trials / best[1], "us_per_step": 1e6 * best[1] / w.n_steps,
                               "accept_rate": float(stn["n_accept"].sum()) / (w.n_chains * w.n_steps),
                               "null_rate": float(stn["n_null"].sum()) / trials,
                               "last_accept_step_max": int(stn["last_accept_step"][stn["n_accept"] > 0].max()),
                               "J_mean": float(stn["J"].mean()), "J_max": float(stn["J"].max())})
        h.close()
    print(json.dumps(out))


def run_peaks(args):
    import torch
    from paper_2411_18906_b200 import binding, workloads
    torch.cuda.set_device(0)
    h = binding.Hea(*workloads.config(1).create_args(), device=0)
    print(json.dumps({"measured_peaks": h.measure_peaks(), "how": "hea_measure_peaks (csrc/hea_peaks.cu): one 512-thread block "
                      "per SM, best of 3, CUDA events"}))


# ------------------------------------------------------------------------------------------ GPU arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--mc-steps", type=int, default=0, help="MC steps per chain per bench step (0 = the whole trajectory of the config: 1e7 for c4)")
    ap.add_argument("--ref-mc-steps", type=int, default=2_000, help="MC steps per bench step of the reference arm")
    ap.add_argument("--recount-L", type=int, default=100, help="fcc L^3 cells of the recount roofline point")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-recount", action="store_true")
    ap.add_argument("--workload", type=int, default=4, help="BASELINE.json config 1..4 (default 4 = the metric's)")
    ap.add_argument("--chains", type=int, default=0, help="override the chain count (exploration only)")
    ap.add_argument("--opt", action="append", default=[], help="tuning option name=value (hea_set_option)")
    ap.add_argument("--sweep", action="store_true", help="run the configs[4] throughput sweeps instead of the bench step")
    ap.add_argument("--configs", action="store_true", help="time configs c1..c4 as configured instead of the bench step")
    ap.add_argument("--peaks", action="store_true", help="run the library's roofline micro-benchmarks and print them")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        args.warmup = 3                                   # timing rule: W >= 3
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.configs:
        return run_configs(args)
    if args.peaks:
        return run_peaks(args)

    import torch
    import torch.distributed as dist
    from paper_2411_18906_b200 import binding, sharding, workloads

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libhea_b200 has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    # under torchrun (RANK / WORLD_SIZE / MASTER_* in the environment) the process group is created even for one rank, so
    # that `torchrun --nproc-per-node 1 bench.py` exercises the NCCL plumbing (barrier, MAX all-reduce of the times) on one GPU
    use_dist = world > 1 or ("RANK" in os.environ and "MASTER_ADDR" in os.environ)
    if use_dist:
        dist.init_process_group("nccl", device_id=dev)
    hbm_peak, sm_max_mhz, peak_src = load_peaks()

    w = workloads.config(args.workload) if not args.chains else workloads.config(args.workload, n_chains=args.chains)
    h = binding.Hea(*w.create_args(), device=local_rank)
    for kv in args.opt:
        k, v = kv.split("=")
        h.set_option(k, int(v))
    C, K, N = w.n_chains, w.K, w.n_sites
    n_mc = args.mc_steps if args.mc_steps > 0 else w.n_steps
    SMM = h.S * h.M * h.M
    chain0, _ = sharding.weak_chain_range(rank, C)
    occ_init = h.init_random(C, w.seed, chain0)                           # the seeded random start of the config
    occ = occ_init.clone()
    counts = torch.empty((C, h.S, h.M, h.M), dtype=torch.int32, device=dev)
    stats = h.new_stats(C)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2

    def one_step(ev=None):
        # one pass of the whole hot path over the batch: recount of the C start configurations, then the whole MC
        # trajectory of every chain from step 0.  Restoring the start and resetting the stats is not part of the path.
        occ.copy_(occ_init)
        h.reset_stats(stats)
        if ev: ev[0].record()
        h.sro_full(occ, counts=counts)
        if ev: ev[1].record()
        h.mc_run(occ, counts, n_mc, K, w.seed, chain0=chain0, step0=0, stats=stats)
        if ev: ev[2].record()

    def barrier():
        torch.cuda.synchronize()
        if use_dist:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    l0 = h.launch_count()
    barrier()
    t_wall0 = time.perf_counter()
    for i in range(args.steps):
        flush.fill_(i & 0xFF)                              # L2 flush between timed iterations (outside the events)
        one_step(evs[i])
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = h.launch_count() - l0 - args.steps          # minus the stats resets (outside the events)
    t_rc = sum(e[0].elapsed_time(e[1]) for e in evs) * 1e-3
    t_mc = sum(e[1].elapsed_time(e[2]) for e in evs) * 1e-3
    t_dev = t_rc + t_mc
    st1 = binding.stats_to_numpy(stats).copy()

    # sanity outside the timed region: the incremental counts equal a fresh recount of the final occupancies
    chk, _, _ = h.sro_full(occ)
    assert bool((chk == counts).all()), "incremental counts diverged from the recount"

    # ---- the two regimes of the trajectory, timed separately (information, not the metric): the first steps from the
    # random start (accept regime: nearly every step applies a move) and steps after the whole trajectory (reject regime)
    def timed_mc(n, step0):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        h.mc_run(occ, counts, n, K, w.seed, chain0=chain0, step0=step0, stats=stats)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3
    n_tail = min(1_000_000, max(1000, n_mc // 10))
    a0 = int(st1["n_accept"].sum())
    t_tail = timed_mc(n_tail, n_mc)
    a1 = int(binding.stats_to_numpy(stats)["n_accept"].sum())
    n_head = min(20_000, n_mc)
    occ.copy_(occ_init); h.reset_stats(stats); h.sro_full(occ, counts=counts)
    t_head = timed_mc(n_head, 0)
    a2 = int(binding.stats_to_numpy(stats)["n_accept"].sum())
    regimes = {"first_steps": {"mc_steps": n_head, "trials_per_s": world * C * n_head * K / t_head,
                               "us_per_step": 1e6 * t_head / n_head, "accept_rate": a2 / (C * n_head)},
               "after_trajectory": {"mc_steps": n_tail, "trials_per_s": world * C * n_tail * K / t_tail,
                                    "us_per_step": 1e6 * t_tail / n_tail, "accept_rate": (a1 - a0) / (C * n_tail)}}

    # ---- e2e: host buffers through hea_mc_run_host, copies inside the timed region
    occ_host0 = occ_init.cpu()
    occ_host = torch.empty((C, N), dtype=torch.uint8).pin_memory()
    occ_np = occ_host.numpy()
    cnt_host = np.empty((C, h.S, h.M, h.M), dtype=np.int32)
    for _ in range(1):
        occ_host.copy_(occ_host0)
        st_host = binding.fresh_stats_host(C)
        h.mc_run_host(occ_np, n_mc, K, w.seed, chain0=chain0, step0=0, stats=st_host, counts_out=cnt_host)
    barrier()
    t_e2e = 0.0
    for _ in range(args.steps):
        occ_host.copy_(occ_host0)
        st_host = binding.fresh_stats_host(C)
        t0 = time.perf_counter()
        h.mc_run_host(occ_np, n_mc, K, w.seed, chain0=chain0, step0=0, stats=st_host, counts_out=cnt_host)
        torch.cuda.synchronize()
        t_e2e += time.perf_counter() - t0
    assert (st_host["hash"] == st1["hash"]).all(), "host-buffer path and device path disagree"
    clocks = sampler.stop()
    h2d = C * N + 40 * C
    d2h = C * N + 4 * SMM * C + 40 * C

    # ---- recount roofline point: table larger than L2 (inputs > L2, so no flush needed)
    recount = recount_stencil = None
    if not args.no_recount:
        wr = workloads.recount_sweep_workload(args.recount_L, 1)
        hr = binding.Hea(*wr.create_args(), device=local_rank)
        occ_r = hr.init_random(1, wr.seed)
        cnt_r = torch.empty((1, hr.S, hr.M, hr.M), dtype=torch.int32, device=dev)
        def time_recount(engine, reps=10):
            hr.set_option("sro_engine", engine)
            for _ in range(3):
                hr.sro_full(occ_r, counts=cnt_r, want_alpha=False, want_obj=False)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps):
                hr.sro_full(occ_r, counts=cnt_r, want_alpha=False, want_obj=False)
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) * 1e-3 / reps

        t_r = time_recount(1)                      # table-driven kernel: the HBM-bound one
        ref_r = cnt_r.clone()
        t_s = time_recount(2)                      # table-free stencil kernel (what hea_sro_full runs by default)
        assert bool((cnt_r == ref_r).all()), "recount engines disagree"
        Zr = sum(hr.z)
        bytes_r = (4 * Zr + 1) * hr.N
        recount = {"bound": "hbm", "achieved": bytes_r / t_r / 1e9, "peak": hbm_peak, "unit": "GB/s",
                   "frac": bytes_r / t_r / 1e9 / hbm_peak,
                   "traffic": NCU["recount_table_L100_dram_bytes"][0] if args.recount_L == 100 else None,
                   "traffic_source": NCU["recount_table_L100_dram_bytes"][1], "peak_source": peak_src,
                   "kernel": "sro_count_kernel (sro_engine = 1)", "workload": f"fcc {args.recount_L}^3 ({hr.N} atoms), 5 species, "
                   f"3 shells (Z={Zr}), batch 1; table {4 * Zr * hr.N / 1e6:.0f} MB > L2",
                   "bytes_per_atom": 4 * Zr + 1, "atoms_per_s": hr.N / t_r, "ms_per_launch": t_r * 1e3}
        ops_s = stencil_ops_per_atom(Zr, hr.S, hr.M)
        sm_mhz_r = float(clocks.get("sm_max_mhz") or 1965.0)
        n_sms_r = torch.cuda.get_device_properties(dev).multi_processor_count
        recount_stencil = {"bound": "alu", "achieved": hr.N / t_s * ops_s / 1e12, "peak": issue_peak(n_sms_r, sm_mhz_r),
                           "unit": "T thread-instr/s", "frac": hr.N / t_s * ops_s / 1e12 / issue_peak(n_sms_r, sm_mhz_r),
                           "traffic": NCU["recount_stencil_L100_dram_bytes"][0] if args.recount_L == 100 else None,
                           "traffic_source": NCU["recount_stencil_L100_dram_bytes"][1],
                           "kernel": "sro_stencil_kernel (sro_engine = 2, the default)", "ops_per_atom": ops_s,
                           "workload": f"fcc {args.recount_L}^3 ({hr.N} atoms), 5 species, 3 shells, batch 1; 1 byte per atom",
                           "atoms_per_s": hr.N / t_s, "ms_per_launch": t_s * 1e3,
                           "hbm_GBps": hr.N / t_s / 1e9, "speedup_vs_table_kernel": t_r / t_s,
                           "peak_source": "SMs x 128 lanes/clk x max SM clock (DESIGN.md section 6)",
                           "executed_warp_instr_per_launch": NCU["recount_stencil_L100_warp_instr"][0] if args.recount_L == 100 else None,
                           "executed_source": NCU["recount_stencil_L100_warp_instr"][1]}
        hr.close()

    # ---- reduce over ranks: max time
    times = torch.tensor([t_dev, t_rc, t_mc, t_e2e, t_wall], dtype=torch.float64, device=dev)
    if use_dist:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
    t_dev, t_rc, t_mc, t_e2e, t_wall = [float(x) for x in times.cpu()]
    trials_per_step = world * C * n_mc * K
    value = trials_per_step * args.steps / t_dev
    ops = mc_ops_per_trial(sum(h.z), h.S, h.M)
    n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    alu_peak = n_sms * 128 * sm_max_mhz * 1e6 / 1e12                    # nominal: 4 SMSPs x 32 lanes / clk
    mc_rate_1gpu = C * n_mc * K * args.steps / t_mc
    # ---- roofline of the dominant kernel (mc_halo_kernel).  The kernel moves no HBM bytes in steady state; what binds it is
    # instruction issue, the shared-memory data pipe and (long windows) the random L2 sectors of the site-histogram table.  Denominators: this box's own micro-benchmarks (hea_measure_peaks).
    # achieved = warp-instructions the kernel EXECUTES per launch (ncu, committed profile) x 32 / measured launch duration.
    peaks = h.measure_peaks()
    is_metric_run = args.workload == 4 and not args.chains and n_mc == w.n_steps
    full_instr, full_src = NCU["mc_c4_full_warp_instr"]
    rej_instr, rej_src = NCU["mc_reject_warp_instr_per_32_trials"]
    rej_wf, _ = NCU["mc_reject_smem_wavefronts_per_32_trials"]
    rej_l2, _ = NCU["mc_reject_l2_sectors_per_32_trials"]
    issue_peak_T = peaks["issue_instr_per_s"] / 1e12
    t_launch = t_mc / args.steps
    achieved_T = full_instr * 32 / t_launch / 1e12 if is_metric_run else None
    rej_rate = regimes["after_trajectory"]["trials_per_s"] / world
    reject_roof = {
        "issue": {"achieved": rej_rate * rej_instr / 1e12, "peak": issue_peak_T, "unit": "T thread-instr/s",
                  "frac": rej_rate * rej_instr / 1e12 / issue_peak_T},
        "smem_pipe": {"achieved": rej_rate / 32 * rej_wf / 1e12, "peak": peaks["lds_wavefronts_per_s"] / 1e12,
                      "unit": "T wavefronts/s", "frac": rej_rate / 32 * rej_wf / peaks["lds_wavefronts_per_s"]},
        # random 32-byte sectors of the site-histogram table against the measured random-sector rate
        "l2_sectors": {"achieved": rej_rate / 32 * rej_l2 / 1e12, "peak": peaks["l2_random_sector_GBps"] * 1e9 / 32 / 1e12,
                       "unit": "T sectors/s", "frac": rej_rate / 32 * rej_l2 / (peaks["l2_random_sector_GBps"] * 1e9 / 32)},
        "per_32_trials": {"warp_instr": rej_instr, "smem_wavefronts": rej_wf, "l2_sectors": rej_l2, "source": rej_src},
        # what the measured denominators allow for this formulation: the lowest of the three per-resource limits
        "trials_per_s_bound": min(peaks["issue_instr_per_s"] / rej_instr, peaks["lds_wavefronts_per_s"] * 32 / rej_wf,
                                  peaks["l2_random_sector_GBps"] * 1e9 / 32 * 32 / rej_l2),
        "trials_per_s": rej_rate}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": DTYPE, "data": "synthetic",
        "config": {"workload": "c4: fcc 40x40x40 (256,000 atoms), 4 species 0.25 each, shells 1-2 (w 1, 0.5), "
                               "first-shell target in [-0.2, 0.2] from seed 11, 16 chains per GPU, K=128, chain seed 4",
                   "mc_steps_per_step": n_mc, "chains_per_gpu": C, "K": K, "l2": "flushed between timed iterations "
                   "(256 MB fill, outside the events)", "parallelism": f"chains sharded, {world} rank(s), no collective"},
        "recount_atoms_per_s": world * C * N * args.steps / t_rc,
        "mc_trials_per_s": world * mc_rate_1gpu,
        "accept_rate": float(st1["n_accept"].sum()) / (C * n_mc),
        "null_rate": float(st1["n_null"].sum()) / (C * n_mc * K),
        "regimes": regimes,
        "J_mean": float(st1["J"].mean()),
        "wall_ms_per_step_incl_flush": 1e3 * t_wall / args.steps,
        "clocks": clocks,
        "e2e": {"value": trials_per_step * args.steps / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "api": "hea_mc_run_host (pinned host occupancies)"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "achieved": achieved_T, "peak": issue_peak_T, "unit": "T thread-instr/s",
                     "frac": (achieved_T / issue_peak_T) if achieved_T else None,
                     "traffic": NCU["mc_c4_full_dram_bytes"][0] if is_metric_run else None,
                     "traffic_source": NCU["mc_c4_full_dram_bytes"][1],
                     "kernel": "mc_halo_kernel (whole launch: accept regime + reject regime)", "ms_per_launch": 1e3 * t_launch,
                     "executed_warp_instr_per_launch": full_instr if is_metric_run else None, "executed_source": full_src,
                     "peak_source": "measured on this box: hea_measure_peaks, LOP3 + IMAD interleaved on every SM (issue ceiling)",
                     "reject_regime": reject_roof,
                     "model": {"ops_per_trial": ops, "achieved": mc_rate_1gpu * ops / 1e12, "nominal_peak": alu_peak,
                               "frac_of_nominal": mc_rate_1gpu * ops / 1e12 / alu_peak,
                               "note": "round-1 figure: thread-instructions the method needs per trial (DESIGN.md 6) against "
                                       f"{n_sms} SMs x 128 lanes/clk x {sm_max_mhz:.0f} MHz"}},
        "measured_peaks": peaks,
    }
    if args.workload != 4 or args.chains:
        line["config"]["workload"] = f"EXPLORATION (not the metric's workload): {w.name}, {C} chains, K={K}, N={N}"
    if recount:
        if recount_stencil.get("executed_warp_instr_per_launch"):
            ex_T = recount_stencil["executed_warp_instr_per_launch"] * 32 / (recount_stencil["ms_per_launch"] * 1e-3) / 1e12
            recount_stencil["executed"] = {"achieved": ex_T, "peak": issue_peak_T, "unit": "T thread-instr/s",
                                           "frac": ex_T / issue_peak_T, "peak_source": "measured issue ceiling (hea_measure_peaks)"}
        line["recount_roofline"] = recount
        line["recount_stencil"] = recount_stencil
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w)
        print(json.dumps(line))
    if use_dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
