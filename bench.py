#!/usr/bin/env python
"""bench.py -- population-annealing hot path on B200 (arxiv 2006.00561), driver contract.

    python bench.py --gpus N --steps K --warmup W            # our CUDA path (default N=1, config 3)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle as it stands (reference arm)

A "step" is one pa_step: Q/tau reduction, Poisson resampling, scan, partition balance, replica copy, theta
Metropolis sweeps, observables.  Workload: BASELINE.json configs[2] ("config 3": L=64, R0=2^21, dbeta=0.005,
theta=10, P=148) -- the paper's own workload shape on one GPU; its population (1 GiB)
is larger than L2.  metric = spin-flip attempts/s over the whole step.  The resampling/redistribution path
(config 5, theta=0) is measured in the same run and reported under "resample".  N > 1: ONE population of N x R0 replicas sharded over the N GPUs, rank =
partition (the paper's partitioned redistribution): weak scaling.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2006_00561_b200 import inputs  # noqa: E402

# Roofline of the sweep kernel: bound by the integer datapath of an SMSP, which retires the
# kernel's two instruction classes -- LOP3 (ALU pipe) and IMAD.WIDE.U32 (FMA-heavy pipe; Philox's 32 x 32 -> 64 multiplies)
# -- TOGETHER at one warp instruction per 2 cycles = 16 lanes/clk/SMSP.  Evidence: profiles/r3_pipe_probe_ncu.md (mixes of
# the two at the sweep kernel's occupancy: 16 IMAD.WIDE + 32 LOP3 take 98 cycles, not 64; under ncu the pipes' active
# cycles ADD to 98-99 % while smsp__issue_active stays at 49-50 %).
# Algorithmic lane-operations per flip attempt of the bit-sliced lazy comparator (reading G20), per plane word of 32 sites:
# E_BLK Philox blocks x (16 IMAD.WIDE + 19 LOP3 of Philox4x32-10 with the loop-invariant first round hoisted + 8 LOP3 of the
# comparator specialised on the threshold bits, 2 per bit) + 9 per word (neighbour classes 7, flip mask 1, flip 1);
# E_BLK = 2 + sum_{c>=2} [1 - (1 - 2^-4c)^32] = 2.126 blocks that a (lane, word) pair needs when every site of the word
# needs a uniform.  -> 3.138 per attempt: `roofline.frac`.  `roofline.frac_alu_pipe_only` leaves the IMAD.WIDE out (2.075 per
# attempt against the same 16 lanes/clk: what the ALU pipe alone would allow if the multiplies were free -- they are not).
E_BLK = 2.0 + sum(1.0 - (1.0 - 2.0 ** (-4 * c)) ** 32 for c in range(2, 8))
ALU_OPS_PER_ATTEMPT = (E_BLK * (19 + 8) + 9) / 32.0
INT_OPS_PER_ATTEMPT = (E_BLK * (16 + 19 + 8) + 9) / 32.0
I_MIN_SURVEY = 12.0   # one 32-bit Philox word per attempt at 1 warp-instr/clk/SMSP (kept for continuity)
SM_COUNT, SMSP, LANES, ALU_LANES = 148, 4, 32, 16
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the `ncu --set full` captures.  These are CAPTURED
# constants, not something this run measures: each carries the profiles/ file it was read from and the commit the
# captured library was built from, and the bench line prints both (`traffic_src`) so that a stale figure is visible.
# Reported only for the workload it was captured on.
NCU_SWEEP_CAPTURE_COMMIT = "8ae95eb"
NCU_CAPTURE_COMMIT = "b3dc885"
# config 3, one launch of k_sweep<64> = gather + theta sweeps of R' ~ 2^21 replicas (algorithmic S*(U + R') + 8R')
NCU_TRAFFIC_BYTES = {("k_sweep<64>", 3): 0.652404e9 + 1.032230e9}
NCU_TRAFFIC_SRC = {"file": "profiles/r2_sweep64_ncu.md", "commit": NCU_SWEEP_CAPTURE_COMMIT}
# executed lane-instructions per flip attempt (smsp__inst_executed.sum x 32 / attempts of the captured launch): the
# distance to the 3.138 algorithmic ones is the kernel's overhead (queue, shuffles, moves, branches)
NCU_LANE_INSTR_PER_ATTEMPT = {("k_sweep<64>", 3): 4.26}
# a1-a6 chain of config 5: q_reduce (+ level tables) + poisson_scan + copy, read + write
NCU_RESAMPLE_TRAFFIC_BYTES = 67.15e6 + (67.25e6 + 20.55e6) + (604.61e6 + 2156.73e6)
NCU_RESAMPLE_TRAFFIC_SRC = {"file": "profiles/r2_resample_ncu.md", "commit": NCU_CAPTURE_COMMIT}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "src": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu, self.proc, self.lines = gpu_index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._pump, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
                pw.append(float(f[3]))
            except ValueError:
                continue
            for nm, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def schedule(wl, first_step, count):
    dbeta = (wl.beta_K - wl.beta0) / wl.K
    return [wl.beta0 + dbeta * k for k in range(first_step, first_step + count)]


# ---------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of our arm; the whole reference arm)
# ---------------------------------------------------------------------------------------------------
def oracle_sample_run(wl, R_sample, steps, warmup, threads=None):
    """the oracle, as it stands, on a bounded sample of the workload: same L, dbeta, theta, P; R = R_sample"""
    from oracle import pa_oracle as orc
    all_cores = orc.max_threads()
    if threads:
        orc.set_threads(threads)
    cores = threads or all_cores
    small = wl.scaled(R_sample)
    pa = orc.OraclePA(small.L, small.R0, P=small.P, seed=small.seed, beta0=small.beta0)
    betas = schedule(wl, 1, warmup + steps)
    for b in betas[:warmup]:
        pa.step(b, wl.theta)
    attempts = 0
    t0 = time.perf_counter()
    for b in betas[warmup:]:
        pa.step(b, wl.theta)
        attempts += wl.theta * wl.N * pa.R
    dt = time.perf_counter() - t0
    if threads:
        orc.set_threads(all_cores)
    return {"attempts": attempts, "seconds": dt, "cores": cores, "R_sample": R_sample, "steps": steps,
            "lnZ": pa.lnZ}


def oracle_resample_run(R_sample):
    """the oracle's a1-a6 (Q, tau, Poisson counts, scan, partition table, gather copy) on a bounded sample of config 5;
    the population is built (untimed) by the oracle itself"""
    from oracle import pa_oracle as orc
    wl = inputs.CONFIGS[5].scaled(R_sample)
    pa = orc.OraclePA(wl.L, wl.R0, P=wl.P, seed=wl.seed, beta0=wl.beta0)
    t0 = time.perf_counter()
    info = pa.resample(wl.beta_K)
    dt = time.perf_counter() - t0
    return {"replicas": info["Rnew"], "seconds": dt, "cores": orc.max_threads(), "R_sample": R_sample}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = inputs.CONFIGS[args.config]
    if args.theta > 0:
        import dataclasses
        wl = dataclasses.replace(wl, theta=args.theta, name=wl.name + "_theta%d" % args.theta)
    R_sample = min(4096, wl.R0)
    r = oracle_sample_run(wl, R_sample, args.steps, args.warmup)
    value = r["attempts"] / r["seconds"]
    sample = "oracle on %s at R=%d (same L, dbeta, theta, P), %d steps" % (wl.name, R_sample, args.steps)
    line = {"impl": "reference", "metric": "spin_flip_attempts_per_s", "value": value, "unit": "attempts/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * r["seconds"] / max(args.steps, 1), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32+f64", "data": "synthetic",
            "config": {"workload": wl.name + " (bounded sample R=%d)" % R_sample, "L": wl.L, "theta": wl.theta, "P": wl.P},
            "cpu_baseline": {"value": value, "unit": "attempts/s", "cores": r["cores"], "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "attempts/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def resample_leg(binding, torch, peaks, repeats=5):
    """config 5: a1-a6 only (theta=0) on R=2^24 L=32 lattices; algorithmic bytes S*(U+R') + 28*R per step"""
    wl = inputs.CONFIGS[5]
    S = wl.bytes_per_replica
    times, spans, res = [], [], None
    for rep in range(2 * repeats + 2):  # a fresh context per repeat: same parents, same step (pa_init is deterministic)
        # odd repeats: events around every kernel (breakdown); even repeats: only the a1-a6 span pair, so that the kernels
        # are launched back to back with programmatic dependent launch as in an unprofiled run (the headline span)
        span_only = rep % 2 == 0
        pa = binding.PopulationAnnealer(wl.L, wl.R0, P=wl.P, seed=wl.seed, beta0=wl.beta0,
                                        flags=binding.PA_PROFILE_SPAN if span_only else binding.PA_PROFILE)
        pa.profile_read()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(pa.stream)
        pa.step(wl.beta_K, 0)
        ev1.record(pa.stream)
        torch.cuda.synchronize()
        prof = pa.profile_read()
        R, Rn = pa.parents(), pa.R
        off = pa.counts_device()
        U = int(torch.count_nonzero(off[1:] != off[:-1]).item())
        k_ms = {k: v[0] for k, v in prof.items()}
        # a1-a6 as ONE span on the caller's stream (start of k_q_reduce .. end of k_copy)
        chain_ms = k_ms["resample_span"]
        k_ms["sum_of_kernels"] = sum(k_ms[k] for k in ["levels_w", "q_reduce", "levels_tau", "poisson_scan", "balance", "copy"])
        if rep >= 2:
            (spans if span_only else times).append((chain_ms, ev0.elapsed_time(ev1), k_ms))
        res = (R, Rn, U)
        del pa, off
    torch.cuda.empty_cache()
    R, Rn, U = res
    # the other resampling rules on the same population (A4b, A4c): a1-a6 span only
    rules = {}
    for name, flag in (("nearest", binding.PA_RESAMPLE_NEAREST), ("systematic", binding.PA_RESAMPLE_SYSTEMATIC)):
        tt, Rr = [], None
        for rep in range(3):
            pa = binding.PopulationAnnealer(wl.L, wl.R0, P=wl.P, seed=wl.seed, beta0=wl.beta0, flags=binding.PA_PROFILE_SPAN | flag)
            pa.profile_read()
            pa.step(wl.beta_K, 0)
            tt.append(pa.profile_read()["resample_span"][0])
            Rr = pa.R
            del pa
        rules[name] = {"ms_a1_a6_kernels": statistics.median(tt), "R_new": Rr}
    torch.cuda.empty_cache()
    chain = statistics.median(t[0] for t in spans)
    chain_profiled = statistics.median(t[0] for t in times)
    wall = statistics.median(t[1] for t in spans)
    copy_ms = statistics.median(t[2]["copy"] for t in times)
    scan_ms = statistics.median(t[2]["poisson_scan"] for t in times)
    red_ms = statistics.median(t[2]["q_reduce"] for t in times)
    alg_bytes = S * (U + Rn) + 28 * R
    copy_bytes = S * (U + Rn) + 4 * R + 8 * Rn + 8 * U  # lattices + offsets read + E,M written/read
    ksum = statistics.median(t[2]["sum_of_kernels"] for t in times)
    return {"workload": wl.name, "R": R, "R_new": Rn, "U": U, "algorithmic_bytes": alg_bytes,
            "ms_a1_a6_kernels": chain, "ms_a1_a6_with_events_between_kernels": chain_profiled,
            "ms_sum_of_kernel_durations": ksum, "ms_step_wall": wall, "ms_copy": copy_ms, "ms_poisson_scan": scan_ms,
            "ms_q_reduce": red_ms, "replicas_per_s": Rn / (chain * 1e-3), "other_rules": rules,
            "roofline": {"bound": "hbm", "achieved": alg_bytes / (chain * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                         "unit": "GB/s", "frac": alg_bytes / (chain * 1e-3) / 1e9 / peaks["hbm_gbs"],
                         "peak_src": peaks["src"], "traffic": NCU_RESAMPLE_TRAFFIC_BYTES,
                         "traffic_src": NCU_RESAMPLE_TRAFFIC_SRC,
                         "copy_kernel_GBps": copy_bytes / (copy_ms * 1e-3) / 1e9,
                         "frac_vs_8000": alg_bytes / (chain * 1e-3) / 1e9 / 8000.0}}


def e2e_leg(pa, torch, wl, first_step, steps, step_fn=None):
    """same metric through the C ABI with HOST buffers: every step uploads the population from pinned host memory
    (pa_set_spins), runs pa_step, and reads the new population + E, M back to pinned host memory."""
    room = pa.R + max(65536, pa.R // 2)  # a shard's population may grow past its initial share
    host_pop = torch.empty(room * pa.wpr, dtype=torch.int32).pin_memory()
    host_E = torch.empty(room, dtype=torch.int32).pin_memory()
    host_M = torch.empty(room, dtype=torch.int32).pin_memory()
    R = pa.R
    pa.spins_into_host_tensor(host_pop, R)
    betas = schedule(wl, first_step, steps)
    h2d = d2h = 0
    attempts = 0
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for b in betas:
        pa.set_spins_host_tensor(host_pop, R)            # H2D: R*S bytes
        h2d += R * pa.wpr * 4
        (step_fn or pa.step)(b, wl.theta)
        R = pa.R
        pa.spins_into_host_tensor(host_pop, R)           # D2H: R'*S bytes
        pa.energies_into_host_tensors(host_E, host_M, R)  # D2H: 8 R' bytes
        d2h += R * pa.wpr * 4 + 8 * R
        attempts += wl.theta * wl.N * R
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    return {"attempts": attempts, "seconds": dt, "h2d_bytes_per_step": h2d // steps, "d2h_bytes_per_step": d2h // steps}


# exact ln Z of the L x L torus at the final temperature of configs 1-4 (Kaufman closed form, 30 digits by mpmath:
# tests/golden/ising_exact.json, written by tests/golden/make_ising_exact.py; SURVEY.md 8(c) "Reference values")
EXACT_LNZ = {1: 128.715437337408418, 2: 2049.04978969008727, 3: 4202.34050797894262, 4: 19827.5021968979168}


def anneal_leg(binding, torch, configs):
    """BASELINE.json metric "anneal wall time": the whole schedule of a config queued with ONE pa_run call (no host
    round trip between steps), timed with CUDA events on the stream and with the host clock around the call."""
    out = []
    for ci in configs:
        wl = inputs.CONFIGS[ci]
        pa = binding.PopulationAnnealer(wl.L, wl.R0, P=wl.P, seed=wl.seed, beta0=wl.beta0)
        betas = [wl.beta(k) for k in range(1, wl.K + 1)]
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ev0.record(pa.stream)
        done = pa.run(betas, wl.theta)
        ev1.record(pa.stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        sec = ev0.elapsed_time(ev1) * 1e-3
        rs = pa.replica_steps()
        lz = pa.log_Z()["lnZ"]
        ob = pa.observables()
        out.append({"workload": wl.name, "steps_done": done, "K": wl.K, "theta": wl.theta, "seconds_device": sec,
                    "seconds_wall": wall, "replica_steps": rs, "attempts_per_s": wl.theta * wl.N * rs / sec,
                    "replica_steps_per_s": rs / sec, "R_final": pa.R, "lnZ": lz, "lnZ_exact": EXACT_LNZ.get(ci),
                    "lnZ_minus_exact_per_spin": (lz - EXACT_LNZ[ci]) / wl.N if ci in EXACT_LNZ else None,
                    "mean_E_per_spin": ob["mean_E"] / wl.N, "mean_absM_per_spin": ob["mean_absM"] / wl.N,
                    "launches": pa.launch_count()})
        del pa
        torch.cuda.empty_cache()
    return out


def theta1_leg(binding, torch, wl, steps=20, warmup=3):
    """theta = 1, the paper's scalability regime ("the most time of simulations is spending for the population
    re-weighting and redistribution"): the same workload with one sweep per temperature step"""
    pa = binding.PopulationAnnealer(wl.L, wl.R0, P=wl.P, seed=wl.seed, beta0=wl.beta0, flags=binding.PA_PROFILE)
    pa.run(schedule(wl, 1, warmup), 1)
    pa.profile_read()
    rs0 = pa.replica_steps()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record(pa.stream)
    pa.run(schedule(wl, warmup + 1, steps), 1)
    ev1.record(pa.stream)
    torch.cuda.synchronize()
    sec = ev0.elapsed_time(ev1) * 1e-3
    prof = pa.profile_read()
    rs = pa.replica_steps() - rs0
    total = sum(v[0] for k, v in prof.items() if k != "resample_span")
    out = {"theta": 1, "steps": steps, "attempts_per_s": wl.N * rs / sec, "ms_per_step": 1e3 * sec / steps,
           "replicas_per_s": rs / sec, "share_a1_a5_and_map": prof["resample_span"][0] / total,
           "share_sweep_incl_gather": prof["sweep"][0] / total}
    del pa
    torch.cuda.empty_cache()
    # the same steps through the multi-GPU driver with ONE rank (rank = partition protocol: four library calls, plan, pack,
    # exchange of nothing): what the sharded step costs on top of the queued one-GPU step where it matters most
    from paper_2006_00561_b200 import dist
    sh = dist.ShardedAnnealer(wl.L, wl.R0, seed=wl.seed, beta0=wl.beta0, group=dist.Group())
    for b_ in schedule(wl, 1, warmup):
        sh.step(b_, 1)
    torch.cuda.synchronize()
    t0 = time.perf_counter()  # host clock: the sharded step synchronises four times per step by construction
    for b_ in schedule(wl, warmup + 1, steps):
        sh.step(b_, 1)
    torch.cuda.synchronize()
    out["sharded_one_rank_ms_per_step"] = 1e3 * (time.perf_counter() - t0) / steps
    del sh
    torch.cuda.empty_cache()
    return out


def glass_leg(binding, torch, wl, peaks, steps=20, warmup=3):
    """SURVEY.md 8(f)-4 / PAPER.md:213: the same workload shape with the second Hamiltonian, one seeded 2D +-J spin-glass
    sample (inputs.bond_sample, P(J = -1) = 1/2) set through pa_set_bonds: flip attempts/s of the sweep kernel's +-J
    variant against the same ALU roofline, and the order-parameter histogram pa_overlap_hist (one pass over the
    population: HBM-bound)."""
    Jx, Jy = inputs.bond_sample(wl.L, wl.seed)
    pa = binding.PopulationAnnealer(wl.L, wl.R0, P=wl.P, seed=wl.seed, beta0=wl.beta0, flags=binding.PA_PROFILE)
    pa.set_bonds(inputs.pack_pm1(Jx), inputs.pack_pm1(Jy))
    pa.run(schedule(wl, 1, warmup), wl.theta)
    pa.profile_read()
    rs0 = pa.replica_steps()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record(pa.stream)
    pa.run(schedule(wl, warmup + 1, steps), wl.theta)
    ev1.record(pa.stream)
    torch.cuda.synchronize()
    sec = ev0.elapsed_time(ev1) * 1e-3
    prof = pa.profile_read()
    rs = pa.replica_steps() - rs0
    attempts = wl.theta * wl.N * rs
    sweep_rate = attempts / (prof["sweep"][0] * 1e-3)
    peak = SM_COUNT * SMSP * ALU_LANES * peaks["sm_max_mhz"] * 1e6 / 1e12
    pa.overlap_hist()  # warm-up
    t = []
    for _ in range(5):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h = pa.overlap_hist()
        t.append(time.perf_counter() - t0)
    ovl_s = statistics.median(t)  # host clock around the synchronous call: memset + kernel + (N+1)*8-byte read-back
    pairs = int(h.sum())
    q = (2.0 * torch.arange(wl.N + 1, dtype=torch.float64) - wl.N) / wl.N
    hq = torch.from_numpy(h.astype("float64"))
    out = {"workload": wl.name + " with a +-J sample (seed %d, %d of %d bonds negative)" % (wl.seed, int((Jx < 0).sum() + (Jy < 0).sum()), 2 * wl.N),
           "steps": steps, "attempts_per_s": attempts / sec, "kernel_attempts_per_s": sweep_rate,
           "roofline_frac": sweep_rate * INT_OPS_PER_ATTEMPT / 1e12 / peak,
           "roofline_frac_alu_pipe_only": sweep_rate * ALU_OPS_PER_ATTEMPT / 1e12 / peak, "ms_per_step": 1e3 * sec / steps,
           "overlap_hist": {"pairs": pairs, "seconds_call": ovl_s, "GBps": pa.R * wl.bytes_per_replica / ovl_s / 1e9,
                            "mean_abs_q": float((hq * q.abs()).sum() / max(pairs, 1)), "mean_q2": float((hq * q * q).sum() / max(pairs, 1))},
           "lnZ": pa.log_Z()["lnZ"], "beta": pa.beta_steps()[0], "mean_E_per_spin": pa.observables()["mean_E"] / wl.N}
    del pa
    torch.cuda.empty_cache()
    return out


def policies_leg(binding, torch, out_csv=None):
    """SURVEY.md 8(f)-2 / PAPER.md:94-118 (Fig. 1-2): the paper's 8-GPU task with the 8 GPUs as 8 logical partitions of
    one device, under the redistribution policies none / naive / main (blocks of 1024, maxexc 1 and 2) / balanced.
    The population, Q and copy counts are the same under every policy (the policy only draws the partition
    boundaries), so one seed gives directly comparable traces.  Per step: replicas per partition after
    redistribution.  'relative_makespan' = sum over steps of the largest partition / sum of the mean partition: the
    time a synchronous multi-GPU run would take relative to perfect balance (the paper: naive runs 1.45x longer than
    main)."""
    wl = inputs.PAPER_TASK
    runs = [("none", binding.PA_POLICY_NONE, 1024, 1), ("naive", binding.PA_POLICY_NAIVE, 1024, 1),
            ("main_maxexc1", binding.PA_POLICY_MAIN, 1024, 1), ("main_maxexc2", binding.PA_POLICY_MAIN, 1024, 2),
            ("balanced", binding.PA_POLICY_BALANCED, 1024, 1)]
    rows, summary = [], {}
    for name, pol, block, maxexc in runs:
        pa = binding.PopulationAnnealer(wl.L, wl.R0, P=wl.P, seed=wl.seed, beta0=wl.beta0, policy=pol, block=block,
                                        maxexc=maxexc)
        mx, mean, moved_total = [], [], 0
        for k in range(1, wl.K + 1):
            pa.step(wl.beta(k), wl.theta)
            _, st, moved = pa.partitions()
            cnt = [int(x) for x in st[:, 0]]
            rows.append([name, k, "%.3f" % wl.beta(k), pa.R, moved] + cnt)
            mx.append(max(cnt))
            mean.append(pa.R / wl.P)
            moved_total += moved
        peak = max(range(wl.K), key=lambda i: mx[i])
        summary[name] = {"max_partition": mx[peak], "at_step": peak + 1, "max_over_desired": mx[peak] / mean[peak],
                         "relative_makespan": sum(mx) / sum(mean), "replicas_moved_per_step": moved_total / wl.K,
                         "lnZ": pa.log_Z()["lnZ"], "block": block, "maxexc": maxexc}
        del pa
    if out_csv:
        with open(out_csv, "w") as f:
            f.write("policy,step,beta,R,moved," + ",".join("cnt%d" % p for p in range(wl.P)) + "\n")
            for r in rows:
                f.write(",".join(str(x) for x in r) + "\n")
    summary["naive_over_main_makespan"] = summary["naive"]["relative_makespan"] / summary["main_maxexc1"]["relative_makespan"]
    return {"workload": wl.name, "L": wl.L, "R0": wl.R0, "K": wl.K, "theta": wl.theta, "P": wl.P, "policies": summary}


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` without a torchrun environment: start the N ranks ourselves (one process per GPU) --
    or fail loudly; never report a single-GPU number as an N-GPU one."""
    import socket
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus:
        sys.stderr.write("bench.py: --gpus %d requested but %d CUDA device(s) visible; refusing to run fewer ranks than asked\n"
                         % (args.gpus, have))
        return 2
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_ours(args):
    import torch
    from paper_2006_00561_b200 import binding, dist
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(args)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    g = dist.init_from_env()
    if g.world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but the launcher started %d rank(s)" % (args.gpus, g.world))
    torch.cuda.set_device(g.local_rank)
    peaks = measured_peaks()
    wl = inputs.CONFIGS[args.config]
    if args.theta > 0:
        import dataclasses
        wl = dataclasses.replace(wl, theta=args.theta, name=wl.name + "_theta%d" % args.theta)
    K, W = args.steps, max(args.warmup, 0)

    # N = 1: one context, the whole schedule queued with one pa_run call.  N > 1: ONE population of N x R0 replicas
    # sharded over the ranks (rank = partition): per-GPU work is fixed as N grows (weak scaling), and
    # every step exchanges the ranks' weight sums, their offspring totals and the lattice slices that cross rank
    # boundaries (dist.ShardedAnnealer).
    use_shards = g.world > 1 or args.sharded
    if not use_shards:
        pa = binding.PopulationAnnealer(wl.L, wl.R0, P=wl.P, seed=wl.seed, beta0=wl.beta0, flags=binding.PA_PROFILE)
        run_steps = lambda betas: pa.run(betas, wl.theta)
    else:
        sharded = dist.ShardedAnnealer(wl.L, wl.R0 * g.world, seed=wl.seed, beta0=wl.beta0, group=g, flags=binding.PA_PROFILE)
        pa = sharded.shards[0]

        def run_steps(betas):
            for b in betas:
                sharded.step(b, wl.theta)
            return len(betas)
    if W > 0:
        run_steps(schedule(wl, 1, W))
    pa.profile_read()
    betas = schedule(wl, W + 1, K)
    sampler = ClockSampler(g.local_rank)
    sampler.start()
    time.sleep(0.25)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier(g)
    torch.cuda.synchronize()
    rs0, l0 = pa.replica_steps(), pa.launch_count()
    ev0.record(pa.stream)
    done = run_steps(betas)
    ev1.record(pa.stream)
    torch.cuda.synchronize()
    dist.barrier(g)
    seconds = ev0.elapsed_time(ev1) * 1e-3
    clocks = sampler.stop()
    assert done == K
    replica_steps = pa.replica_steps() - rs0
    launches = pa.launch_count() - l0
    prof = pa.profile_read()
    units = wl.theta * wl.N * replica_steps if wl.theta > 0 else replica_steps
    value, total_units, tmax = dist.aggregate_throughput(g, units, seconds)
    launches_total = int(dist.sum_over_ranks(g, launches))

    # dominant kernel: the Metropolis sweep (ALU / issue bound)
    sweep_ms, sweep_n = prof["sweep"]
    step_kernel_ms = sum(v[0] for k, v in prof.items() if k != "resample_span")
    line = None
    extra = {}
    if wl.theta > 0 and sweep_n > 0:
        attempts_per_launch = units / sweep_n
        sweep_rate = attempts_per_launch / (sweep_ms / sweep_n * 1e-3)  # attempts/s inside the kernel
        achieved = sweep_rate * INT_OPS_PER_ATTEMPT / 1e12
        peak = SM_COUNT * SMSP * ALU_LANES * peaks["sm_max_mhz"] * 1e6 / 1e12
        kkey = ("k_sweep<%d>" % wl.L, args.config)
        roof = {"bound": "alu", "achieved": achieved, "peak": peak,
                "unit": "T integer lane-ops/s (%.3f algorithmic per flip attempt: per 32-site word %.3f Philox blocks x "
                        "(16 IMAD.WIDE + 19 + 8 LOP3) + 9 LOP3)" % (INT_OPS_PER_ATTEMPT, E_BLK),
                "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get(kkey),
                "traffic_src": NCU_TRAFFIC_SRC if kkey in NCU_TRAFFIC_BYTES else None,
                "traffic_algorithmic": (2 * wl.bytes_per_replica + 8) * (replica_steps / sweep_n),  # upper bound: U = R'
                "kernel": "k_sweep<%d>" % wl.L,
                "kernel_attempts_per_s": sweep_rate, "kernel_ms_per_launch": sweep_ms / sweep_n,
                "kernel_share_of_step": sweep_ms / step_kernel_ms,
                "peak_src": "148 SM x 4 SMSP x 16 lanes/clk (LOP3 and IMAD.WIDE.U32 retire together at one warp instruction "
                            "per 2 cycles per SMSP: profiles/r3_pipe_probe_ncu.md) x %d MHz (clocks.max.sm)" % peaks["sm_max_mhz"],
                "lane_instr_per_attempt": NCU_LANE_INSTR_PER_ATTEMPT.get(kkey),
                "lane_instr_src": NCU_TRAFFIC_SRC if kkey in NCU_LANE_INSTR_PER_ATTEMPT else None,
                "frac_alu_pipe_only": sweep_rate * ALU_OPS_PER_ATTEMPT / 1e12 / peak,
                "alu_pipe_only_note": "LOP3 only (%.3f per attempt), IMAD.WIDE taken as free: lower than `frac` by construction, "
                                      "kept because rounds 1-2 reported it" % ALU_OPS_PER_ATTEMPT,
                "frac_survey_12_instr_per_attempt_at_issue_rate":
                    sweep_rate * I_MIN_SURVEY / (SM_COUNT * SMSP * LANES * peaks["sm_max_mhz"] * 1e6)}
        if clocks.get("sm_mhz"):
            roof["frac_at_measured_clock"] = achieved / (SM_COUNT * SMSP * ALU_LANES * clocks["sm_mhz"] * 1e6 / 1e12)
    else:
        roof = None
    per_kernel = {k: {"ms_total": v[0], "launches": v[1]} for k, v in prof.items()}

    e2e = cpu = resample = None
    if g.is_main or g.world > 1:
        if not args.no_e2e:
            n_e2e = max(1, min(K, 6))
            r = e2e_leg(pa, torch, wl, W + K + 1, n_e2e, sharded.step if use_shards else None)
            e2e_value, _, _ = dist.aggregate_throughput(g, r["attempts"], r["seconds"])
            e2e = {"value": e2e_value, "unit": "attempts/s", "h2d_bytes_per_step": r["h2d_bytes_per_step"],
                   "d2h_bytes_per_step": r["d2h_bytes_per_step"], "steps": n_e2e}
    lnZ = pa.log_Z()["lnZ"]
    beta_now = pa.beta_steps()[0]
    R_final = pa.R
    del pa
    if use_shards:
        del sharded
    torch.cuda.empty_cache()
    theta1 = glass = None
    if g.is_main and g.world == 1:
        if wl.theta > 1 and not args.no_resample:
            theta1 = theta1_leg(binding, torch, wl)
        if wl.theta > 0 and not args.no_resample:
            glass = glass_leg(binding, torch, wl, peaks)
        if not args.no_resample:
            resample = resample_leg(binding, torch, peaks, repeats=args.resample_repeats)
        if not args.no_cpu_baseline:
            r = oracle_sample_run(wl, 4096, 24, 1)
            cpu = {"value": r["attempts"] / r["seconds"], "unit": "attempts/s", "cores": r["cores"], "kind": "oracle",
                   "sample": "%s at R=%d (same L, dbeta, theta, P), %d steps, %.1f s" % (wl.name, r["R_sample"], r["steps"], r["seconds"])}
            r1 = oracle_sample_run(wl, 1024, 4, 1, threads=1)  # the single-thread figure beside the all-core one
            cpu["single_thread"] = {"value": r1["attempts"] / r1["seconds"], "unit": "attempts/s", "cores": 1,
                                    "sample": "%s at R=%d, %d steps, %.1f s" % (wl.name, r1["R_sample"], r1["steps"], r1["seconds"])}
            if resample is not None:
                rr = oracle_resample_run(1 << 22)
                resample["cpu_baseline"] = {"value": rr["replicas"] / rr["seconds"], "unit": "resampled replicas/s",
                                            "cores": rr["cores"], "kind": "oracle",
                                            "sample": "oracle a1-a6 on config 5 at R=2^22 (same L, beta, dbeta, P), one step, %.2f s"
                                                      % rr["seconds"]}
    if g.is_main:
        line = {"metric": "spin_flip_attempts_per_s", "value": value, "unit": "attempts/s", "n_gpus": g.world, "steps": K,
                "warmup": W, "ms_per_step": 1e3 * tmax / K, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "u32 bit-packed spins, i32 energies, f64 weights", "data": "synthetic",
                "config": {"workload": wl.name, "L": wl.L, "R0": wl.R0, "dbeta": (wl.beta_K - wl.beta0) / wl.K,
                           "theta": wl.theta, "P": wl.P, "beta_range": [betas[0], betas[-1]],
                           "parallelism": ("one context, whole schedule queued by pa_run" if not use_shards else
                                           "ONE population of %d x R0 replicas sharded over %d ranks (rank = partition): per step "
                                           "all-gather of weight sums and offspring totals + all-to-all-v of the lattice slices "
                                           "that cross rank boundaries (NCCL point-to-point)" % (g.world, g.world)),
                           "l2": "population %.0f MiB per buffer > 126 MB L2, no flush needed" % (wl.R0 * wl.bytes_per_replica / 2 ** 20)},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches_total, "roofline": roof, "cpu_baseline": cpu,
                "resample": resample, "theta1": theta1, "spin_glass": glass, "kernels": per_kernel, "anneal": {"lnZ": lnZ, "beta": beta_now, "R": R_final,
                                                                         "replica_steps": replica_steps}}
        if g.world > 1:
            line["config"]["R0"] = wl.R0 * g.world
        print(json.dumps(line))
    dist.shutdown(g)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=97,
                    help="timed steps; the default 97 + 3 warm-up steps = the whole 100-step schedule of config 3 "
                         "(beta 0 -> 0.5 across beta_c)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4])
    ap.add_argument("--theta", type=int, default=0,
                    help="override the sweeps per step of the workload (theta = 1 is the paper's scalability regime, "
                         "PAPER.md:126: resampling and redistribution dominate); 0 = the config's own theta")
    ap.add_argument("--sharded", action="store_true",
                    help="drive the step through the multi-GPU path (dist.ShardedAnnealer) even with one rank: exercises the "
                         "rank = partition protocol on a single GPU")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-resample", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--leg", default="all", choices=["all", "resample", "anneal", "policies"],
                    help="'resample': only the config-5 resampling/redistribution leg (short; used for ncu captures); "
                         "'anneal': whole anneals of --anneal-configs (wall time, ln Z against the exact value); "
                         "'policies': the paper's 8-GPU task under the redistribution policies none / naive / main")
    ap.add_argument("--anneal-configs", default="1,2,3,4")
    ap.add_argument("--resample-repeats", type=int, default=5)
    ap.add_argument("--trace-csv", default=None, help="--leg policies: write the per-step partition counts to this file")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3  # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        return run_reference(args)
    if args.leg == "anneal":
        import torch
        from paper_2006_00561_b200 import binding
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
        print(json.dumps({"anneal": anneal_leg(binding, torch, [int(x) for x in args.anneal_configs.split(",")])}))
        return 0
    if args.leg == "policies":
        import torch
        from paper_2006_00561_b200 import binding
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
        print(json.dumps({"policies": policies_leg(binding, torch, args.trace_csv)}))
        return 0
    if args.leg == "resample":
        import torch
        from paper_2006_00561_b200 import binding
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
        print(json.dumps({"resample": resample_leg(binding, torch, measured_peaks(), repeats=args.resample_repeats)}))
        return 0
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
