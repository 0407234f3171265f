#!/usr/bin/env python
"""bench.py -- one JSON line for the driver (contract: the build prompt, section 4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg 3] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path over one batch = one GA generation (App. B):
    fire_params_upload (a2)  ->  fire_simulate_batch (a3-a6)  ->  fire_fitness (a7)  [-> group stats (a8), config 4]
on the synthetic workload of BASELINE.json config 3 (1024 x 1024, 256 vectors x 8 replicates = 2,048 sims,
near the spread / no-spread transition) -- the config north_star quotes the roofline target on.

metric  = cell-neighbour trials/s: (target cell, direction) Bernoulli trials of the CA (C-4) per second.
          The numerator is counted on the device by the kernel (out_trials) and equals the oracle's counter
          (tests/test_gpu_parity.py checks that equality on every config).
value   = trials of all ranks / max-over-ranks device time of K steps, inputs resident in HBM.
e2e     = the same through fire_generation_host: pinned HOST buffers in, scores out, copies inside the timed region.
roofline= the propagation kernel (fire_propagate_kernel) alone: algorithmic bytes per launch
          (32 B per distinct target cell + 2 x H*W/8 B of state per simulation) over its
          mean launch duration, measured with CUDA events recorded by the library on the launching stream.
N > 1   : simulations are independent -> every rank runs its own generation of S sims
          (replicates r*S .. r*S+S-1 of the same vectors: other seeds, other sim ids), no data-path collective;
          one all-gather of the S x 4 B scores per step hands them to the GA's rank.  scaling = "weak" (default).
          --scaling strong: ONE generation partitioned by parameter vector: rank r uploads only its P / N
          vectors, so it builds P / N of the threshold table, and simulates their sims with batch positions as sim ids.

--backend gloo : dry run of the N > 1 logic with ranks sharing one GPU (timings then mean nothing).

--impl reference : this tier has no reference implementation; that arm times the CPU oracle (oracle/) as it
stands, on a bounded sample of the same workload, on the host cores (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "cell-neighbour trials/s"
UNIT = "trials/s"
# ncu --set full capture of the propagation kernel on the workload below: dram__bytes_read.sum + dram__bytes_write.sum per
# launch, with the commit the captured kernel was built from (profiles/README.md names the file and the command).  Refresh
# the number together with every change of the propagation kernel; None until a capture exists for that config.
NCU_TRAFFIC_BYTES = {3: 17864354000 + 212908000}      # profiles/r2_propagate_ncu.md: capture of commit 1aef2ce
NCU_TRAFFIC_SOURCE = {3: "profiles/r2_propagate_ncu.md (ncu --set full; two-phase kernel as of commit 1aef2ce)"}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ------------------------------------------------------------------------------------------ oracle arm
def oracle_sample(cfg: int, budget_sims: int):
    """The bounded sample of the workload the CPU oracle is timed on: `budget_sims` simulations taken at a constant stride over
    the whole batch (so every region of the parameter-vector axis is represented), with their own batch positions as sim ids."""
    from paper_1701_03549_b200 import workloads as wl
    w = wl.load_workload(cfg)
    n = min(budget_sims, w.S)
    idx = (np.arange(n, dtype=np.int64) * w.S) // n
    return w, idx


def time_oracle(w, idx, repeats: int = 1, nthreads: int = 0):
    """Oracle as it stands (OpenMP over sims, thresholds on demand, Eq. 2 counts per sim) on the sims `idx` of the batch.
    Returns (trials, seconds per pass, threads)."""
    from oracle import fire_oracle as orc
    orc.build()
    ls = w.landscape
    Lo = orc.Landscape(ls["veg"], ls["slope"], ls["aspect"], ls["wind"])
    ref = orc.simulate(Lo, w.ref_beta, w.ref_ignition, w.ref_seed, sim=0)["burned"]
    best = None
    trials = threads = 0
    for _ in range(repeats):
        t0 = time.perf_counter()
        r = orc.simulate_batch(Lo, w.betas, w.ignitions[idx], w.sim_param[idx], w.seeds[idx],
                               sim_index=idx.astype(np.int32), nthreads=nthreads)
        orc.fitness(ref, r["burned"], Lo.W, w.metric)
        dt = time.perf_counter() - t0
        trials, threads = int(r["trials"].sum()), int(r["threads"])
        best = dt if best is None else min(best, dt)
    return trials, best, threads


def sample_text(w, idx) -> str:
    if len(idx) == w.S:
        return f"all {w.S} simulations of {w.name} (+ Eq. 2 counts)"
    return (f"{len(idx)} of {w.S} simulations of {w.name}, every {w.S // len(idx)}th of the batch (+ Eq. 2 counts); "
            f"the rate is EXTRAPOLATED from this sample to the whole batch")


def sample_budget(cfg: int) -> int:
    # about 10-30 s of oracle work on the GPU box's 16 host threads (measured ~73 M trials/s): cfg3 mean 0.94 M trials per sim
    return {1: 64, 2: 256, 3: 1024, 4: 8192, 5: 4}[cfg]


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # the whole run (warm-up + K steps) should end within a few minutes: the per-step sample shrinks with K
    budget = sample_budget(args.cfg)
    w, idx = oracle_sample(args.cfg, max(budget // 16, min(budget, budget * 5 // max(args.steps, 1))))
    n = len(idx)
    for _ in range(min(args.warmup, 1)):                 # the oracle has no caches to warm beyond page-in
        time_oracle(w, idx[:: 16])
    per_step = []
    trials = threads = 0
    for _ in range(args.steps):
        trials, dt, threads = time_oracle(w, idx)
        per_step.append(dt)
    total = float(np.sum(per_step))
    value = trials * args.steps / total
    sample = sample_text(w, idx) + " per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": w.name, "sample": sample},
        "sims_per_s": n * args.steps / total,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md, the clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in out.splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ our arm
def run_ours(args) -> None:
    import torch
    import torch.distributed as dist

    from paper_1701_03549_b200 import build as fire_build
    from paper_1701_03549_b200 import libfire as lf
    from paper_1701_03549_b200 import workloads as wl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.backend != "nccl":
        local = local % max(torch.cuda.device_count(), 1)
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libfire has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        # NCCL's own account of the communicator (ranks, transports, NVLS) goes to stderr: stdout carries the one JSON line
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:                                            # dry run of the N > 1 logic where there are fewer GPUs than ranks
            dist.init_process_group(args.backend)
    if rank == 0:
        fire_build.build()
    if world > 1:
        dist.barrier()
    lf.load()

    cfg = args.cfg
    w = wl.load_workload(cfg)
    ls = w.landscape
    wl.validate_landscape(ls)
    S, P = w.S, w.P
    golden = json.loads((ROOT / "tests" / "golden" / f"cfg{cfg}_expected.json").read_text())

    def dev(a):
        a = np.ascontiguousarray(a)
        if a.dtype == np.uint32:
            a = a.view(np.int32)
        if a.dtype == np.uint64:
            a = a.view(np.int64)
        return torch.from_numpy(a).cuda()

    def pin(a):
        a = np.ascontiguousarray(a)
        if a.dtype == np.uint32:
            a = a.view(np.int32)
        if a.dtype == np.uint64:
            a = a.view(np.int64)
        return torch.from_numpy(a.copy()).pin_memory()

    strong = args.scaling == "strong"
    if strong:
        # ONE generation partitioned by parameter vector: rank r builds only its P / N slice of the threshold table
        # and runs the sims of those vectors, with their batch positions as sim ids (so every fire is the full batch's fire)
        sh = wl.shard_by_param(w, rank, world)
        l_betas, l_ign, l_par, seeds_np, sim_ids_np, l_index = sh.betas, sh.ignitions, sh.sim_param, sh.seeds, sh.sim_ids, sh.index
    else:
        # rank r simulates replicates r*S .. r*S+S-1 of the same population (weak scaling)
        sim_ids_np = (np.arange(S, dtype=np.int64) + rank * S).astype(np.int32)
        seeds_np = (np.uint64(cfg) << np.uint64(32)) | (np.arange(S, dtype=np.uint64) + np.uint64(rank * S))
        l_betas, l_ign, l_par, l_index = w.betas, w.ignitions, w.sim_param, np.arange(S)
        if rank == 0:
            assert (seeds_np == w.seeds).all()
    S_all, S = S, int(len(l_index))                      # S = sims of this rank from here on
    S_pad = S                                            # all_gather needs equal shards: the largest shard of any rank
    if world > 1:
        t_pad = torch.tensor([S], dtype=torch.int64, device="cuda")
        dist.all_reduce(t_pad, op=dist.ReduceOp.MAX)
        S_pad = int(t_pad.item())

    L = lf.fire_landscape_create(dev(ls["veg"]), dev(ls["slope"]), dev(ls["aspect"]), dev(ls["wind"]))
    H, Ww = L.H, L.Ww
    d_beta_ref = dev(w.ref_beta[None, :])
    d_beta = dev(l_betas)
    d_ign, d_par, d_seed, d_ids = dev(l_ign), dev(l_par), dev(seeds_np), dev(sim_ids_np)
    # the reference burnt map A: its own simulation from the stored vector, ignition and seed
    ref = torch.empty((1, H, Ww), dtype=torch.int32, device="cuda")
    lf.fire_params_upload(L, d_beta_ref)
    lf.fire_simulate_batch(L, dev(np.array([w.ref_ignition], np.int32)), dev(np.zeros(1, np.int32)),
                           dev(np.array([w.ref_seed], np.uint64)), ref, sim_ids=dev(np.zeros(1, np.int32)))
    torch.cuda.synchronize()
    burned = torch.empty((S, H, Ww), dtype=torch.int32, device="cuda")
    steps_out = torch.empty((S,), dtype=torch.int32, device="cuda")
    trials_out = torch.empty((S,), dtype=torch.int64, device="cuda")
    score_buf = torch.full((max(S_pad, S),), float("nan"), dtype=torch.float32, device="cuda")
    score = score_buf[:S]
    counts = torch.empty((S, 2), dtype=torch.int32, device="cuda")
    gathered = torch.empty((world * max(S_pad, S),), dtype=torch.float32, device="cuda") if world > 1 else None
    if w.groups:
        G, R = w.groups
        g_sums = torch.empty((G, 2), dtype=torch.int64, device="cuda")
        g_mv = torch.empty((G, 2), dtype=torch.float64, device="cuda")
        ref_area = int(np.unpackbits(ref.cpu().numpy().view(np.uint8)).sum())

    def generation():
        lf.fire_params_upload(L, d_beta)
        lf.fire_simulate_batch(L, d_ign, d_par, d_seed, burned, steps_out, trials_out, sim_ids=d_ids)
        lf.fire_fitness(L, ref[0], burned, w.metric, score, counts)
        if w.groups:
            lf.fire_fitness_group_stats(counts, ref_area, G, R, g_sums, g_mv)
        if world > 1:
            dist.all_gather_into_tensor(gathered, score_buf)

    def fence():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(ms: float) -> float:
        if world == 1:
            return ms
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(v: int) -> int:
        if world == 1:
            return v
        t = torch.tensor([v], dtype=torch.int64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return int(t.item())

    # ---- warm-up (also the correctness gate of this run: rank 0's counters must equal the oracle's stored ones)
    for _ in range(max(args.warmup, 1)):
        generation()
    fence()
    trials_rank = int(trials_out.sum().item())
    bad = 0
    if rank == 0 or strong:                              # these sims are sims of the stored config: every counter must match
        if not (trials_out.cpu().numpy().view(np.uint64) == np.array(golden["trials"], np.uint64)[l_index]).all():
            bad |= 1
        if not (steps_out.cpu().numpy().view(np.uint32) == np.array(golden["steps"], np.uint32)[l_index]).all():
            bad |= 2
        if not (counts.cpu().numpy().view(np.uint32)[:, 1] == np.array(golden["area"], np.uint32)[l_index]).all():
            bad |= 4
    elif not (0.5 * golden["totals"]["trials"] < trials_rank < 2.0 * golden["totals"]["trials"]) or \
            trials_rank == golden["totals"]["trials"]:   # other replicates of the same population: same law, other fires
        bad |= 8
    bad_any = sum_over_ranks(1 if bad else 0)
    if bad_any:
        raise RuntimeError(f"rank {rank}: counters differ from the oracle's stored values (flags {bad}; {bad_any} rank(s) failed)")
    trials_all = sum_over_ranks(trials_rank)

    # ---- device-resident timing: K steps between two events on the launching stream
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    lf.fire_set_profiling(L, True)
    launches0 = lf.fire_launch_count(L)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    phase_ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    prop_ms = []
    fence()
    ev0.record()
    for k in range(args.steps):
        if world == 1:                                   # per-phase events (cheap; same stream)
            phase_ev[k][0].record()
            lf.fire_params_upload(L, d_beta)
            phase_ev[k][1].record()
            lf.fire_simulate_batch(L, d_ign, d_par, d_seed, burned, steps_out, trials_out, sim_ids=d_ids)
            phase_ev[k][2].record()
            lf.fire_fitness(L, ref[0], burned, w.metric, score, counts)
            if w.groups:
                lf.fire_fitness_group_stats(counts, ref_area, G, R, g_sums, g_mv)
            phase_ev[k][3].record()
        else:
            generation()
        if (k + 1) % 32 == 0:                            # the library keeps at most 64 event pairs between reads
            prop_ms += lf.fire_profile_read(L)
    ev1.record()
    fence()
    ms_total = max_over_ranks(ev0.elapsed_time(ev1))
    prop_ms += lf.fire_profile_read(L)
    lf.fire_set_profiling(L, False)
    launches = lf.fire_launch_count(L) - launches0
    clocks = sampler.stop() if rank == 0 else None
    ms_per_step = ms_total / args.steps
    value = trials_all * args.steps / (ms_total * 1e-3)
    sims_per_s = sum_over_ranks(S) * args.steps / (ms_total * 1e-3)
    phases = None
    if world == 1:
        phases = {"params_upload_ms": float(np.mean([e[0].elapsed_time(e[1]) for e in phase_ev])),
                  "simulate_batch_ms": float(np.mean([e[1].elapsed_time(e[2]) for e in phase_ev])),
                  "fitness_ms": float(np.mean([e[2].elapsed_time(e[3]) for e in phase_ev]))}

    # ---- end to end: host buffers in, scores out, every step (fire_generation_host synchronises)
    h_beta, h_ign, h_par = pin(l_betas), pin(l_ign), pin(l_par)
    h_seed, h_ids, h_ref = pin(seeds_np), pin(sim_ids_np), pin(ref[0].cpu().numpy())
    h_score = torch.empty(S, dtype=torch.float32).pin_memory()
    h_counts = torch.empty((S, 2), dtype=torch.int32).pin_memory()
    h2d = sum(t.numel() * t.element_size() for t in (h_beta, h_ign, h_par, h_seed, h_ids, h_ref))
    d2h = sum(t.numel() * t.element_size() for t in (h_score, h_counts))

    def generation_host():
        lf.fire_generation_host(L, h_beta, h_ign, h_par, h_seed, h_ref, w.metric, h_score, h_counts, sim_ids=h_ids)
        if world > 1:
            score_buf[:S].copy_(h_score, non_blocking=True)
            dist.all_gather_into_tensor(gathered, score_buf)

    generation_host()
    fence()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        generation_host()
    e1.record()
    fence()
    wall_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms = max_over_ranks(max(e0.elapsed_time(e1), wall_ms))   # the call synchronises: host wall time is the honest one
    e2e_value = trials_all * args.steps / (e2e_ms * 1e-3)
    if rank == 0 and not np.array_equal(h_score.numpy().view(np.uint32), score.cpu().numpy().view(np.uint32)):
        raise RuntimeError("end-to-end scores differ from the device-resident path")

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (rank 0's launches; its workload is the stored config)
    peaks_file = ROOT / "MEASURED_PEAKS.json"
    if peaks_file.exists():
        peak, peak_src = float(json.loads(peaks_file.read_text())["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    else:
        peak, peak_src = 6650.0, "B200_PROFILING.md fallback (of fallback)"
    plane_bytes = H * Ww * 4
    alg_bytes = 32 * int(np.array(golden["distinct"], np.int64)[l_index].sum()) + 2 * plane_bytes * S
    k_ms = float(np.mean(prop_ms)) if prop_ms else float("nan")
    achieved = alg_bytes / (k_ms * 1e-3) / 1e9
    # which propagation kernel fire_simulate_batch picks by default (propagate.cu, fire_simulate_batch: geometry and family)
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    if S >= 2 * sms or L.W * L.H < 2048 * 2048:
        kname = "fire_propagate_kernel (two-phase, one CTA per simulation)"
    elif 2 * S <= sms:
        kname = f"fire_propagate_async_kernel (clusters of {4 if 4 * S <= sms else 2} CTAs per simulation)"
    else:
        kname = "fire_propagate_async_kernel (one CTA per simulation)"
    roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get(cfg) if world == 1 else None,
                "traffic_source": NCU_TRAFFIC_SOURCE.get(cfg) if world == 1 else None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": k_ms, "launches_timed": len(prop_ms),
                "share_of_step": k_ms / ms_per_step,
                "philox_calls_per_s": trials_rank / (k_ms * 1e-3)}
    # second ceiling: the arithmetic the method cannot avoid is one Philox4x32-10 call per trial = 18 wide
    # multiplies (IMAD.WIDE.U32; rounds 0 and 1 share their products over a step) + 18 three-input xors.  The wide multiplies run
    # on the FMA-heavy pipe only, one warp instruction per 4 cycles per SM sub-partition (measured: sm__pipe_fmaheavy_cycles_active
    # against the executed IMAD mix, profiles/r2_propagate_ncu.md), so peak = SMs x 4 sub-partitions x clock x 32 lanes / (18 x 4).
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    sm_clock_hz = 1e6 * float((clocks or {}).get("sm_max_mhz") or 1965.0)
    alu_peak = sm_count * 4 * sm_clock_hz * 32 / (18 * 4)
    alu_ach = trials_rank / (k_ms * 1e-3)
    roofline["alu"] = {"bound": "alu", "achieved": alu_ach / 1e9, "peak": alu_peak / 1e9, "unit": "G Philox calls/s",
                       "frac": alu_ach / alu_peak,
                       "note": "18 IMAD.WIDE per Philox4x32-10 call on the FMA-heavy pipe at 1 per 4 cycles per SM sub-partition"}

    # ---- CPU baseline: the oracle as it stands on a bounded sample of the same workload
    cpu = None
    if world == 1 and not args.no_cpu:
        wq, idx = oracle_sample(cfg, sample_budget(cfg))
        tr, dt, threads = time_oracle(wq, idx)
        idx1 = idx[:: max(1, threads)]                    # the single-thread figure on a 1/threads sub-sample: the same wall time
        tr1, dt1, _ = time_oracle(wq, idx1, nthreads=1)
        cpu = {"value": tr / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": sample_text(wq, idx) + f", {dt:.1f} s", "sims_per_s": len(idx) / dt,
               "single_thread": {"value": tr1 / dt1, "unit": UNIT, "cores": 1, "sims": int(len(idx1)), "seconds": dt1}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None,
        "dtype": "u32", "data": "synthetic",
        "config": {"workload": w.name, "lattice": f"{L.W}x{L.H}", "param_vectors": P, "sims_per_gpu": S,
                   "param_vectors_per_gpu": int(l_betas.shape[0]), "comm_nranks": world,
                   "step": "params_upload + simulate_batch + fitness (one GA generation)",
                   "l2": "inputs larger than L2: the threshold table is "
                         f"{P * L.W * L.H * 32 / 2**30:.2f} GiB and is rewritten every step",
                   "parallelism": (f"one generation partitioned by parameter vector over {world} GPU(s): each builds P/N of the table"
                                   if strong else f"one generation of S sims per GPU on {world} GPU(s) (replicates r*S..), no data-path collective")
                                  + ", landscape replicated, one all-gather of the scores per step"},
        "sims_per_s": sims_per_s, "trials_per_step": trials_all, "phases_ms": phases,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / args.steps},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    L.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one generation of S sims per GPU (default); strong = ONE generation partitioned by parameter vector")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="torch.distributed backend; gloo only to dry-run the N > 1 logic with ranks sharing a GPU (timings then mean nothing)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        world = int(os.environ.get("WORLD_SIZE", "1"))
        if world != args.gpus:
            log(f"note: --gpus {args.gpus} but WORLD_SIZE={world}; launch with torch.distributed.run for N > 1")
        run_ours(args)


if __name__ == "__main__":
    main()
