#!/usr/bin/env python
"""bench.py -- photon packages/s and shell-crossings/s of the DIES hot path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config2] [--packages P]

A "step" is one pass of the whole hot path over one batch of synthetic input: dies_run on config 2 (externally
heated sphere, 100 shells, 200 frequencies, 1e7 packages, full IRE).  `value` is timed with CUDA events around
dies_run with the model resident in HBM; `e2e` times create_model + set_sources + run + get_temperature +
get_escape_spectrum through the C ABI with host buffers.  Full IRE on one model does not shard (DESIGN.md,
"Multi-GPU": replicas only): with --gpus N every rank runs an independent replica (its own seed).  `--gpus N` with
N > 1 outside torchrun starts the N ranks itself (torch.distributed.run on 127.0.0.1); under torchrun it is one rank.
--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload.
"""
from __future__ import annotations

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

from paper_2408_13807_b200 import sharding, synth  # noqa: E402

# Algorithmic thread-instructions per unit of work in the shipped tracker dies_fly (profiles/r2_ncu_full.md,
# profiles/r2_cross_step.sass): crossing = SASS instructions of one crossing step on a live lane; scattering /
# absorption / package = predicated-on thread-instructions of the unit's own code (+ its share of the code the two event
# types have in common) per unit, from the ncu source page of this workload through
# `python profile_parts.py`.  Stack handling, batch composition, slot load / store, block ends and
# idle lanes are NOT work.  The constants belong to ONE version of the kernel sources: KERNEL_SHA256 is the hash they were
# derived at, and a roofline is only printed while the sources still have it.
INSTR = dict(crossing=8, scattering=174, absorption=345, package=260)
# The same constants frozen at their round-2 values: `roofline.frac_frozen_r2` counts work with these whatever the
# kernel has become, so that a leaner event routine shows as a gain and not as less counted work (INSTR itself is
# re-derived after every kernel change and would shrink with the code).  Derived on config 2; applied to every workload.
INSTR_FROZEN_R2 = dict(crossing=8, scattering=174, absorption=345, package=260)
KERNEL_SHA256 = "a84e3db16bb33b0ed5791fb51d0a618d4104bd72c7814918120e8f7f5da46b41"
# The second workload, dies_tmc (python bench.py --mode tmc): predicated-on thread-instructions of the unit's own code per
# unit, from profiles/r3_tmc_ncu_full.md (`python profile_parts.py source.csv --kernel tmc`); crossing = step +
# continuous absorption (L37) + weight guard.  They belong to the csrc/dies_tmc.cuh that hashes to TMC_SHA256.
INSTR_TMC = dict(crossing=102, scattering=154, package=537)
TMC_SHA256 = "0e8fa2c536f7b5514b0e3a29466b046f67b3ef332e364f808a2d51c4c8e9ac2b"
TMC_TRAFFIC_BYTES_PER_LAUNCH = 264192
TMC_NCU_PIPE_BUSY = dict(issue=0.904, smem_data=0.281)
# frozen at their first derivation (the kernel with the scattering inside the step loop, 8.15 ms per iteration): the
# fraction under these does not shrink when the code gets leaner
INSTR_TMC_FROZEN = dict(crossing=115, scattering=380, package=575)
# of the same ncu --set full capture (one dies_fly launch of config 2, 1e7 packages):
# dram__bytes_read.sum + dram__bytes_write.sum; busy fractions of the XU pipe (MUFU.SQRT of the crossings, 8 cycles per
# warp instruction) and of the shared-memory data pipe (l1tex__data_pipe_lsu_wavefronts, 1 wavefront per cycle and SM)
TRAFFIC_BYTES_PER_LAUNCH = 731904
NCU_PIPE_BUSY = dict(issue=0.795, xu=0.305, smem_data=0.810)
XU_CYCLES_PER_WARP_INSTR = 8
SM_COUNT, SCHEDULERS, LANES = 148, 4, 32


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d.get("sm_max_mhz", 1965.0)), "measured sm_max_mhz of MEASURED_PEAKS.json"
    return 1965.0, "fallback clocks.max.sm of B200_PROFILING.md"


def make_problem(workload, packages):
    if workload == "config1":
        p = synth.config1()
    elif workload == "config2":
        p = synth.config2()
    elif workload == "config2_kbg":
        p = synth.config2(k_bg=0.2)
    elif workload == "config3":
        p = synth.config3()
    elif workload == "config3_thick":
        p = synth.config3(tau_V=1000.0)
    elif workload == "config4":
        p = synth.config4()
    elif workload == "config4_noffi":
        p = synth.config4(ffi=0)
    elif workload == "config5":
        p = synth.config5()
    else:
        raise SystemExit(f"unknown workload {workload}")
    if packages:
        p.n_packages = int(packages)
    return p


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "10"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0=None, t1=None):
        """Summary of the samples taken in [t0, t1] (perf_counter times; all samples if none fall inside)."""
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        rows = [r for t, r in self.rows if t0 is None or t0 <= t <= t1 + 0.02]
        if not rows:
            rows = [r for _, r in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def oracle_rate(p, n_sample, seed=1):
    """The oracle as it stands on one host core: packages/s and crossings/s on a bounded sample."""
    from oracle import dies_oracle as orc
    if isinstance(p, synth.BatchProblem):
        # a batch is sampled model by model (8 models, n_sample / 8 packages each)
        tot_n, tot_c, tot_t = 0, {}, 0.0
        for mi in range(min(8, p.n_models)):
            r, cr, dt, c = oracle_rate(p.model(mi), max(1, n_sample // 8), seed)
            tot_n += max(1, n_sample // 8); tot_t += dt
            for k, v in c.items():
                tot_c[k] = tot_c.get(k, 0) + v
        return tot_n / tot_t, tot_c["crossings"] / tot_t, tot_t, tot_c
    o = orc.Oracle(p)
    t0 = time.perf_counter()
    o.run(n_sample, seed=seed, k_bg=getattr(p, "k_bg", 0.5), ffi=getattr(p, "ffi", 0))
    dt = time.perf_counter() - t0
    c = o.counters
    return n_sample / dt, c["crossings"] / dt, dt, c


def _oracle_worker(a):
    workload, packages, n_sample, seed = a
    p = make_problem(workload, packages)
    r, cr, dt, c = oracle_rate(p, n_sample, seed=seed)
    return n_sample, c["crossings"], dt


def oracle_rate_all_cores(workload, packages, n_sample, procs):
    """Independent seeds of the serial oracle, one process per core: aggregate packages/s and crossings/s."""
    import multiprocessing as mp
    t0 = time.perf_counter()
    with mp.get_context("spawn").Pool(procs) as pool:
        res = pool.map(_oracle_worker, [(workload, packages, n_sample, 100 + i) for i in range(procs)])
    wall = time.perf_counter() - t0
    slowest = max(r[2] for r in res)
    return sum(r[0] for r in res) / slowest, sum(r[1] for r in res) / slowest, slowest, wall


def run_reference(args, rank, world):
    if rank != 0:
        return
    p = make_problem(args.workload, args.packages)
    # bounded sample per step: the whole --steps K run follows about --ref-total packages (tens of seconds of CPU)
    n_sample = min(p.n_packages, args.ref_sample, max(2000, args.ref_total // max(args.steps, 1)))
    for _ in range(args.warmup):
        oracle_rate(p, max(1, n_sample // 10))
    times, cross = [], 0
    for s in range(args.steps):
        r, cr, dt, c = oracle_rate(p, n_sample, seed=1 + s)
        times.append(dt); cross += c["crossings"]
    tot = float(np.sum(times))
    value = n_sample * args.steps / tot
    line = dict(impl="reference", metric="packages_per_s", value=value, unit="packages/s", n_gpus=args.gpus,
                steps=args.steps, warmup=args.warmup, ms_per_step=1e3 * tot / args.steps, higher_is_better=True,
                scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                crossings_per_s=cross / tot,
                config=dict(workload=args.workload, n_shells=int(p.rho.shape[-1]), n_freq=int(p.freq.size),
                            n_T=int(p.T_grid.size), packages_per_step=n_sample, mode="full IRE", note="serial CPU oracle on a bounded sample"),
                cpu_baseline=dict(value=value, unit="packages/s", cores=1, kind="oracle",
                                  sample=f"{n_sample} packages of {args.workload} per step, {args.steps} steps"),
                e2e=dict(value=value, unit="packages/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line))


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2408_13807_b200 import binding as dies

    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if args.tune:
        dies.dies_set_tuning(**{k: int(v) for k, v in (kv.split("=") for kv in args.tune.split(","))})
    p = make_problem(args.workload, args.packages)
    batch = isinstance(p, synth.BatchProblem)
    model0 = 0
    if batch and world > 1:
        # config 5 shards: the spheres are dealt to the ranks, no exchange
        p, model0 = sharding.batch_shard(p, rank, world)
    n_models = p.n_models if batch else 1
    n_per_model = p.n_packages
    n = n_per_model * n_models                              # packages per step on this rank
    k_bg, ffi = getattr(p, "k_bg", 0.5), getattr(p, "ffi", 0)
    n_shells, n_freq, n_T = int(p.rho.shape[-1]), int(p.freq.size), int(p.T_grid.size)
    opts = dict(k_bg=k_bg, ffi=ffi)
    weighted = {}
    if args.run_opts:
        # weighting of Table 1 for the timing table of BASELINE.md, e.g. k_A=3,k_S=2 or g_E=0.5,g_S=0.2 (dies_run_opts)
        weighted = {k: float(v) for k, v in (kv.split("=") for kv in args.run_opts.split(","))}
        if "reemit_cell" in weighted:
            weighted["reemit_cell"] = int(weighted["reemit_cell"])
        opts.update(weighted)
        if any(k in weighted for k in ("k_A", "k_A_dilute", "k_S", "g_E", "g_S", "reemit_cell")):
            opts["ffi"] = ffi = 0                           # weighting and forced first interaction are alternatives
    tmc = args.mode == "tmc"
    if tmc:
        # the second workload (R22): a step is one iteration of the traditional Monte Carlo with continuous
        # absorption in its steady state (sources + as many dust packages); plain runs only
        opts = dict(mode=dies.DIES_MODE_TMC)
    def make():
        if not batch:
            return dies.Model(p, device=str(dev))
        mm = dies.Model(batch=p, device=str(dev))
        mm.dies_set_model_offset(model0)
        return mm
    m = make()
    info = dies.dies_device_info()
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    sampler = ClockSampler(local_rank)                      # (started before the warm-up: nvidia-smi takes a while to report)
    sampler.start()
    for w in range(args.warmup):
        m.dies_run(n_per_model, seed=sharding.replica_seed(1000, w, 0 if batch else rank), **opts)
    torch.cuda.synchronize(dev)
    c0 = m.dies_get_counters()

    # ---- device-timed steps: CUDA events on the launching stream, L2 flushed between steps
    barrier()
    t_wall = time.perf_counter()
    t_begin = t_wall
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    tot_counts = dict(crossings=0, scatterings=0, absorptions=0, packages=0)
    for s in range(args.steps):
        flush.fill_(s & 0xFF)
        ev[s][0].record(stream)
        m.dies_run(n_per_model, seed=sharding.replica_seed(1, s, 0 if batch else rank), **opts)
        ev[s][1].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop(t_begin, t_begin + t_wall)
    ms = [a.elapsed_time(b) for a, b in ev]
    c1 = m.dies_get_counters()
    # counters are zeroed by every non-accumulating run: c1 holds the last step; steps are statistically identical
    for k in tot_counts:
        tot_counts[k] = c1[k]
    step_ms = float(np.sum(ms)) / args.steps
    total_ms = sharding.max_over_ranks(float(np.sum(ms)), dev)
    if tmc:
        n = int(c1["packages"])                             # sources + dust packages of an iteration
    n_all = sharding.sum_over_ranks(n, dev)                # packages per step of the whole job
    value = n_all * args.steps / (total_ms * 1e-3)
    crossings_per_s = sharding.sum_over_ranks(c1["crossings"], dev) * args.steps / (total_ms * 1e-3)

    # ---- end to end through the C ABI with host buffers: create + sources + run + both getters.  The inputs sit in
    #      pinned host memory (the binding passes their addresses through: numpy views of pinned torch tensors)
    import dataclasses
    pin = {f.name: torch.from_numpy(np.ascontiguousarray(getattr(p, f.name), dtype=np.float64)).pin_memory().numpy()
           for f in dataclasses.fields(p) if isinstance(getattr(p, f.name), np.ndarray)}
    p_pinned = dataclasses.replace(p, **pin)

    def make_e2e():
        if not batch:
            return dies.Model(p_pinned, device=str(dev))
        mm = dies.Model(batch=p_pinned, device=str(dev))
        mm.dies_set_model_offset(model0)
        return mm

    e2e_t = []
    for s in range(max(1, min(args.steps, 5))):
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        m2 = make_e2e()
        m2.dies_run(n_per_model, seed=1 + s, **opts)
        T = m2.dies_get_temperature()
        Lesc = m2.dies_get_escape_spectrum()
        e2e_t.append(time.perf_counter() - t0)
        m2.close()
    # (a fresh handle's first TMC iteration has no dust packages yet: its end-to-end figure counts the source packages)
    e2e_n = sharding.sum_over_ranks(n_per_model * n_models, dev) if tmc else n_all
    e2e_val = e2e_n / sharding.max_over_ranks(float(np.median(e2e_t)), dev)
    h2d = 8 * (p.emis.size + p.T_grid.size + 3 * n_freq + p.r_bounds.size + p.rho.size + 2 * n_freq * n_models)
    d2h = 8 * n_models * (n_shells + n_freq) + 64

    if rank != 0:
        return
    # the atomic side of the roofline: the absorption step's returning 64-bit atomicAdd pattern alone on n_shells
    # tallies (merged per warp when all quanta are equal, as in this run), measured on this GPU outside the timed region
    uniform_q = (k_bg == 0.5 and not ffi and not (p.ext_bin_intensity is not None and getattr(p, "L_point", 0.0) > 0))
    raw_abs, _, _ = m.dies_get_absorbed()                     # per-shell absorption histogram of the last step
    hist = np.asarray(raw_abs, dtype=np.float64).reshape(n_models, n_shells).sum(0)
    atom = dies.dies_bench_atomics(n_shells * min(n_models, 64), weights=np.tile(hist, min(n_models, 64)),
                                   aggregate=1 if uniform_q else 0)
    sm_max, peak_src = load_peaks()
    peak = SM_COUNT * SCHEDULERS * LANES * sm_max * 1e6 / 1e12          # thread-instructions/s, 1e12
    def work_of(instr):
        # (the crossings of the forced-first-interaction chord walk are crossings too: PAPER.md L132-149)
        return ((c1["crossings"] + c1["ffi_crossings"]) * instr["crossing"] + c1["scatterings"] * instr["scattering"] +
                c1["absorptions"] * instr["absorption"] + c1["packages"] * instr["package"])
    achieved = work_of(INSTR) / (step_ms * 1e-3) / 1e12
    achieved_frozen = work_of(INSTR_FROZEN_R2) / (step_ms * 1e-3) / 1e12
    held = clocks.get("sm_mhz") or sm_max
    from paper_2408_13807_b200 import build as dies_build
    stale = dies_build.kernel_hash() != KERNEL_SHA256
    # the XU pipe executes the one square root of every crossing: 8 cycles per warp instruction and scheduler
    xu_peak = SM_COUNT * SCHEDULERS * LANES * sm_max * 1e6 / XU_CYCLES_PER_WARP_INSTR
    line = dict(metric="packages_per_s", value=value, unit="packages/s", n_gpus=world, steps=args.steps,
                warmup=args.warmup, ms_per_step=total_ms / args.steps, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f32", data="synthetic",
                crossings_per_s=crossings_per_s,
                config=dict(workload=args.workload, n_models=n_models, n_shells=n_shells, n_freq=n_freq, n_T=n_T,
                            packages_per_step=int(n_all), mode="full IRE", k_bg=k_bg, ffi=ffi,
                            parallelism=("model shards, no collective" if batch else "replicas only") if world > 1 else "1 GPU", l2="flushed between steps (256 MiB fill)",
                            per_package=dict(crossings=c1["crossings"] / n, scatterings=c1["scatterings"] / n,
                                             absorptions=c1["absorptions"] / n),
                            grid=dict(**info)),
                clocks=clocks,
                e2e=dict(value=e2e_val, unit="packages/s", h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                         ms_per_step=1e3 * float(np.median(e2e_t)), host_buffers="pinned inputs, pageable outputs"),
                gpu_launches=int(2 * args.steps),
                roofline=dict(bound="alu", achieved=achieved, peak=peak, unit="Tinstr/s", frac=achieved / peak,
                              frac_at_held_clock=achieved / (peak * held / sm_max),
                              frac_frozen_r2=achieved_frozen / peak, instr_per_unit_frozen_r2=INSTR_FROZEN_R2,
                              traffic=TRAFFIC_BYTES_PER_LAUNCH,
                              atomic=dict(absorptions_per_s=c1["absorptions"] / (step_ms * 1e-3),
                                          peak_absorptions_per_s=atom["lane_ops_per_s"],
                                          peak_atomic_instr_per_s=atom["atomics_per_s"],
                                          frac=c1["absorptions"] / (step_ms * 1e-3) / atom["lane_ops_per_s"],
                                          peak_source=f"dies_bench_atomics({n_shells * min(n_models, 64)} tallies, the run's shell histogram, warp-merged={int(uniform_q)}) on this GPU"),
                              xu=dict(crossings_per_s=c1["crossings"] / (step_ms * 1e-3), peak_sqrt_per_s=xu_peak,
                                      frac=c1["crossings"] / (step_ms * 1e-3) / xu_peak,
                                      note="one MUFU.SQRT per crossing; the XU pipe takes 8 cycles per warp instruction"),
                              ncu_pipe_busy=NCU_PIPE_BUSY,
                              peak_source=f"148 SMs x 4 schedulers x 32 lanes x {sm_max:.0f} MHz ({peak_src})",
                              instr_per_unit=INSTR, kernel="dies_fly<0,false,4>", kernel_ms=step_ms),
                wall_s=t_wall)
    if tmc:
        line["config"]["mode"] = "TMC iteration (continuous absorption), steady state"
        import hashlib
        tmc_src = os.path.join(ROOT, "paper_2408_13807_b200", "csrc", "dies_tmc.cuh")
        tmc_stale = hashlib.sha256(open(tmc_src, "rb").read()).hexdigest() != TMC_SHA256
        def tmc_work(instr):
            return (c1["crossings"] * instr["crossing"] + c1["scatterings"] * instr["scattering"] +
                    c1["packages"] * instr["package"]) / (step_ms * 1e-3) / 1e12
        w_tmc = tmc_work(INSTR_TMC)
        line["roofline"] = dict(bound="alu", achieved=None if tmc_stale else w_tmc, peak=peak, unit="Tinstr/s",
                                frac=None if tmc_stale else w_tmc / peak,
                                traffic=None if tmc_stale else TMC_TRAFFIC_BYTES_PER_LAUNCH,
                                frac_frozen=tmc_work(INSTR_TMC_FROZEN) / peak, instr_per_unit_frozen=INSTR_TMC_FROZEN,
                                ncu_pipe_busy=TMC_NCU_PIPE_BUSY, instr_per_unit=INSTR_TMC,
                                peak_source=f"148 SMs x 4 schedulers x 32 lanes x {sm_max:.0f} MHz ({peak_src})",
                                kernel="dies_tmc", kernel_ms=step_ms,
                                note="second workload (DESIGN.md R22); constants from profiles/r3_tmc_ncu_full.md"
                                     + ("; csrc/dies_tmc.cuh changed since: no fraction claimed" if tmc_stale else ""))
    elif weighted:
        line["config"]["run_opts"] = weighted
        line["roofline"] = dict(bound="alu", achieved=None, peak=peak, unit="Tinstr/s", frac=None, traffic=None,
                                frac_frozen_r2=achieved_frozen / peak, instr_per_unit_frozen_r2=INSTR_FROZEN_R2,
                                kernel="dies_track<0,false,true>", kernel_ms=step_ms,
                                note="weighted run: dies_track, for which no work-per-unit constants were derived; the "
                                     "frozen dies_fly constants count the same physical units")
    elif stale:
        # the work-per-unit constants were derived from other kernel sources: no fraction is claimed
        line["roofline"] = dict(bound="alu", achieved=None, peak=peak, unit="Tinstr/s", frac=None, traffic=None,
                                frac_frozen_r2=achieved_frozen / peak, instr_per_unit_frozen_r2=INSTR_FROZEN_R2,
                                stale="kernel sources changed since INSTR was derived: run an ncu source page through "
                                      "profile_parts.py and update INSTR and KERNEL_SHA256",
                                kernel_ms=step_ms)
    # ---- the oracle timed beside it on this box's host cores (rank 0, N = 1 only)
    if world == 1 and not args.no_cpu_baseline:
        # bounded sample: a pilot of 4000 packages sizes the sample to about --cpu-seconds of CPU work
        r0, _, _, _ = oracle_rate(p, 4000)
        n_cpu = int(min(n, args.cpu_sample, max(4000, r0 * args.cpu_seconds)))
        r, cr, dt, c = oracle_rate(p, n_cpu)
        line["cpu_baseline"] = dict(value=r, unit="packages/s", cores=1, kind="oracle", crossings_per_s=cr,
                                    sample=f"{n_cpu} packages of {args.workload} ({dt:.1f} s), serial fp64 oracle",
                                    host_cores=os.cpu_count())
        if args.cpu_all_cores:
            procs = os.cpu_count() or 1
            ra, ca, slow, wall = oracle_rate_all_cores(args.workload, args.packages, max(4000, n_cpu // 2), procs)
            line["cpu_baseline"]["all_cores"] = dict(value=ra, unit="packages/s", crossings_per_s=ca, processes=procs,
                                                     sample=f"{max(4000, n_cpu // 2)} packages per process, independent seeds "
                                                            f"(slowest {slow:.1f} s)")
    print(json.dumps(line))
    m.close()


def run_noise_study(args):
    """Accuracy against the number of packages (section 3.1, Fig. 2-3; section 3.2; BASELINE.json
    configs[3] "noise per shell vs packages reported"): for configs 2 (k_bg = 0.5 and 0.2), 3 and 4 (FFI on / off) the shell
    temperatures of 8 seeds at N = 1e5 ... 1e8 packages against a reference run with 1e9 packages.  Per radius decile:
    the statistical error (standard deviation over the seeds / mean) and the systematic error (mean over the seeds
    against the reference).  One JSON line; every run goes through the C ABI (dies_run + dies_get_temperature),
    nothing is timed here."""
    import torch
    from paper_2408_13807_b200 import binding as dies
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    seeds = list(range(1, 9))
    cases = [("config2", synth.config2(), {}), ("config2_kbg0.2", synth.config2(k_bg=0.2), dict(k_bg=0.2)),
             ("config3", synth.config3(), {}), ("config4_ffi", synth.config4(ffi=1), dict(ffi=1)),
             ("config4_noffi", synth.config4(ffi=0), {})]
    rows = []
    for name, p, kw in cases:
        m = dies.Model(p, device=str(dev))
        m.dies_run(10**9, seed=1001, **kw)
        Tref = m.dies_get_temperature()
        edges = np.linspace(0, p.n_shells, 11).astype(int)
        for n in (10**5, 10**6, 10**7, 10**8):
            T = []
            for sd in seeds:
                m.dies_run(n, seed=sd, **kw)
                T.append(m.dies_get_temperature())
            T = np.array(T)
            ok = T.min(0) > p.T_grid[0] * 1.001                   # shells every seed reached
            rel = np.where(ok, T.std(0, ddof=1) / T.mean(0), np.nan)
            sys_ = np.where(ok, T.mean(0) / Tref - 1.0, np.nan)
            dec = lambda v: [None if not np.any(np.isfinite(v[a:b])) else float(np.nanmean(v[a:b]))
                             for a, b in zip(edges[:-1], edges[1:])]
            rows.append(dict(case=name, packages=n, shells_reached=int(ok.sum()),
                             rel_sigma_T_mean=float(np.nanmean(rel)), rel_sigma_T_max=float(np.nanmax(rel)),
                             rel_sigma_T_deciles=dec(rel), sys_error_deciles=dec(sys_),
                             abs_sys_error_mean=float(np.nanmean(np.abs(sys_))), T_mean_K=float(T.mean())))
        m.close()
    print(json.dumps(dict(study="noise and systematic error per radius decile vs packages", seeds=len(seeds),
                          reference_packages=10**9, data="synthetic", rows=rows)))


def spawn_command(n_gpus, argv):
    """The launch line of N ranks on this node (the one the driver uses for N > 1), on a free local port."""
    import socket

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--packages", type=float, default=0)
    ap.add_argument("--cpu-sample", type=int, default=20_000_000)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--ref-sample", type=int, default=1_000_000)
    ap.add_argument("--ref-total", type=int, default=20_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", default="ire", choices=["ire", "tmc"], help="full IRE (the headline) or one TMC iteration per step")
    ap.add_argument("--run-opts", default="", help="dies_run options of a weighted run, e.g. k_A=3,k_S=2 (include/dies.h: dies_run_opts)")
    ap.add_argument("--tune", default="", help="launch tuning for dies_set_tuning, e.g. visit=2,slots_uniform=5 (include/dies.h: dies_tuning)")
    ap.add_argument("--cpu-all-cores", action="store_true", help="also time the oracle on all host cores (one process each)")
    ap.add_argument("--noise-study", action="store_true", help="configs 2, 3, 4: sigma_T and systematic error per radius decile over 8 seeds vs packages")
    args = ap.parse_args(argv)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours" and not args.noise_study:
        # `python bench.py --gpus N` by itself: start the N ranks (one process per GPU) and let rank 0 print the line
        sys.exit(subprocess.call(spawn_command(args.gpus, sys.argv[1:] if argv is None else list(argv))))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.noise_study:
        if rank == 0:
            run_noise_study(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        if args.warmup < 3:
            args.warmup = 3
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
