#!/usr/bin/env python
"""bench.py -- super-droplet-steps/s of the full particle step (sort + cond x10 + coal + adve/sedi +
compaction) on the 3D prescribed-flow configuration of BASELINE.json (configs[3]: 128x128x64 cells,
64 SD/cell, 67M SDs, fp64), one process per GPU.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 3d|2d|sweep]

Prints ONE JSON line (rank 0).  `--impl reference` times the oracle (a deliberately plain CPU program)
on a bounded sample of the same workload.  See DESIGN.md "Measurement" for every definition used here.
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

METRIC = "super-droplet-steps/s (sort+coal+cond+sedi)"
UNIT = "SD-steps/s"

# Algorithmic work per unit:
#  - whole step, fp64, 3D: 350 B of HBM traffic per SD-step;
#  - condensation kernel: fp64 operations per growth-rate evaluation and per SD-substep set-up, counted
#    from the formulae (an FMA counts 2; a division, sqrt, rsqrt, exp, cbrt count as the length of their
#    fp64 instruction sequences).
BYTES_PER_SD_STEP = {(3, 8): 350.0, (2, 8): 350.0 - 16.0 - 8.0,      # fp64 state: SURVEY.md 8d
                     (3, 4): 232.0, (2, 4): 232.0 - 8.0 - 4.0}       # fp32 state: the six reals at 4 bytes


def stage_bytes(ndim, rb):
    """Algorithmic HBM bytes per SD of each timed stage (one pass over the attributes a stage must touch;
    fp64 3D: 32 + 20 + 124 + 40 + 132 = 348).  rb = bytes of a real attribute, ndim = stored coordinates."""
    state = 8 + (3 + ndim) * rb + 4                      # n, rw2, rd3, kappa, coordinates, id
    return {"hist": ndim * rb + 8,                       # a1: read the position, write cell + key
            "rank": 20.0,                                # a2: sort within the cell (SURVEY's figure)
            "scatter": 2 * state + 4,                    # a3: read state + permutation, write state
            "cond": 8 + 3 * rb + rb,                     # a4: read n, rw2, rd3, kappa, write rw2
            "coal_move": 2 * (8 + 3 * rb) + (ndim * rb + rb + 4) + (ndim * rb + 8)}   # a5 + a6


# k_cond4, fp64 thread-instructions executed per unit of work, fitted to ncu's per-launch counters of 38 launches of this
# build (profiles/r2_k_cond4_ncu_full.md: smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum and
# smsp__inst_executed_pipe_fp64.sum against the SD-substeps and evaluations sdm_stats reports for the same launches).
# "first" = everything an SD-substep costs with ONE growth-rate evaluation: ventilation set-up, eq. 18-19, the certificate of
# R-roots, f and f', the Newton step, N d(r^3), its share of the cells' thermodynamics; "more" = every further evaluation with
# its third-order corrected Newton step; "other" = the remaining lane slots of fp64-pipe warp instructions (DSETP, conversions,
# lanes that are predicated off).  flops: DFMA = 2, DMUL = DADD = 1.
FP64_INSTR = {"first": {"dfma": 48.9, "dmul": 61.0, "dadd": 21.5, "other": 52.6},
              "more": {"dfma": 40.2, "dmul": 55.2, "dadd": 16.5, "other": 27.0}}
FP64_INSTR_SOURCE = "profiles/r2_k_cond4_ncu_full.md"
FP64_LANES_PER_SM = 64        # fp64 FMA lanes per SM per clock on sm_100 (B200_PROFILING.md; sdm_measure_fp64_peak confirms)
# --cond-arith 4 (k_cond4f): fp32 operations of one evaluation with derivative and curvature bound (62 instructions, 20 of
# them FMA, 4 MUFU) and of the per-SD-substep set-up, first step and N d(r^3) (45 instructions, 15 FMA); DESIGN.md section 7
FLOP_PER_EVAL_F32 = 86.0
FLOP_PER_SETUP_F32 = 60.0
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12  # SMs x fp32 FMA lanes x 2 x max SM clock = 74.4
# dram__bytes_read.sum + dram__bytes_write.sum of one launch on the default workload, from the ncu capture named beside it
NCU_COND_DRAM_BYTES = (2.314134e9 + 0.552060e9, "profiles/r2_k_cond4_ncu_full.md")
NCU_COND32_DRAM_BYTES = (1.509464e9 + 0.313273e9, "profiles/r1_k_cond4f_ncu_full.md")


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="3d", choices=["3d", "2d", "sweep"])
    ap.add_argument("--sd-per-cell", type=int, default=0)
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the horizontal grid (debugging only; reported in config)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fp32-mode", action="store_true", help="skip the extra fp32-mode measurement of the default run")
    ap.add_argument("--group", type=int, default=0)
    ap.add_argument("--cond-arith", type=int, default=8, choices=[8, 4], help="arithmetic of the condensation sweep; 4 = fp32 (needs --real-bytes 4)")
    ap.add_argument("--recycle", action="store_true", help="the paper's recycling of zero-multiplicity SDs (:641) instead of compaction only")
    ap.add_argument("--real-bytes", type=int, default=8, choices=[8, 4], help="storage type of the SD attributes (configs[4]: fp32 state)")
    ap.add_argument("--cond-adapt-tol", type=float, default=0.0, help="adaptive condensation substeps per cell (sdm_opts.cond_adapt_tol, DESIGN.md R-adapt); "
                    "0 = the fixed sstp_cond of the paper and of the headline")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"], help="N > 1: independent replicas (default), or one domain of "
                    "N x 128 columns decomposed into x-slabs, one per rank, SDs that cross a face exchanged every step (slab.py; weak scaling)")
    ap.add_argument("--step-stats", default="", help="profiling aid: write one JSON line per step of the device-timed context (warm-up steps "
                    "included) with the growth-rate evaluations and SD-substeps of that step's condensation launch (sdm_stats deltas); "
                    "synchronises after every step, so the run's timings are not bench values")
    ap.add_argument("--long-run", type=int, default=-1, help="after the timed region, continue the run to this many steps in all and report "
                    "ms/step, evaluations per SD-substep, slow-list fraction and the launch configuration per 100-step window "
                    "(default: 600 = the length of configs[3] for the default workload, 0 otherwise)")
    return ap.parse_args()


def workload_args(a):
    if a.workload == "3d":
        n = max(int(round(128 * a.scale)), 2)
        return dict(kind="3d", nx=n, ny=n, nz=64, sd=a.sd_per_cell or 64)
    if a.workload == "2d":
        return dict(kind="2d", nx=75, ny=0, nz=75, sd=a.sd_per_cell or 128)
    return dict(kind="sweep", nx=256, ny=0, nz=256, sd=a.sd_per_cell or 128)


def make_workload(wa, seed, device):
    from paper_1310_1905_b200 import workloads as W

    if wa["kind"] == "3d":
        return W.cfg4_3d(sd_per_cell=wa["sd"], nx=wa["nx"], ny=wa["ny"], nz=wa["nz"], seed=seed, device=device)
    if wa["kind"] == "2d":
        return W.cfg3_2d_drizzle(sd_per_cell=wa["sd"], seed=seed, device=device)
    return W.cfg5_sweep(wa["sd"], seed=seed, device=device)


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled during the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def oracle_rate(wa, steps, warmup, seed=42):
    """The oracle as it stands on the host cores, on a bounded sample of the workload: a block of full
    columns of the same recipe (same vertical profile, same SD/cell), OpenMP over cells."""
    import oracle
    from tests.util import make_oracle

    nx = 8 if wa["kind"] == "3d" else 16
    sub = dict(wa)
    sub.update(nx=nx, ny=(4 if wa["kind"] == "3d" else 0))
    if wa["kind"] != "3d":
        sub["nz"] = min(wa["nz"], 75)
    from paper_1310_1905_b200 import workloads as W

    if wa["kind"] == "3d":
        w = W.cfg4_3d(sd_per_cell=wa["sd"], nx=sub["nx"], ny=sub["ny"], nz=sub["nz"], seed=seed)
    elif wa["kind"] == "2d":
        w = W.cfg3_2d_drizzle(sd_per_cell=wa["sd"], nx=sub["nx"], nz=sub["nz"], seed=seed)
    else:
        w = W.kinematic(sub["nx"], 0, wa["nz"], 1500.0 / wa["nz"], wa["sd"], seed=seed)
    cores = oracle.lib().orc_max_threads()
    o = make_oracle(w, threads=cores)
    oo = oracle.make_opts(**w.opts)
    for _ in range(warmup):
        o.step(oo)
    n, t0 = 0, time.perf_counter()
    for _ in range(steps):
        n += o.n_live()
        o.step(oo)
    dt = time.perf_counter() - t0
    # the same sample on ONE thread (the serial oracle is the stated baseline, the OpenMP one the fair one)
    o.set_threads(1)
    n1, t1 = o.n_live(), time.perf_counter()
    o.step(oo)
    oracle_rate.one_thread = n1 / (time.perf_counter() - t1)
    desc = (f"{w.name}: {w.n_sd} SDs in {sub['nx']}x{max(sub['ny'], 1)}x{sub['nz']} full columns of the same recipe, "
            f"{steps} steps after {warmup} warm-up, OpenMP over cells")
    return n / dt, cores, desc, dt / steps * 1e3, w.n_sd


def run_reference(a, wa):
    """The oracle as it stands on the host cores, K steps after W warm-up steps, every step on a bounded sample of the
    workload (a block of full columns of the same recipe; the 67M-SD domain would take ~50 s per step on 16 cores)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    v, cores, desc, ms, n_sample = oracle_rate(wa, max(a.steps, 1), max(a.warmup, 0))
    cfg = config_of(wa)
    cfg["n_sd_per_gpu"] = n_sample
    cfg["sample"] = desc
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": a.gpus, "steps": max(a.steps, 1), "warmup": max(a.warmup, 0),
           "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": cfg, "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def config_of(wa):
    return {"workload": f"{wa['kind']} prescribed-flow {wa['nx']}x{max(wa['ny'], 1)}x{wa['nz']} cells, {wa['sd']} SD/cell, "
                        "bimodal lognormal aerosol (kappa=0.61), sort+cond(10 substeps)+coal+adve+sedi+compaction, dt=1 s, RH_max=1.05",
            "n_sd_per_gpu": wa["nx"] * max(wa["ny"], 1) * wa["nz"] * wa["sd"],
            "l2": "state (60 B/SD) far exceeds the 126 MB L2; no flush needed",
            "parallelism": "independent replicas (single-GPU path, no collective)"}


def make_particles(binding, torch, w, wa, a, rank=0):
    slab_mode = a.decomp == "slab"
    p = binding.Particles(max_sd=int(w.n_sd * (1.05 if slab_mode else 1.0)), sd_conc_mean=wa["sd"], real_bytes=a.real_bytes, open_x=slab_mode, **w.init)
    s = w.state
    if slab_mode:   # ids are unique over the whole domain: they key the Philox streams and travel with the SDs
        s = dict(s, id=(s["id"].to(torch.int64) + rank * w.n_sd).to(torch.int32))
    if a.real_bytes == 4:
        s = {k: (v if v is None or k in ("n", "id") else v.to(torch.float32)) for k, v in s.items()}
    cs = list(w.courants) + [None] * (3 - len(w.courants))
    p.init_from_arrays(w.rhod, s["n"], s["rw2"], s["rd3"], s["kappa"], s["x"], s["y"], s["z"], s["id"], courant_1=cs[0],
                       courant_2=cs[1], courant_3=cs[2])
    if a.group:
        p.set_group_size(a.group)
    if a.recycle:
        p.set_recycle(True)
    if a.cond_arith == 4:
        p.set_cond_arith(4)
    return p


def cond_fp64_work(evals, subs):
    """fp64 thread-instructions and flops (DFMA = 2, DMUL = DADD = 1) of k_cond4 for `subs` SD-substeps solved with `evals`
    growth-rate evaluations, from the per-unit counts of FP64_INSTR."""
    more = max(evals - subs, 0)
    instr = {k: subs * FP64_INSTR["first"][k] + more * FP64_INSTR["more"][k] for k in ("dfma", "dmul", "dadd", "other")}
    flops = 2.0 * instr["dfma"] + instr["dmul"] + instr["dadd"]
    return instr, flops


def main():
    a = parse()
    wa = workload_args(a)
    if a.impl == "reference":
        return run_reference(a, wa)

    import torch
    import torch.distributed as dist

    from paper_1310_1905_b200 import binding, replicas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = f"cuda:{local}"
    warm = max(a.warmup, 3)
    full3d = wa["kind"] == "3d" and a.scale == 1.0 and wa["sd"] == 64
    long_run = a.long_run if a.long_run >= 0 else (600 if full3d and world == 1 and not a.recycle and a.cond_adapt_tol == 0.0 and a.decomp == "replicas" else 0)

    w = make_workload(wa, seed=replicas.replica_seed(42, rank), device=dev)
    p = make_particles(binding, torch, w, wa, a, rank)
    p_host = make_particles(binding, torch, w, wa, a, rank)   # a second, identically initialised context for the end-to-end leg
    slab_widths = [wa["nx"] * 20.0] * world
    from paper_1310_1905_b200 import slab

    def hand_over(q):   # --decomp slab: SDs that crossed a face of this rank's slab go to the neighbour (nccl send/recv)
        if a.decomp == "slab":
            slab.exchange(q, slab_widths, 1 << 20, rank, world)
    n_sd0 = w.n_sd
    th, rv = w.th.clone(), w.rv.clone()
    th_h, rv_h = w.th.cpu().pin_memory(), w.rv.cpu().pin_memory()
    ndim = 3 if wa["ny"] > 0 else 2
    del w
    torch.cuda.empty_cache()
    po = binding.make_opts(adve=True, sedi=True, cond=True, coal=True, RH_max=1.05, sstp_cond=10, sstp_coal=1, cond_adapt_tol=a.cond_adapt_tol)
    fp64_peak_tflops, fp64_lanes = binding.measure_fp64_peak()   # measured on this device, before the timed region

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    step_log = open(a.step_stats, "w") if a.step_stats and rank == 0 else None
    prev = [p.stats()] if step_log else None

    def log_step():
        if step_log:
            cur = p.stats()
            step_log.write(json.dumps({"step": cur["step"], "evals": cur["newton_iters"] - prev[0]["newton_iters"],
                                       "sd_substeps": cur["sd_substeps"] - prev[0]["sd_substeps"],
                                       "slow": cur["cond_slow"] - prev[0]["cond_slow"]}) + "\n")
            step_log.flush()
            prev[0] = cur

    for _ in range(warm):
        p.step_sync(po, th, rv)
        p.step_async(po)
        hand_over(p)
        log_step()
    # ---- device-resident timing ------------------------------------------------------------------
    p.set_timing(True)
    p.stage_times(reset=True)
    st0 = p.stats()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sd_steps = 0
    ev0.record()
    for _ in range(a.steps):
        p.step_sync(po, th, rv)
        sd_steps += p.n_sd()      # live SDs of this step (host-known after the sort, no extra sync)
        p.step_async(po)
        hand_over(p)
        log_step()
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    st1 = p.stats()
    stages = p.stage_times(reset=True)
    p.set_timing(False)
    ms_max, sd_total = replicas.job_totals(ms, sd_steps, device=dev)   # slowest rank's device time, all ranks' SD-steps
    value = sd_total / (ms_max * 1e-3)

    # ---- end to end: the SAME steps (the second context, same initial state, same warm-up) with the Eulerian fields in
    # pinned host memory, copied in and out inside every timed step through sdm_step_host ------------------------------
    for _ in range(warm):
        p_host.step_host(po, th_h, rv_h)
        hand_over(p_host)
    barrier()
    e_sd, t0 = 0, time.perf_counter()
    for _ in range(a.steps):
        e_sd += p_host.n_sd()
        p_host.step_host(po, th_h, rv_h)
        hand_over(p_host)
    torch.cuda.synchronize()
    e_dt = time.perf_counter() - t0
    e_s, e_tot = replicas.job_totals(e_dt, e_sd, device=dev)
    ncell = th.numel()
    e2e = {"value": e_tot / e_s, "unit": UNIT, "h2d_bytes_per_step": 2 * ncell * 8,
           "d2h_bytes_per_step": 2 * ncell * 8 + 8, "api": "sdm_step_host (th, rv in pinned host memory)",
           "window": f"steps {warm + 1}..{warm + a.steps} after the initial condition, the same as the device-timed region"}
    del p_host
    torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- the rest of the run (configs[3]: 600 steps): the cloud forms, drops grow, rain starts -----------------------
    long = None
    if long_run > warm + a.steps:
        long = {"total_steps": long_run, "windows": []}
        done = warm + a.steps
        t_all, n_all = 0.0, 0
        while done < long_run:
            k = min(100 - done % 100, long_run - done)
            s0 = p.stats()
            p.set_timing(True)
            p.stage_times(reset=True)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            n_w = 0
            e0.record()
            for _ in range(k):
                p.step_sync(po, th, rv)
                n_w += p.n_sd()
                p.step_async(po)
            e1.record()
            torch.cuda.synchronize()
            s1 = p.stats()
            stg = p.stage_times(reset=True)
            p.set_timing(False)
            w_ms = e0.elapsed_time(e1)
            subs = max(s1["sd_substeps"] - s0["sd_substeps"], 1)
            long["windows"].append({"steps": [done + 1, done + k], "ms_per_step": w_ms / k, "value": n_w / (w_ms * 1e-3),
                                    "evals_per_sd_substep": (s1["newton_iters"] - s0["newton_iters"]) / subs,
                                    "slow_list_fraction": (s1["cond_slow"] - s0["cond_slow"]) / subs,
                                    "collisions_per_step": (s1["collisions"] - s0["collisions"]) / k,
                                    "max_cell_count": s1["max_cell_count"], "n_sd_live": s1["n_sd"],
                                    "cond_variant": s1["cond_variant"], "cond_tile_cells": s1["cond_tile_cells"],
                                    "coal_tile_cells": s1["coal_tile_cells"],
                                    "cond_ms": stg["cond"][0] / max(stg["cond"][1], 1), "coal_move_ms": stg["coal_move"][0] / max(stg["coal_move"][1], 1)})
            t_all += w_ms
            n_all += n_w
            done += k
        long["value"] = (n_all + sd_steps) / ((t_all + ms) * 1e-3)
        long["unit"] = UNIT
        long["note"] = f"device-timed SD-steps/s over steps {warm + 1}..{long_run} of the run (the headline window included)"

    # ---- roofline of the dominant kernel (condensation), measured live ---------------------------
    hbm_peak, peak_src = peaks()
    cond_ms, cond_n = stages["cond"]
    evals = st1["newton_iters"] - st0["newton_iters"]
    subs = st1["sd_substeps"] - st0["sd_substeps"]
    f32 = a.cond_arith == 4
    stage_ms = {k: (v[0] / v[1] if v[1] else 0.0) for k, v in stages.items()}
    step_ms = ms / a.steps
    sm_hz = (clocks.get("sm_mhz") or 1965.0) * 1e6
    n_sm = torch.cuda.get_device_properties(local).multi_processor_count
    if f32:
        flops = evals * FLOP_PER_EVAL_F32 + subs * FLOP_PER_SETUP_F32
        ach = flops / (cond_ms * 1e-3) / 1e12 if cond_ms > 0 else 0.0
        roofline = {"kernel": "k_cond4f (condensation, 10 fused substeps, fp32 sweep)", "bound": "alu", "achieved": ach, "peak": FP32_PEAK_TFLOPS,
                    "unit": "TFLOP/s", "frac": ach / FP32_PEAK_TFLOPS,
                    "peak_source": "derived: 148 SMs x 128 fp32 FMA/clk x 2 x 1.965 GHz (DESIGN.md)",
                    "traffic": NCU_COND32_DRAM_BYTES[0] if full3d else None, "traffic_source": "from profile: " + NCU_COND32_DRAM_BYTES[1]}
    else:
        instr, flops = cond_fp64_work(evals, subs)
        ach = flops / (cond_ms * 1e-3) / 1e12 if cond_ms > 0 else 0.0
        n_instr = instr["dfma"] + instr["dmul"] + instr["dadd"] + instr["other"]
        slots = n_sm * FP64_LANES_PER_SM * sm_hz * (cond_ms * 1e-3)
        roofline = {"kernel": "k_cond4 (condensation, 10 fused substeps)", "bound": "alu", "achieved": ach, "peak": fp64_peak_tflops,
                    "unit": "TFLOP/s", "frac": ach / fp64_peak_tflops,
                    "peak_source": "measured on this device before the timed region: sdm_measure_fp64_peak (independent DFMA chains, "
                                   "%.1f FMA/clk/SM); flops executed: DFMA = 2, DMUL = DADD = 1" % fp64_lanes,
                    "fp64_issue_slot_frac": n_instr / slots if slots > 0 else None,
                    "fp64_thread_instr_per_sd_substep": n_instr / max(subs, 1),
                    "fp64_instr_mix": {k: v / n_instr for k, v in instr.items()}, "fp64_instr_source": FP64_INSTR_SOURCE,
                    "traffic": NCU_COND_DRAM_BYTES[0] if full3d and a.real_bytes == 8 else None,
                    "traffic_source": "from profile: " + NCU_COND_DRAM_BYTES[1]}
    roofline.update({"evals_per_sd_substep": evals / max(subs, 1),
                     "slow_list_fraction": (st1["cond_slow"] - st0["cond_slow"]) / max(subs, 1), "ms_per_launch": cond_ms / max(cond_n, 1),
                     "share_of_step": (cond_ms / max(cond_n, 1)) / step_ms})
    bytes_step = BYTES_PER_SD_STEP[(ndim, a.real_bytes)] * (sd_steps / a.steps)
    hbm = {"bound": "hbm", "achieved": bytes_step / (step_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
           "frac": bytes_step / (step_ms * 1e-3) / 1e9 / hbm_peak, "peak_source": peak_src,
           "algorithmic_bytes_per_sd_step": BYTES_PER_SD_STEP[(ndim, a.real_bytes)]}
    sb = stage_bytes(ndim, a.real_bytes)
    roofline_stages = {k: {"bytes_per_sd": sb[k], "achieved": sb[k] * (sd_steps / a.steps) / (stage_ms[k] * 1e-3) / 1e9, "unit": "GB/s",
                           "frac": sb[k] * (sd_steps / a.steps) / (stage_ms[k] * 1e-3) / 1e9 / hbm_peak}
                       for k in sb if stage_ms.get(k, 0.0) > 0}
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": warm,
           "ms_per_step": ms_max / a.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32" if a.cond_arith == 4 else "f64",
           "data": "synthetic", "config": dict(config_of(wa), state="fp64" if a.real_bytes == 8 else ("fp32 storage, fp32 condensation sweep (thermodynamics, feedback, coalescence probability, movement in fp64)" if a.cond_arith == 4 else "fp32 storage, fp64 arithmetic")), "clocks": clocks, "e2e": e2e,
           "gpu_launches": st1["kernel_launches"] - st0["kernel_launches"], "host_syncs_per_step": (st1["host_syncs"] - st0["host_syncs"]) / a.steps,
           "roofline": roofline, "roofline_step_hbm": hbm, "roofline_stages_hbm": roofline_stages,
           "stage_ms": stage_ms, "n_sd_live": st1["n_sd"], "n_sd_initial": n_sd0,
           "launch_config": {k: st1[k] for k in ("cond_variant", "cond_tile_cells", "coal_tile_cells", "max_cell_count")}}
    if long is not None:
        out["long_run"] = long
    if a.cond_adapt_tol > 0.0:
        out["config"]["cond_adapt_tol"] = a.cond_adapt_tol
        out["sd_substeps_per_sd_step"] = subs / max(sd_steps, 1)
    if a.decomp == "slab":
        out["config"]["parallelism"] = "one domain of %d x %d columns in x-slabs, one per rank; leavers exchanged every step (slab.py)" % (world, wa["nx"])
    if a.recycle:
        out["config"]["recycling"] = "on (PAPER.md :641)"
        out["recycled"] = st1["recycled"] - st0["recycled"]
    if not a.no_cpu_baseline:
        v, cores, desc, _, _ = oracle_rate(wa, 2, 1)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                               "value_1_thread": getattr(oracle_rate, "one_thread", None)}
    if world == 1 and a.real_bytes == 8 and a.cond_arith == 8 and not a.recycle and not a.no_fp32_mode and not a.no_cpu_baseline and a.cond_adapt_tol == 0.0 and a.decomp == "replicas":
        # the same workload and step counts in the fp32 mode of configs[4] (fp32 state, fp32 condensation sweep; radii to
        # 1e-4 instead of 1e-9): a second line of context, measured by the same code in a child process
        try:
            del p
            torch.cuda.empty_cache()
            cmd = [sys.executable, os.path.abspath(__file__), "--steps", str(a.steps), "--warmup", str(a.warmup), "--workload", a.workload,
                   "--sd-per-cell", str(a.sd_per_cell), "--scale", str(a.scale), "--real-bytes", "4", "--cond-arith", "4", "--no-cpu-baseline",
                   "--long-run", "0"]
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
            d = json.loads(r.stdout.strip().splitlines()[-1])
            out["fp32_mode"] = {k: d[k] for k in ("value", "unit", "ms_per_step", "dtype", "stage_ms", "gpu_launches")}
            out["fp32_mode"]["state"] = d["config"]["state"]
            out["fp32_mode"]["e2e"] = d["e2e"]["value"]
            out["fp32_mode"]["roofline"] = {k: d["roofline"][k] for k in ("kernel", "bound", "achieved", "peak", "unit", "frac")}
            out["fp32_mode"]["roofline_step_hbm_frac"] = d["roofline_step_hbm"]["frac"]
            out["fp32_mode"]["parity"] = "radii within 1e-4 of the fp64 oracle (tests/test_parity_gpu.py::test_fp32_arithmetic_condensation_2d_3d_and_first_step)"
        except Exception as ex:   # context only: never fails the bench line
            out["fp32_mode"] = {"unavailable": str(ex)[:200]}
        # ... and with the adaptive substepping the paper plans (:566; DESIGN.md R-adapt) at cond_adapt_tol = 5e-4: changes the
        # results by its time-discretisation error (radii of droplets: 99th percentile 2e-3 after 70 steps), hence context only
        try:
            cmd = [sys.executable, os.path.abspath(__file__), "--steps", str(a.steps), "--warmup", str(a.warmup), "--workload", a.workload,
                   "--sd-per-cell", str(a.sd_per_cell), "--scale", str(a.scale), "--cond-adapt-tol", "5e-4", "--no-cpu-baseline", "--long-run", "0"]
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
            d = json.loads(r.stdout.strip().splitlines()[-1])
            out["adaptive_substeps_mode"] = {k: d[k] for k in ("value", "unit", "ms_per_step", "stage_ms", "sd_substeps_per_sd_step")}
            out["adaptive_substeps_mode"]["cond_adapt_tol"] = 5e-4
            out["adaptive_substeps_mode"]["parity"] = "tests/test_parity_gpu.py::test_adaptive_condensation_substeps_match_the_oracle"
        except Exception as ex:
            out["adaptive_substeps_mode"] = {"unavailable": str(ex)[:200]}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
