#!/usr/bin/env python
"""The calling sequence of PAPER.md Figure 7 (section 5.2.2, :831-852) on the 2D prescribed-flow set-up of section 2
(:89-138): a prototype Eulerian solver (first-order upstream advection of theta and r_v, ``sdm_upstream_advect``) and the
particle-based scheme running side by side on one GPU.

    python -m paper_1310_1905_b200.examples.kinematic_2d [--steps 600] [--sd-per-cell 32] [--outfreq 100]

Per time step (Fig. 7, "adjustments"):
  stream A:  step_sync (sort + condensation; theta, r_v final)  ->  step_async (coalescence, advection, sedimentation)
  stream B:  wait for step_sync  ->  advect theta, r_v   (runs WHILE step_async runs, :816)
  join:      the next step_sync waits for both.
Every ``outfreq`` steps (Fig. 7, "output"): diag_wet_rng / diag_wet_mom for the cloud- and rain-water mixing ratios, diag_sd_conc.
Everything numerical happens in libsdm's kernels; this file only orders the calls.  There is no CPU fallback.
"""
import argparse
import math

import torch

from paper_1310_1905_b200 import binding, workloads


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=600)
    ap.add_argument("--sd-per-cell", type=int, default=32)
    ap.add_argument("--outfreq", type=int, default=100)
    ap.add_argument("--serial", action="store_true", help="no overlap: the solver waits for step_async (for comparison)")
    a = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("kinematic_2d: needs a CUDA device (libsdm has no CPU fallback)")
    w = workloads.cfg2_2d(sd_per_cell=a.sd_per_cell, device="cuda")
    p = binding.Particles(max_sd=w.n_sd, sd_conc_mean=a.sd_per_cell, **w.init)
    s = w.state
    p.init_from_arrays(w.rhod, s["n"], s["rw2"], s["rd3"], s["kappa"], s["x"], s["y"], s["z"], s["id"],
                       courant_1=w.courants[0], courant_2=w.courants[1])
    th, rv = w.th.clone(), w.rv.clone()
    opts = binding.make_opts(**w.opts)
    lib, solver = torch.cuda.Stream(), torch.cuda.Stream()
    rho_w = 1000.0
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t0.record(lib)
    rain = 0.0
    for step in range(1, a.steps + 1):
        with torch.cuda.stream(lib):
            p.step_sync(opts, th, rv)             # theta, r_v are final once this stream work completes (:816)
            fields_ready = torch.cuda.Event()
            fields_ready.record(lib)
            p.step_async(opts)                    # only enqueues
        if a.serial:
            lib.synchronize()
        with torch.cuda.stream(solver):           # the host model's own work, concurrent with step_async
            solver.wait_event(fields_ready)
            p.upstream_advect(th)
            p.upstream_advect(rv)
        lib.wait_stream(solver)                   # "wait for ..." of Fig. 7: the next step_sync reads the solver's fields
        with torch.cuda.stream(lib):
            rain += p.step_async_result()
            if step % a.outfreq == 0:
                p.diag_wet_rng(0.5e-6, 25e-6)
                qc = p.diag_wet_mom(3).clone() * (4.0 / 3.0) * math.pi * rho_w     # cloud water [kg/kg]
                p.diag_wet_rng(25e-6, 1.0)
                qr = p.diag_wet_mom(3).clone() * (4.0 / 3.0) * math.pi * rho_w     # rain water [kg/kg]
                conc = p.diag_sd_conc()
                print(f"step {step:5d}  SDs {p.n_sd():8d}  q_c max {float(qc.max()) * 1e3:7.4f} g/kg  q_r max {float(qr.max()) * 1e3:9.6f} g/kg  "
                      f"SD/cell {float(conc.min()):.0f}..{float(conc.max()):.0f}  rain {rain:.3e} kg  "
                      f"theta {float(th.min()):.3f}..{float(th.max()):.3f} K", flush=True)
    t1.record(lib)
    torch.cuda.synchronize()
    st = p.stats()
    print(f"{a.steps} steps, {t0.elapsed_time(t1) / a.steps:.3f} ms/step ({'serial' if a.serial else 'overlapped'}), "
          f"{st['collisions']} collisions, {st['kernel_launches']} kernel launches")


if __name__ == "__main__":
    main()
